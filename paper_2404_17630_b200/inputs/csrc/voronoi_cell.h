// Input generator, not part of the RT method: one Voronoi cell of a jittered-lattice
// generator set, built by clipping a convex polyhedron against the bisector planes of the
// 5x5x5 block of lattice neighbours.
//
// The cell is kept in dual form: a list of half-spaces (planes) and a list of oriented
// triangles (i,j,k) of plane indices, each triangle being one vertex of the polyhedron
// (the intersection of its three planes).  Clipping by a new plane removes the triangles
// whose vertex lies outside, and closes the hole with a fan (a,b,new) over the hole's
// boundary edges.  Compiles for host (g++/OpenMP) and device (nvcc) alike.
#pragma once
#include <stdint.h>
#include <math.h>

#ifdef __CUDACC__
#define VC_HD __host__ __device__
#else
#define VC_HD
#endif

#define VC_MAXP 72
#define VC_MAXT 112
#define VC_MAXE 96

// status bits
#define VC_OK 0
#define VC_E_PLANES 1    // plane list overflow
#define VC_E_TRIS 2      // triangle list overflow
#define VC_E_TOPO 4      // hole boundary is not a simple cycle
#define VC_E_EMPTY 8     // cell clipped away
#define VC_E_SECURITY 16 // a vertex is too far: the 5x5x5 block is not enough
#define VC_E_OPEN 32     // periodic cell still touches the initial cube

struct VCell {
  double pa[VC_MAXP], pb[VC_MAXP], pc[VC_MAXP], pd[VC_MAXP]; // a x + b y + c z + d <= 0 inside
  int32_t pid[VC_MAXP];                                       // neighbour cell id, or -1-k: cube plane k
  int np;
  uint8_t t[VC_MAXT][3];
  double vx[VC_MAXT], vy[VC_MAXT], vz[VC_MAXT];               // vertex of each triangle, seed at origin
  int nt;
  int status;
};

VC_HD inline void vc_vertex(const VCell& c, int i, int j, int k, double& x, double& y, double& z) {
  // Cramer's rule for n_i.x = -d_i, n_j.x = -d_j, n_k.x = -d_k
  double a1 = c.pa[i], b1 = c.pb[i], c1 = c.pc[i], d1 = -c.pd[i];
  double a2 = c.pa[j], b2 = c.pb[j], c2 = c.pc[j], d2 = -c.pd[j];
  double a3 = c.pa[k], b3 = c.pb[k], c3 = c.pc[k], d3 = -c.pd[k];
  double m11 = b2 * c3 - c2 * b3, m12 = a2 * c3 - c2 * a3, m13 = a2 * b3 - b2 * a3;
  double det = a1 * m11 - b1 * m12 + c1 * m13;
  double inv = 1.0 / det;
  x = (d1 * m11 - b1 * (d2 * c3 - c2 * d3) + c1 * (d2 * b3 - b2 * d3)) * inv;
  y = (a1 * (d2 * c3 - c2 * d3) - d1 * m12 + c1 * (a2 * d3 - d2 * a3)) * inv;
  z = (a1 * (b2 * d3 - d2 * b3) - b1 * (a2 * d3 - d2 * a3) + d1 * m13) * inv;
}

// Start from the axis-aligned box [lo, hi] (coordinates relative to the seed).
VC_HD inline void vc_init(VCell& c, const double lo[3], const double hi[3]) {
  c.status = VC_OK;
  c.np = 6;
  for (int k = 0; k < 6; k++) { c.pa[k] = c.pb[k] = c.pc[k] = 0.0; c.pid[k] = -1 - k; }
  c.pa[0] = -1.0; c.pd[0] = lo[0];   // -x + lo <= 0
  c.pa[1] = 1.0;  c.pd[1] = -hi[0];  //  x - hi <= 0
  c.pb[2] = -1.0; c.pd[2] = lo[1];
  c.pb[3] = 1.0;  c.pd[3] = -hi[1];
  c.pc[4] = -1.0; c.pd[4] = lo[2];
  c.pc[5] = 1.0;  c.pd[5] = -hi[2];
  // the 8 corners as oriented dual triangles: det[n_i,n_j,n_k] > 0
  c.nt = 0;
  for (int sx = 0; sx < 2; sx++)
    for (int sy = 0; sy < 2; sy++)
      for (int sz = 0; sz < 2; sz++) {
        int i = sx, j = 2 + sy, k = 4 + sz;
        int neg = (sx == 0) + (sy == 0) + (sz == 0); // normals -e flip the determinant
        int q = c.nt++;
        c.t[q][0] = (uint8_t)i;
        if (neg & 1) { c.t[q][1] = (uint8_t)k; c.t[q][2] = (uint8_t)j; }
        else         { c.t[q][1] = (uint8_t)j; c.t[q][2] = (uint8_t)k; }
        vc_vertex(c, c.t[q][0], c.t[q][1], c.t[q][2], c.vx[q], c.vy[q], c.vz[q]);
      }
}

// Clip by the half-space a x + b y + c z + d <= 0 tagged with neighbour id.
VC_HD inline void vc_clip(VCell& c, double a, double b, double cc, double d, int32_t id) {
  if (c.status) return;
  int nrem = 0;
  uint8_t rem[VC_MAXT];
  for (int q = 0; q < c.nt; q++) {
    double s = a * c.vx[q] + b * c.vy[q] + cc * c.vz[q] + d;
    rem[q] = (s > 0.0);
    nrem += rem[q];
  }
  if (nrem == 0) return;
  if (nrem == c.nt) { c.status |= VC_E_EMPTY; return; }
  if (c.np >= VC_MAXP) { c.status |= VC_E_PLANES; return; }
  int p = c.np++;
  c.pa[p] = a; c.pb[p] = b; c.pc[p] = cc; c.pd[p] = d; c.pid[p] = id;
  // directed edges of removed triangles
  uint8_t ea[VC_MAXE], eb[VC_MAXE];
  int ne = 0;
  for (int q = 0; q < c.nt; q++)
    if (rem[q]) {
      if (ne + 3 > VC_MAXE) { c.status |= VC_E_TRIS; return; }
      ea[ne] = c.t[q][0]; eb[ne] = c.t[q][1]; ne++;
      ea[ne] = c.t[q][1]; eb[ne] = c.t[q][2]; ne++;
      ea[ne] = c.t[q][2]; eb[ne] = c.t[q][0]; ne++;
    }
  // compact the kept triangles
  int w = 0;
  for (int q = 0; q < c.nt; q++)
    if (!rem[q]) {
      if (w != q) {
        c.t[w][0] = c.t[q][0]; c.t[w][1] = c.t[q][1]; c.t[w][2] = c.t[q][2];
        c.vx[w] = c.vx[q]; c.vy[w] = c.vy[q]; c.vz[w] = c.vz[q];
      }
      w++;
    }
  c.nt = w;
  // boundary edges: those whose reverse is not an edge of a removed triangle
  int nb = 0;
  for (int e = 0; e < ne; e++) {
    int twin = 0;
    for (int f = 0; f < ne; f++)
      if (ea[f] == eb[e] && eb[f] == ea[e]) { twin = 1; break; }
    if (twin) continue;
    if (c.nt >= VC_MAXT) { c.status |= VC_E_TRIS; return; }
    int q = c.nt++;
    c.t[q][0] = ea[e]; c.t[q][1] = eb[e]; c.t[q][2] = (uint8_t)p;
    vc_vertex(c, ea[e], eb[e], p, c.vx[q], c.vy[q], c.vz[q]);
    nb++;
  }
  if (nb < 3) c.status |= VC_E_TOPO;
}

// Polygon of plane p: area, centroid (relative to the seed). Returns number of vertices
// (0 if the plane carries no face).
VC_HD inline int vc_face(VCell& c, int p, double& area, double& cx, double& cy, double& cz) {
  // triangles containing p, rotated so that p comes first: (p, a, b)
  uint8_t fa[32], fb[32];
  int16_t fq[32];
  int k = 0;
  for (int q = 0; q < c.nt; q++) {
    int i = c.t[q][0], j = c.t[q][1], l = c.t[q][2];
    int a, b;
    if (i == p) { a = j; b = l; }
    else if (j == p) { a = l; b = i; }
    else if (l == p) { a = i; b = j; }
    else continue;
    if (k >= 32) { c.status |= VC_E_TRIS; return 0; }
    fa[k] = (uint8_t)a; fb[k] = (uint8_t)b; fq[k] = (int16_t)q; k++;
  }
  if (k < 3) return 0;
  // chain: next triangle's a equals this one's b
  for (int s = 0; s + 1 < k; s++) {
    int found = -1;
    for (int r = s + 1; r < k; r++)
      if (fa[r] == fb[s]) { found = r; break; }
    if (found < 0) { c.status |= VC_E_TOPO; return 0; }
    uint8_t ta = fa[s + 1], tb = fb[s + 1]; int16_t tq = fq[s + 1];
    fa[s + 1] = fa[found]; fb[s + 1] = fb[found]; fq[s + 1] = fq[found];
    fa[found] = ta; fb[found] = tb; fq[found] = tq;
  }
  if (fb[k - 1] != fa[0]) { c.status |= VC_E_TOPO; return 0; }
  // fan about vertex 0
  double x0 = c.vx[fq[0]], y0 = c.vy[fq[0]], z0 = c.vz[fq[0]];
  double nn = sqrt(c.pa[p] * c.pa[p] + c.pb[p] * c.pb[p] + c.pc[p] * c.pc[p]);
  double nx = c.pa[p] / nn, ny = c.pb[p] / nn, nz = c.pc[p] / nn;
  double A = 0.0, sx = 0.0, sy = 0.0, sz = 0.0;
  for (int s = 1; s + 1 < k; s++) {
    double ux = c.vx[fq[s]] - x0, uy = c.vy[fq[s]] - y0, uz = c.vz[fq[s]] - z0;
    double wx = c.vx[fq[s + 1]] - x0, wy = c.vy[fq[s + 1]] - y0, wz = c.vz[fq[s + 1]] - z0;
    double ax = uy * wz - uz * wy, ay = uz * wx - ux * wz, az = ux * wy - uy * wx;
    double ta = 0.5 * (ax * nx + ay * ny + az * nz);
    A += ta;
    sx += ta * (ux + wx); sy += ta * (uy + wy); sz += ta * (uz + wz);
  }
  if (A == 0.0) return 0;
  cx = x0 + sx / (3.0 * A); cy = y0 + sy / (3.0 * A); cz = z0 + sz / (3.0 * A);
  area = fabs(A);
  return k;
}
