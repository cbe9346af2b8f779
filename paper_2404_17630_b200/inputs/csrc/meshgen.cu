// Input generator library (libmeshgen.so): jittered-lattice Voronoi meshes for configs 2-4
// of BASELINE.json, on the host (OpenMP) or directly in device memory.  It serves the oracle
// tests and the CUDA path alike and holds none of the RT method's arithmetic (task rule 3).
//
// Two passes, both recomputing the cell: (1) per cell: volume, centroid, number of faces
// the cell emits (faces towards a higher cell id, and box faces); (2) given the exclusive
// prefix sum of those counts, write each face once: area, unit normal (left -> right),
// centroid (in the left cell's frame; may lie outside the box when periodic), left, right.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include "voronoi_cell.h"

extern "C" {
typedef struct {
  int32_t n;        // lattice cells per dimension, C = n^3 (2 n^3 if staggered), lattice id = (ix*n+iy)*n+iz
  int32_t periodic; // 1: periodic in all three directions, 0: clipped to the box
  int32_t bc_code;  // `right` code of box faces when not periodic (-1 outflow, -2 reflective)
  int32_t stagger;  // 1: two interleaved lattices (body-centred, the "2 x N^3 staggered grid" of PAPER.md:180, 290):
                    // cell id = sub * n^3 + lattice id, generators at (i + 0.25 + 0.5 sub + jitter*(2u-1)) * box/n
  double box;       // box side
  double jitter;    // generator = (i + 0.5 + jitter*(2u-1)) * box/n per axis (not staggered)
  uint64_t seed;
} mg_params;
}

VC_HD inline uint64_t mg_mix(uint64_t z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
VC_HD inline double mg_u01(uint64_t seed, uint64_t stream, uint64_t index) {
  uint64_t base = mg_mix(seed + stream * 0x632BE59BD9B4E019ull);
  return (double)(mg_mix(base ^ index) >> 11) * (1.0 / 9007199254740992.0);
}

#define MG_NOFF 124
struct mg_offsets { int8_t o[MG_NOFF][3]; };

static mg_offsets mg_make_offsets() {
  mg_offsets T;
  int k = 0;
  // sorted by squared length so near neighbours clip first (few dead planes)
  for (int r2 = 1; r2 <= 12; r2++)
    for (int x = -2; x <= 2; x++)
      for (int y = -2; y <= 2; y++)
        for (int z = -2; z <= 2; z++)
          if (x * x + y * y + z * z == r2) { T.o[k][0] = x; T.o[k][1] = y; T.o[k][2] = z; k++; }
  return T;
}

VC_HD inline double mg_jit(const mg_params& P, int64_t cell, int axis) {
  return P.jitter * (2.0 * mg_u01(P.seed, (uint64_t)axis, (uint64_t)cell) - 1.0);
}
// position of a generator in units of the lattice spacing, relative to its lattice site's corner
VC_HD inline double mg_site(const mg_params& P, int sub) { return P.stagger ? 0.25 + 0.5 * sub : 0.5; }

// Build the Voronoi cell of `cell`; seed position returned in pos.
VC_HD inline void mg_build(const mg_params& P, const mg_offsets& T, int64_t cell, VCell& c, double pos[3]) {
  const int n = P.n;
  const double h = P.box / n;
  const int64_t n3 = (int64_t)n * n * n;
  const int sub = (int)(cell / n3);
  const int64_t lat = cell - sub * n3;
  int iz = (int)(lat % n), iy = (int)((lat / n) % n), ix = (int)(lat / ((int64_t)n * n));
  double ui[3] = {mg_jit(P, cell, 0), mg_jit(P, cell, 1), mg_jit(P, cell, 2)};
  const double s0 = mg_site(P, sub);
  pos[0] = (ix + s0 + ui[0]) * h; pos[1] = (iy + s0 + ui[1]) * h; pos[2] = (iz + s0 + ui[2]) * h;
  double lo[3], hi[3];
  for (int a = 0; a < 3; a++) {
    if (P.periodic) { lo[a] = -2.5 * h; hi[a] = 2.5 * h; }
    else { lo[a] = -pos[a]; hi[a] = P.box - pos[a]; }
  }
  vc_init(c, lo, hi);
  auto clip_by = [&](int ox, int oy, int oz, int osub) {
    int jx = ix + ox, jy = iy + oy, jz = iz + oz;
    if (P.periodic) {
      jx = (jx % n + n) % n; jy = (jy % n + n) % n; jz = (jz % n + n) % n;
    } else if (jx < 0 || jx >= n || jy < 0 || jy >= n || jz < 0 || jz >= n) return;
    const int64_t j = osub * n3 + ((int64_t)jx * n + jy) * n + jz;
    const double sh = mg_site(P, osub) - s0;  // 0 on the same lattice, +-0.5 across the two
    double rx = (ox + sh + mg_jit(P, j, 0) - ui[0]) * h;
    double ry = (oy + sh + mg_jit(P, j, 1) - ui[1]) * h;
    double rz = (oz + sh + mg_jit(P, j, 2) - ui[2]) * h;
    vc_clip(c, rx, ry, rz, -0.5 * (rx * rx + ry * ry + rz * rz), (int32_t)j);
  };
  if (P.stagger) {  // the eight nearest generators sit on the other lattice, at (+-0.5, +-0.5, +-0.5)
    const int b = sub ? 0 : -1;  // other-lattice offsets o with o + sh = -0.5, +0.5
    for (int x = b; x <= b + 1; x++)
      for (int y = b; y <= b + 1; y++)
        for (int z = b; z <= b + 1; z++) clip_by(x, y, z, 1 - sub);
  }
  for (int k = 0; k < MG_NOFF; k++) clip_by(T.o[k][0], T.o[k][1], T.o[k][2], sub);
  if (P.stagger) {  // the rest of the other lattice's 4 x 4 x 4 block (relative offsets -1.5 .. 1.5)
    const int b = sub ? -1 : -2;
    for (int x = b; x <= b + 3; x++)
      for (int y = b; y <= b + 3; y++)
        for (int z = b; z <= b + 3; z++) {
          const int in = (x > b && x < b + 3) && (y > b && y < b + 3) && (z > b && z < b + 3);
          if (!in) clip_by(x, y, z, 1 - sub);
        }
  }
  // security: every generator outside the blocks is >= (3 - 2 jitter) h (same lattice) or (2.5 - 2 jitter) h (the
  // other lattice) away along one axis
  double lim = ((P.stagger ? 2.5 : 3.0) - 2.0 * P.jitter) * h;
  for (int q = 0; q < c.nt; q++) {
    double ax = fabs(c.vx[q]), ay = fabs(c.vy[q]), az = fabs(c.vz[q]);
    double m = ax > ay ? (ax > az ? ax : az) : (ay > az ? ay : az);
    if (sqrt(ax * ax + ay * ay + az * az) + m > lim) c.status |= VC_E_SECURITY;
  }
}

// One pass over the cell's faces. mode 0: count + volume + centroid; mode 1: write faces.
VC_HD inline void mg_cell(const mg_params& P, const mg_offsets& T, int64_t cell, int mode,
                          int32_t* counts, double* volume, double* centroid, int64_t C,
                          const int64_t* offsets, double* area, double* normal, double* fcen,
                          int32_t* left, int32_t* right, int64_t F, int32_t* status) {
  VCell c;
  double pos[3];
  mg_build(P, T, cell, c, pos);
  const double h = P.box / P.n;
  const double amin = 1e-13 * h * h;
  int cnt = 0;
  double vol = 0.0, mx = 0.0, my = 0.0, mz = 0.0;
  int64_t base = mode ? offsets[cell] : 0;
  for (int p = 0; p < c.np && !c.status; p++) {
    double A, cx, cy, cz;
    if (vc_face(c, p, A, cx, cy, cz) < 3) continue;
    double nn = sqrt(c.pa[p] * c.pa[p] + c.pb[p] * c.pb[p] + c.pc[p] * c.pc[p]);
    double nx = c.pa[p] / nn, ny = c.pb[p] / nn, nz = c.pc[p] / nn;
    double hgt = cx * nx + cy * ny + cz * nz; // seed-to-plane distance
    double pv = A * hgt / 3.0;                // pyramid with apex at the seed
    vol += pv; mx += pv * 0.75 * cx; my += pv * 0.75 * cy; mz += pv * 0.75 * cz;
    int32_t id = c.pid[p];
    if (id < 0 && P.periodic) { c.status |= VC_E_OPEN; break; }
    if (A <= amin) continue;
    if (id >= 0 && (int64_t)id < cell) continue; // the lower cell emits the face
    if (mode) {
      int64_t f = base + cnt;
      area[f] = A;
      normal[f] = nx; normal[F + f] = ny; normal[2 * F + f] = nz;
      fcen[f] = pos[0] + cx; fcen[F + f] = pos[1] + cy; fcen[2 * F + f] = pos[2] + cz;
      left[f] = (int32_t)cell;
      right[f] = id >= 0 ? id : P.bc_code;
    }
    cnt++;
  }
  if (!mode) {
    counts[cell] = cnt;
    volume[cell] = vol;
    centroid[cell] = pos[0] + mx / vol;
    centroid[C + cell] = pos[1] + my / vol;
    centroid[2 * C + cell] = pos[2] + mz / vol;
  }
  if (c.status) {
#ifdef __CUDA_ARCH__
    atomicOr(status, c.status);
    atomicAdd(status + 1, 1);
#else
#pragma omp critical
    { status[0] |= c.status; status[1] += 1; }
#endif
  }
}

__global__ void __launch_bounds__(64) mg_kernel(mg_params P, mg_offsets T, int mode, int32_t* counts,
                                               double* volume, double* centroid, int64_t C,
                                               const int64_t* offsets, double* area, double* normal,
                                               double* fcen, int32_t* left, int32_t* right, int64_t F,
                                               int32_t* status) {
  int64_t cell = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (cell >= C) return;
  mg_cell(P, T, cell, mode, counts, volume, centroid, C, offsets, area, normal, fcen, left, right, F, status);
}

static int mg_run(const mg_params* P, int on_device, void* stream, int mode, int32_t* counts, double* volume,
                  double* centroid, const int64_t* offsets, double* area, double* normal, double* fcen,
                  int32_t* left, int32_t* right, int64_t F, int32_t* status_out) {
  if (!P || P->n < 1 || (P->periodic && P->n < 5) || P->jitter < 0.0 || P->jitter > 0.45) return -1;
  int64_t C = (int64_t)P->n * P->n * P->n * (P->stagger ? 2 : 1);
  mg_offsets T = mg_make_offsets();
  int32_t st[2] = {0, 0};
  if (on_device) {
    cudaStream_t s = (cudaStream_t)stream;
    int32_t* dst;
    if (cudaMalloc(&dst, 2 * sizeof(int32_t)) != cudaSuccess) return -2;
    cudaMemsetAsync(dst, 0, 2 * sizeof(int32_t), s);
    int64_t nb = (C + 63) / 64;
    mg_kernel<<<(unsigned)nb, 64, 0, s>>>(*P, T, mode, counts, volume, centroid, C, offsets, area, normal, fcen,
                                          left, right, F, dst);
    cudaError_t e = cudaMemcpyAsync(st, dst, 2 * sizeof(int32_t), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cudaFree(dst);
    if (e != cudaSuccess) return -2;
  } else {
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t cell = 0; cell < C; cell++)
      mg_cell(*P, T, cell, mode, counts, volume, centroid, C, offsets, area, normal, fcen, left, right, F, st);
  }
  if (status_out) { status_out[0] = st[0]; status_out[1] = st[1]; }
  return st[0] ? -3 : 0;
}

extern "C" {

// Pass 1. counts[C] int32, volume[C], centroid[3][C]; all host or all device pointers.
// status_out[2] (host): OR of VC_E_* bits, number of bad cells. Returns 0, or <0 on error.
int mg_voronoi_cells(const mg_params* P, int on_device, void* stream, int32_t* counts, double* volume,
                     double* centroid, int32_t* status_out) {
  return mg_run(P, on_device, stream, 0, counts, volume, centroid, 0, 0, 0, 0, 0, 0, 0, status_out);
}

// Pass 2. offsets[C] int64 = exclusive prefix sum of counts; nface = total.
// area[F], normal[3][F], fcentroid[3][F], left[F], right[F].
int mg_voronoi_faces(const mg_params* P, int on_device, void* stream, const int64_t* offsets, int64_t nface,
                     double* area, double* normal, double* fcentroid, int32_t* left, int32_t* right,
                     int32_t* status_out) {
  return mg_run(P, on_device, stream, 1, 0, 0, 0, offsets, area, normal, fcentroid, left, right, nface, status_out);
}

// u01 for tests that check the numpy and C generators agree bit for bit.
double mg_u01_c(uint64_t seed, uint64_t stream, uint64_t index) { return mg_u01(seed, stream, index); }
}
