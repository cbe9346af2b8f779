// rt_mesh_upload's device-side setup: validation, Peano-Hilbert reordering, faces by owner,
// cell -> face lists, and the mesh-only parts of eq (15).
// Runs once per mesh, outside the timed subcycles.  CUB is used for the two radix sorts.
#include <cub/cub.cuh>
#include <string.h>
#include <stdlib.h>
#include <vector>
#include "rt_internal.cuh"
#include "rt_kernels.cuh"

#define SETUP_BLOCK 256
static inline unsigned nblk(int64_t n) { return (unsigned)((n + SETUP_BLOCK - 1) / SETUP_BLOCK); }

struct geom_in {
  const double *volume, *centroid, *area, *normal, *fcentroid;
  const int32_t *left, *right;
};

// component a of face q's record: the face arrays are stored as two halves, [F][2] = components
// 0-1 followed by [F][2] = components 2-3 (rt_internal.cuh)
#define FA(arr, q, a) (arr)[((a) < 2 ? 0 : 2 * F) + 2 * (int64_t)(q) + ((a) & 1)]

// error flag bits
enum { E_LEFT = 1, E_RIGHT = 2, E_VOL = 4, E_AREA = 8, E_NORMAL = 16, E_CLOSURE = 32, E_MATRIX = 64, E_GHOST = 128 };

__global__ void k_validate(geom_in g, int64_t C, int64_t F, int nghost, int *flags) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int e = 0;
  if (i < C && !(g.volume[i] > 0.0)) e |= E_VOL;
  if (i < F) {
    if (g.left[i] < 0 || g.left[i] >= C) e |= E_LEFT;
    int32_t r = g.right[i];
    if (r >= C || r == g.left[i]) e |= E_RIGHT;
    if (r <= RT_BC_DIRICHLET0 && (RT_BC_DIRICHLET0 - r) >= nghost) e |= E_GHOST;
    if (!(g.area[i] > 0.0)) e |= E_AREA;
    double nx = g.normal[i], ny = g.normal[F + i], nz = g.normal[2 * F + i];
    if (!(fabs(nx * nx + ny * ny + nz * nz - 1.0) < 1e-10)) e |= E_NORMAL;
  }
  if (e) atomicOr(flags, e);
}

// Hilbert index of a 3-D point with 21 bits per axis (Skilling's transpose algorithm).
__device__ inline uint64_t hilbert3(uint32_t x, uint32_t y, uint32_t z) {
  const int b = 21;
  uint32_t X[3] = {x, y, z};
  uint32_t M = 1u << (b - 1);
  for (uint32_t Q = M; Q > 1; Q >>= 1) {
    uint32_t P = Q - 1;
    for (int i = 0; i < 3; i++) {
      if (X[i] & Q) X[0] ^= P;
      else { uint32_t t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }
    }
  }
  X[1] ^= X[0]; X[2] ^= X[1];
  uint32_t t = 0;
  for (uint32_t Q = M; Q > 1; Q >>= 1) if (X[2] & Q) t ^= Q - 1;
  X[0] ^= t; X[1] ^= t; X[2] ^= t;
  uint64_t key = 0;
  for (int k = b - 1; k >= 0; k--)
    for (int i = 0; i < 3; i++) key = (key << 1) | ((X[i] >> k) & 1u);
  return key;
}

__global__ void k_cell_keys(const double *centroid, int64_t C, double bx, double by, double bz, uint64_t *keys,
                            int32_t *idx) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= C) return;
  double b[3] = {bx, by, bz};
  uint32_t q[3];
  for (int a = 0; a < 3; a++) {
    double u = centroid[a * C + i] / b[a];
    u -= floor(u);  // wrap into [0,1)
    double v = u * 2097152.0;
    q[a] = v >= 2097151.0 ? 2097151u : (uint32_t)v;
  }
  keys[i] = hilbert3(q[0], q[1], q[2]);
  idx[i] = (int32_t)i;
}

__global__ void k_permute_cells(geom_in g, int64_t C, const int32_t *perm, int32_t *iperm, double *cellS, double *cellV) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= C) return;
  int32_t o = perm[p];
  iperm[o] = (int32_t)p;
  for (int a = 0; a < 3; a++) cellS[4 * p + a] = g.centroid[a * C + o];
  cellS[4 * p + 3] = g.volume[o];
  cellV[p] = g.volume[o];
}

__device__ inline uint64_t face_key(int32_t l, int32_t r) {
  uint32_t sub = r >= 0 ? (uint32_t)r : 0x80000000u + (uint32_t)(-r);
  return ((uint64_t)(uint32_t)l << 32) | sub;
}

__global__ void k_face_keys(geom_in g, int64_t F, const int32_t *iperm, uint64_t *keys, int32_t *idx) {
  int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= F) return;
  int32_t l = iperm[g.left[f]], r = g.right[f];
  if (r >= 0) { r = iperm[r]; if (r < l) { int32_t t = l; l = r; r = t; } }
  keys[f] = face_key(l, r);
  idx[f] = (int32_t)f;
}

__global__ void k_gather_faces(geom_in g, int64_t C, int64_t F, const int32_t *order, const uint64_t *keys,
                               const int32_t *iperm, const double *cellS, double bx, double by, double bz, int p0,
                               int p1, int p2, double *faceC, double *faceN, int32_t *L, int32_t *R) {
  int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= F) return;
  int32_t f = order[q];
  int32_t l = (int32_t)(keys[q] >> 32);
  int32_t ro = g.right[f];
  int32_t r = ro >= 0 ? iperm[ro] : ro;
  bool flip = (iperm[g.left[f]] != l);
  if (flip) r = iperm[g.left[f]];
  L[q] = l; R[q] = r;
  FA(faceN, q, 3) = 0.0;
  FA(faceC, q, 3) = g.area[f];
  double sg = flip ? -1.0 : 1.0;
  double b[3] = {bx, by, bz};
  int per[3] = {p0, p1, p2};
  for (int a = 0; a < 3; a++) {
    FA(faceN, q, a) = sg * g.normal[a * F + f];
    double sl = cellS[4 * (int64_t)l + a];
    FA(faceC, q, a) = rt_wrap(g.fcentroid[a * F + f] - sl, b[a], per[a]);  // relative to the left cell's centroid
  }
}

// first index q in sorted keys with keys[q] >= (i << 32), for i = 0..C
__global__ void k_lower_bounds(const uint64_t *keys, int64_t n, int64_t C, int64_t *out) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i > C) return;
  uint64_t target = (uint64_t)i << 32;
  int64_t lo = 0, hi = n;
  while (lo < hi) {
    int64_t mid = (lo + hi) >> 1;
    if (keys[mid] < target) lo = mid + 1; else hi = mid;
  }
  out[i] = lo;
}

__global__ void k_rkeys(const int32_t *R, int64_t F, uint64_t *keys) {
  int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= F) return;
  keys[q] = R[q] >= 0 ? (((uint64_t)(uint32_t)R[q] << 32) | (uint32_t)q) : ~0ull;
}

__global__ void k_rlist(const uint64_t *keys, int64_t NR, const int32_t *L, int32_t *rl, int32_t *rn) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= NR) return;
  int32_t q = (int32_t)(keys[k] & 0xffffffffu);
  rl[k] = q;
  rn[k] = L[q];
}

// per-face prefactor of eq (15)'s second term, seen from the left cell: w = A d/|d|^2,
// d = s_R - s_L measured through the face; boundary faces use the mirror point (S13).
// faceW = (w, kappa) with kappa = |d|^2 / A, so that d = kappa w: the face centre seen from the
// right cell is (c - s_L) - kappa w, without a min-image test in the kernels.
__global__ void k_face_geom(int64_t C, int64_t F, const double *cellS, const double *faceC, const double *faceN,
                            const int32_t *L, const int32_t *R, double bx, double by, double bz, int p0, int p1, int p2,
                            double *faceW) {
  int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= F) return;
  double b[3] = {bx, by, bz};
  int per[3] = {p0, p1, p2};
  int32_t l = L[q], r = R[q];
  double d[3];
  if (r >= 0) {
    for (int a = 0; a < 3; a++) {
      double rl = FA(faceC, q, a);
      double c = cellS[4 * (int64_t)l + a] + rl;
      d[a] = rl - rt_wrap(c - cellS[4 * (int64_t)r + a], b[a], per[a]);
    }
  } else {
    double n[3] = {FA(faceN, q, 0), FA(faceN, q, 1), FA(faceN, q, 2)};
    double p = 0.0;
    for (int a = 0; a < 3; a++) p += FA(faceC, q, a) * n[a];
    for (int a = 0; a < 3; a++) d[a] = 2.0 * p * n[a];
  }
  double d2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
  double k = FA(faceC, q, 3) / d2;
  for (int a = 0; a < 3; a++) FA(faceW, q, a) = k * d[a];
  FA(faceW, q, 3) = d2 / FA(faceC, q, 3);
}

// per cell: M = sum_f A n n^T (n = d/|d| = w/|w|), its inverse, and the closure check
__global__ void k_cell_geom(int64_t C, int64_t F, const double *faceC, const double *faceN, const double *faceW,
                            const int64_t *fo, const int64_t *ro, const int32_t *rl, double *Minv, int *flags) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= C) return;
  double m[6] = {0, 0, 0, 0, 0, 0}, cl[3] = {0, 0, 0}, sa = 0.0;
  int64_t n_own = fo[i + 1] - fo[i], n_r = ro[i + 1] - ro[i];
  for (int64_t k = 0; k < n_own + n_r; k++) {
    int64_t q = k < n_own ? fo[i] + k : rl[ro[i] + (k - n_own)];
    double sg = k < n_own ? 1.0 : -1.0;
    double a = FA(faceC, q, 3);
    double wx = FA(faceW, q, 0), wy = FA(faceW, q, 1), wz = FA(faceW, q, 2);
    double w2 = wx * wx + wy * wy + wz * wz;
    double f = a / w2;  // A n n^T = A w w^T / |w|^2
    m[0] += f * wx * wx; m[1] += f * wx * wy; m[2] += f * wx * wz;
    m[3] += f * wy * wy; m[4] += f * wy * wz; m[5] += f * wz * wz;
    cl[0] += sg * a * FA(faceN, q, 0); cl[1] += sg * a * FA(faceN, q, 1); cl[2] += sg * a * FA(faceN, q, 2);
    sa += a;
  }
  int e = 0;
  if (!(sqrt(cl[0] * cl[0] + cl[1] * cl[1] + cl[2] * cl[2]) <= 1e-10 * sa)) e |= E_CLOSURE;
  double c00 = m[3] * m[5] - m[4] * m[4], c01 = m[4] * m[2] - m[1] * m[5], c02 = m[1] * m[4] - m[3] * m[2];
  double det = m[0] * c00 + m[1] * c01 + m[2] * c02;
  if (!(fabs(det) > 0.0)) { e |= E_MATRIX; det = 1.0; }
  double id = 1.0 / det;
  Minv[6 * i + 0] = c00 * id;
  Minv[6 * i + 1] = c01 * id;
  Minv[6 * i + 2] = c02 * id;
  Minv[6 * i + 3] = (m[0] * m[5] - m[2] * m[2]) * id;
  Minv[6 * i + 4] = (m[1] * m[2] - m[0] * m[4]) * id;
  Minv[6 * i + 5] = (m[0] * m[3] - m[1] * m[1]) * id;
  if (e) atomicOr(flags, e);
}


// ---- tiles: descriptors and blobs (layout: rt_internal.cuh).  One block per tile.
// MODE 0 measures (blob words per tile, maxima), MODE 1 writes.
#define TILE_BT 128
struct tile_max { int ns, no, nh, nf, words, overflow, pad[2]; };

__device__ inline int halo_pos(const int32_t *halo, int nh, int32_t id) {
  int lo = 0, hi = nh;
  while (lo < hi) { const int mid = (lo + hi) >> 1; if (halo[mid] < id) lo = mid + 1; else hi = mid; }
  return lo;
}

template <int MODE>
__global__ void __launch_bounds__(TILE_BT) k_tile_build(int64_t C, int TC, const int64_t *fo, const int64_t *ro,
                                                        const int32_t *R, const int32_t *rl, const int32_t *rn,
                                                        int64_t *tsize, int64_t *xcnt, int64_t *icnt, int64_t *n2cnt,
                                                        tile_max *mx, int64_t bstride, const int64_t *xoff,
                                                        const int64_t *ibase, const int64_t *k2base, rt_tile *tiles,
                                                        uint32_t *blob, int32_t *faceX, int32_t *k2cell, int32_t *k2off) {
  typedef cub::BlockScan<int, TILE_BT> Scan;
  __shared__ typename Scan::TempStorage scan_tmp;
  __shared__ int32_t s_cand[RT_TILE_LIMIT], s_rank[RT_TILE_LIMIT], s_halo[RT_TILE_LIMIT];
  __shared__ int s_nc, s_run, s_bnd;
  const int64_t t = blockIdx.x;
  const int64_t c0 = t * TC, c1 = c0 + TC < C ? c0 + TC : C;
  const int ncell = (int)(c1 - c0);
  const int64_t fbase = fo[c0], rbase = ro[c0];
  const int64_t nown64 = fo[c1] - fbase, nr64 = ro[c1] - rbase;
  if (nown64 > RT_TILE_LIMIT || nr64 > RT_TILE_LIMIT) {
    if (threadIdx.x == 0) { atomicMax(&mx->overflow, 1); if (MODE == 0) { tsize[t] = 0; xcnt[t] = 0; icnt[t] = 0; n2cnt[t] = 0; } }
    return;
  }
  const int nown = (int)nown64, nr = (int)nr64;
  if (threadIdx.x == 0) { s_nc = 0; s_run = 0; s_bnd = 0; }
  __syncthreads();
  // incoming faces: r-list entries whose owner lies in an earlier tile, ranked in r-list order
  for (int k0 = 0; k0 < nr; k0 += TILE_BT) {
    const int k = k0 + threadIdx.x;
    const int flag = k < nr && rn[rbase + k] < c0;
    int pos, tot;
    Scan(scan_tmp).ExclusiveSum(flag, pos, tot);
    const int base = s_run;
    if (k < nr) s_rank[k] = flag ? base + pos : -1;
    __syncthreads();
    if (threadIdx.x == 0) s_run = base + tot;
    __syncthreads();
  }
  const int ninc = s_run;
  // halo candidates: the far cell of every face that leaves the tile
  for (int s = threadIdx.x; s < nown; s += TILE_BT) {
    const int32_t r = R[fbase + s];
    if (r >= c1) { const int p = atomicAdd(&s_nc, 1); if (p < RT_TILE_LIMIT) s_cand[p] = r; }
    if (r < 0) s_bnd = 1;  // a boundary face: the kernels take their ghost-state path for this tile
  }
  for (int k = threadIdx.x; k < nr; k += TILE_BT)
    if (s_rank[k] >= 0) { const int p = atomicAdd(&s_nc, 1); if (p < RT_TILE_LIMIT) s_cand[p] = rn[rbase + k]; }
  __syncthreads();
  const int nc = s_nc;
  if (nc > RT_TILE_LIMIT) {
    if (threadIdx.x == 0) { atomicMax(&mx->overflow, 1); if (MODE == 0) { tsize[t] = 0; xcnt[t] = 0; icnt[t] = 0; n2cnt[t] = 0; } }
    return;
  }
  int np2 = 1;
  while (np2 < nc) np2 <<= 1;
  for (int k = nc + threadIdx.x; k < np2; k += TILE_BT) s_cand[k] = 0x7fffffff;
  __syncthreads();
  for (int size = 2; size <= np2; size <<= 1)  // bitonic sort, ascending
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int k = threadIdx.x; k < np2; k += TILE_BT) {
        const int j = k ^ stride;
        if (j > k) {
          const int32_t a = s_cand[k], b = s_cand[j];
          const bool up = (k & size) == 0;
          if ((a > b) == up) { s_cand[k] = b; s_cand[j] = a; }
        }
      }
      __syncthreads();
    }
  if (threadIdx.x == 0) s_run = 0;
  __syncthreads();
  for (int k0 = 0; k0 < nc; k0 += TILE_BT) {  // unique
    const int k = k0 + threadIdx.x;
    const int flag = k < nc && (k == 0 || s_cand[k] != s_cand[k - 1]);
    int pos, tot;
    Scan(scan_tmp).ExclusiveSum(flag, pos, tot);
    const int base = s_run;
    if (flag) s_halo[base + pos] = s_cand[k];
    __syncthreads();
    if (threadIdx.x == 0) s_run = base + tot;
    __syncthreads();
  }
  const int nh = s_run, nhf = nown + nr, ns = nown + ninc;
  const int nb = halo_pos(s_halo, nh, (int32_t)c0);  // halo cells before the tile
  __syncthreads();
  // outgoing faces (right cell in a later tile), ranked in face order; s_cand is free again
  if (threadIdx.x == 0) s_run = 0;
  __syncthreads();
  for (int k0 = 0; k0 < nown; k0 += TILE_BT) {
    const int k = k0 + threadIdx.x;
    const int flag = k < nown && R[fbase + k] >= c1;
    int pos, tot;
    Scan(scan_tmp).ExclusiveSum(flag, pos, tot);
    const int base = s_run;
    if (k < nown) s_cand[k] = flag ? base + pos : -1;
    __syncthreads();
    if (threadIdx.x == 0) s_run = base + tot;
    __syncthreads();
  }
  const int nout = s_run;
  // cells with at least one incoming face ("incomplete": k_finish adds those fluxes), in cell
  // order; a cell's incoming faces have consecutive ranks
  __syncthreads();
  if (threadIdx.x == 0) s_run = 0;
  __syncthreads();
  for (int x0 = 0; x0 < ncell; x0 += TILE_BT) {
    const int x = x0 + threadIdx.x;
    int first = -1;
    if (x < ncell)
      for (int64_t k = ro[c0 + x]; k < ro[c0 + x + 1] && first < 0; k++) first = s_rank[k - rbase];
    const int flag = first >= 0;
    int pos, tot;
    Scan(scan_tmp).ExclusiveSum(flag, pos, tot);
    const int base = s_run;
    if (MODE == 1 && flag) {
      k2cell[k2base[t] + base + pos] = (int32_t)(c0 + x);
      k2off[k2base[t] + base + pos] = (int32_t)(ibase[t] + first);
    }
    __syncthreads();
    if (threadIdx.x == 0) s_run = base + tot;
    __syncthreads();
  }
  const int n2 = s_run;
  const int words = rt_blob_words(TC, nhf, nown, nh, ninc, nout);
  if (MODE == 0) {
    if (threadIdx.x == 0) {
      tsize[t] = words; xcnt[t] = nout; icnt[t] = ninc; n2cnt[t] = n2;
      atomicMax(&mx->ns, ns); atomicMax(&mx->no, nown); atomicMax(&mx->nh, nh); atomicMax(&mx->nf, nh - nb); atomicMax(&mx->words, words);
      if (TC + nh >= 0xFF00 || ns > 0x7fff) atomicMax(&mx->overflow, 1);
    }
    return;
  }
  if (threadIdx.x == 0) {
    rt_tile d;
    d.fbase = fbase; d.blob = t * bstride; d.xbase = xoff[t]; d.nown = nown; d.ninc = ninc; d.nh = nh; d.nhf = nhf;
    d.nb = nb; d.nout = nout; d.n2 = n2; d.pad = s_bnd;
    tiles[t] = d;
    *reinterpret_cast<rt_tile *>(blob + t * bstride) = d;  // the blob starts with a copy of the descriptor
    if (t == (int64_t)gridDim.x - 1) k2off[k2base[t] + n2] = (int32_t)(ibase[t] + ninc);  // end of the last cell's rows
  }
  __syncthreads();
  uint32_t *ho = blob + t * bstride + RT_BLOB_HEAD, *hl = ho + TC + 1, *slr = hl + nhf, *halo = slr + nown, *incf = halo + nh;
  uint32_t *outs = incf + ninc;
  for (int k = threadIdx.x; k < nown; k += TILE_BT)
    if (s_cand[k] >= 0) { outs[s_cand[k]] = (uint32_t)k; faceX[fbase + k] = (int32_t)(xoff[t] + s_cand[k]); }
  auto local_of = [&](int32_t id) -> uint32_t {  // id >= 0
    return id >= c0 && id < c1 ? (uint32_t)(id - c0) : (uint32_t)(TC + halo_pos(s_halo, nh, id));
  };
  for (int x = threadIdx.x; x <= TC; x += TILE_BT) {
    const int64_t i = c0 + (x < ncell ? x : ncell);
    ho[x] = (uint32_t)((fo[i] - fbase) + (ro[i] - rbase));
  }
  for (int x = threadIdx.x; x < ncell; x += TILE_BT) {
    const int64_t i = c0 + x;
    uint32_t *h = hl + (fo[i] - fbase) + (ro[i] - rbase);
    for (int64_t q = fo[i]; q < fo[i + 1]; q++) {  // owned slots: left = this cell
      const int32_t r = R[q];
      const uint32_t nbr = r >= 0 ? local_of(r) : (uint32_t)(0x10000 + r);
      *h++ = (nbr << 16) | (uint32_t)(q - fbase);
      slr[q - fbase] = (nbr << 16) | (uint32_t)x;
    }
    for (int64_t k = ro[i]; k < ro[i + 1]; k++) {
      const int rk = s_rank[k - rbase];
      const uint32_t slot = rk >= 0 ? (uint32_t)(nown + rk) : (uint32_t)(rl[k] - fbase);
      *h++ = (local_of(rn[k]) << 16) | 0x8000u | slot;
      if (rk >= 0) incf[rk] = (uint32_t)rl[k];
    }
  }
  for (int k = threadIdx.x; k < nh; k += TILE_BT) halo[k] = (uint32_t)s_halo[k];
  for (int k = TC + 1 + nhf + nown + nh + ninc + nout + threadIdx.x; k < words; k += TILE_BT) ho[k] = 0;
}

// k2row: the xphi row of every incoming face, tile by tile in rank order (= cell by cell)
__global__ void __launch_bounds__(TILE_BT) k_tile_rows(int TC, const rt_tile *tiles, const uint32_t *blob, const int64_t *ibase,
                                                       const int32_t *faceX, int32_t *k2row) {
  const rt_tile d = tiles[blockIdx.x];
  const uint32_t *incf = blob + d.blob + RT_BLOB_HEAD + TC + 1 + d.nhf + d.nown + d.nh;
  for (int j = threadIdx.x; j < d.ninc; j += TILE_BT) k2row[ibase[blockIdx.x] + j] = faceX[incf[j]];
}

// per tile: the four sizes that decide its shared-memory need
__global__ void k_tile_sizes(int64_t T, const rt_tile *tiles, int32_t *nown, int32_t *nf, int32_t *ns, int32_t *nh) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= T) return;
  const rt_tile d = tiles[t];
  nown[t] = d.nown; nf[t] = d.nh - d.nb; ns[t] = d.nown + d.ninc; nh[t] = d.nh;
}
// flag[t] = tile fits both capacities (inv: the opposite)
__global__ void k_tile_fits(int64_t T, const int32_t *a, const int32_t *b, int capa, int capb, int inv, uint8_t *flag) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= T) return;
  const int fits = a[t] <= capa && b[t] <= capb;
  flag[t] = (uint8_t)(inv ? !fits : fits);
}

__global__ void k_tile_totals(int64_t T, const rt_tile *tiles, unsigned long long *tot) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= T) return;
  atomicAdd(tot, (unsigned long long)tiles[t].ninc);
  atomicAdd(tot + 1, (unsigned long long)tiles[t].nh);
}

static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

int rt_setup_mesh(rt_ctx *c, const rt_mesh *m) {
  const int64_t C = c->C, F = c->F;
  const rt_layout &lay = c->lay;
  cudaStream_t st = c->stream;
  // carve the scratch region
  size_t o = lay.temp;
  auto take = [&](size_t bytes) { size_t r = o; o = align256(o + bytes); return r; };
  const int64_t NM = (C > F ? C : F) > 4 * (lay.max_tiles + 2) ? (C > F ? C : F) : 4 * (lay.max_tiles + 2);
  uint64_t *k0 = rt_ptr<uint64_t>(c, take(8 * NM)), *k1 = rt_ptr<uint64_t>(c, take(8 * NM));
  int32_t *v0 = rt_ptr<int32_t>(c, take(4 * NM)), *v1 = rt_ptr<int32_t>(c, take(4 * NM));
  // left / right ids of the sorted faces and the right lists: only the setup needs them
  int32_t *L = rt_ptr<int32_t>(c, take(4 * F)), *R = rt_ptr<int32_t>(c, take(4 * F));
  int32_t *rl = rt_ptr<int32_t>(c, take(4 * F)), *rn = rt_ptr<int32_t>(c, take(4 * F));
  double *cellS = rt_ptr<double>(c, take(32 * C));  // (centroid, V) in the new order: the kernels keep only V
  int *flags = rt_ptr<int>(c, take(256));
  size_t cub_bytes = 0;
  {
    cub::DoubleBuffer<uint64_t> dk(k0, k1);
    cub::DoubleBuffer<int32_t> dv(v0, v1);
    size_t b1 = 0, b2 = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, b1, dk, dv, NM, 0, 64, st);
    cub::DeviceRadixSort::SortKeys(nullptr, b2, dk, NM, 0, 64, st);
    size_t b3 = 0;
    cub::DeviceScan::ExclusiveSum(nullptr, b3, (int64_t *)nullptr, (int64_t *)nullptr, NM + 1, st);
    cub_bytes = b1 > b2 ? b1 : b2;
    if (b3 > cub_bytes) cub_bytes = b3;
  }
  void *cub_tmp = rt_ptr<void>(c, take(cub_bytes));
  geom_in g;
  if (m->mem_kind == RT_MEM_HOST) {
    double *dv = rt_ptr<double>(c, take(8 * C)), *dc = rt_ptr<double>(c, take(24 * C));
    double *da = rt_ptr<double>(c, take(8 * F)), *dn = rt_ptr<double>(c, take(24 * F)), *df = rt_ptr<double>(c, take(24 * F));
    int32_t *dl = rt_ptr<int32_t>(c, take(4 * F)), *dr = rt_ptr<int32_t>(c, take(4 * F));
    if (o > c->ws_bytes) return rt_fail(c, RT_ENOMEM, "workspace too small for host-mesh staging");
    RT_CUDA(c, cudaMemcpyAsync(dv, m->volume, 8 * C, cudaMemcpyHostToDevice, st));
    RT_CUDA(c, cudaMemcpyAsync(dc, m->centroid, 24 * C, cudaMemcpyHostToDevice, st));
    RT_CUDA(c, cudaMemcpyAsync(da, m->area, 8 * F, cudaMemcpyHostToDevice, st));
    RT_CUDA(c, cudaMemcpyAsync(dn, m->normal, 24 * F, cudaMemcpyHostToDevice, st));
    RT_CUDA(c, cudaMemcpyAsync(df, m->fcentroid, 24 * F, cudaMemcpyHostToDevice, st));
    RT_CUDA(c, cudaMemcpyAsync(dl, m->left, 4 * F, cudaMemcpyHostToDevice, st));
    RT_CUDA(c, cudaMemcpyAsync(dr, m->right, 4 * F, cudaMemcpyHostToDevice, st));
    g = {dv, dc, da, dn, df, dl, dr};
  } else {
    g = {m->volume, m->centroid, m->area, m->normal, m->fcentroid, m->left, m->right};
  }
  if (o > c->ws_bytes) return rt_fail(c, RT_ENOMEM, "workspace too small for setup scratch");
  RT_CUDA(c, cudaMemsetAsync(flags, 0, sizeof(int), st));
  k_validate<<<nblk(NM), SETUP_BLOCK, 0, st>>>(g, C, F, m->nghost, flags);
  int hflags = 0;
  RT_CUDA(c, cudaMemcpyAsync(&hflags, flags, sizeof(int), cudaMemcpyDeviceToHost, st));
  RT_CUDA(c, cudaStreamSynchronize(st));
  if (hflags)
    return rt_fail(c, RT_EMESH, "mesh validation failed:%s%s%s%s%s%s", hflags & E_LEFT ? " left index out of range;" : "",
                   hflags & E_RIGHT ? " right index out of range or equal to left;" : "",
                   hflags & E_GHOST ? " Dirichlet ghost index >= nghost;" : "", hflags & E_VOL ? " volume <= 0;" : "",
                   hflags & E_AREA ? " area <= 0;" : "", hflags & E_NORMAL ? " normal not unit;" : "");
  int32_t *perm = rt_ptr<int32_t>(c, lay.perm), *iperm = rt_ptr<int32_t>(c, lay.iperm);
  // 1. cells along the Peano-Hilbert curve
  {
    k_cell_keys<<<nblk(C), SETUP_BLOCK, 0, st>>>(g.centroid, C, c->box[0], c->box[1], c->box[2], k0, v0);
    cub::DoubleBuffer<uint64_t> dk(k0, k1);
    cub::DoubleBuffer<int32_t> dv(v0, v1);
    size_t b = cub_bytes;
    RT_CUDA(c, cub::DeviceRadixSort::SortPairs(cub_tmp, b, dk, dv, C, 0, 63, st));
    RT_CUDA(c, cudaMemcpyAsync(perm, dv.Current(), 4 * C, cudaMemcpyDeviceToDevice, st));
    k_permute_cells<<<nblk(C), SETUP_BLOCK, 0, st>>>(g, C, perm, iperm, cellS, rt_ptr<double>(c, lay.cellV));
  }
  // 2. faces by owner
  double *faceC = rt_ptr<double>(c, lay.faceC), *faceN = rt_ptr<double>(c, lay.faceN);
  double *faceW = rt_ptr<double>(c, lay.faceW);
  int64_t *fo = rt_ptr<int64_t>(c, lay.fo), *ro = rt_ptr<int64_t>(c, lay.ro);
  {
    k_face_keys<<<nblk(F), SETUP_BLOCK, 0, st>>>(g, F, iperm, k0, v0);
    cub::DoubleBuffer<uint64_t> dk(k0, k1);
    cub::DoubleBuffer<int32_t> dv(v0, v1);
    size_t b = cub_bytes;
    RT_CUDA(c, cub::DeviceRadixSort::SortPairs(cub_tmp, b, dk, dv, F, 0, 64, st));
    k_gather_faces<<<nblk(F), SETUP_BLOCK, 0, st>>>(g, C, F, dv.Current(), dk.Current(), iperm, cellS, c->box[0], c->box[1],
                                                    c->box[2], c->per[0], c->per[1], c->per[2], faceC, faceN, L, R);
    k_lower_bounds<<<nblk(C + 1), SETUP_BLOCK, 0, st>>>(dk.Current(), F, C, fo);
  }
  // 3. right lists
  {
    k_rkeys<<<nblk(F), SETUP_BLOCK, 0, st>>>(R, F, k0);
    cub::DoubleBuffer<uint64_t> dk(k0, k1);
    size_t b = cub_bytes;
    RT_CUDA(c, cub::DeviceRadixSort::SortKeys(cub_tmp, b, dk, F, 0, 64, st));
    k_lower_bounds<<<nblk(C + 1), SETUP_BLOCK, 0, st>>>(dk.Current(), F, C, ro);
    int64_t NR = 0;
    RT_CUDA(c, cudaMemcpyAsync(&NR, ro + C, 8, cudaMemcpyDeviceToHost, st));
    RT_CUDA(c, cudaStreamSynchronize(st));
    c->NR = NR;
    if (NR > 0) k_rlist<<<nblk(NR), SETUP_BLOCK, 0, st>>>(dk.Current(), NR, L, rl, rn);
  }
  // 4. geometry of eq (15)
  k_face_geom<<<nblk(F), SETUP_BLOCK, 0, st>>>(C, F, cellS, faceC, faceN, L, R, c->box[0], c->box[1], c->box[2],
                                               c->per[0], c->per[1], c->per[2], faceW);
  k_cell_geom<<<nblk(C), SETUP_BLOCK, 0, st>>>(C, F, faceC, faceN, faceW, fo, ro, rl, rt_ptr<double>(c, lay.Minv), flags);
  RT_CUDA(c, cudaMemcpyAsync(&hflags, flags, sizeof(int), cudaMemcpyDeviceToHost, st));
  // 5. tiles: the largest tile size (from RT_TILE_CELLS, default 64, downwards) whose shared memory
  // lets RT_TILE_BLOCKS (default 2) thread blocks of k_flux share an SM; failing that, the largest
  // that fits one block
  {
    const int64_t Tmax = lay.max_tiles + 2;
    int64_t *tsize = (int64_t *)k0, *xcnt = tsize + Tmax, *icnt = xcnt + Tmax, *n2cnt = icnt + Tmax;
    int64_t *boff = (int64_t *)k1, *xoff = boff + Tmax, *ibase = xoff + Tmax, *k2base = ibase + Tmax;
    int32_t *faceX = v0;
    tile_max *mx = (tile_max *)(flags + 4);
    // (measured: with 3 groups on the Voronoi configs 32 cells per tile and three blocks of k_flux per
    // SM beat 40 cells and two; with one group (128^3 Cartesian) 96 cells beat 64 and equal 128)
    const int tc_default = c->G >= 2 ? 32 : 96;
    const int tc0 = c->tun.tile_cells > 0 ? c->tun.tile_cells : tc_default;
    const int nblocks = c->tun.tile_blocks > 0 ? c->tun.tile_blocks : 2;
    int best = 0;
    tile_max hm;
    memset(&hm, 0, sizeof hm);
    for (int pass = 0; pass < 2 && !best; pass++) {
      const size_t limit = pass == 0 ? (size_t)(233472 / nblocks - 1024 - 512) : RT_SMEM_MAX;
      for (int TC = tc0; TC >= RT_MIN_TILE; TC -= TC > 32 ? 8 : 4) {
        const int64_t T = (C + TC - 1) / TC;
        RT_CUDA(c, cudaMemsetAsync(mx, 0, sizeof(tile_max), st));
        k_tile_build<0><<<(unsigned)T, TILE_BT, 0, st>>>(C, TC, fo, ro, R, rl, rn, tsize, xcnt, icnt, n2cnt, mx, 0, nullptr,
                                                        nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr);
        RT_CUDA(c, cudaMemcpyAsync(&hm, mx, sizeof(tile_max), cudaMemcpyDeviceToHost, st));
        RT_CUDA(c, cudaStreamSynchronize(st));
        const int bs = (hm.words + RT_BLOB_HEAD + 3) & ~3;  // the blob stride the kernels will stage
        if (!hm.overflow && rt_smem_flux(TC, c->G, hm.no, hm.nf, bs) <= limit &&
            rt_smem_grad(TC, c->G, hm.ns, hm.nh, bs) <= (limit > RT_SMEM_TARGET ? limit : RT_SMEM_TARGET)) {
          best = TC;
          break;
        }
      }
    }
    if (!best) return rt_fail(c, RT_EMESH, "a cell has too many faces for one thread block's shared memory");
    c->TC = best; c->smax = hm.ns; c->omax = hm.no; c->hmax = hm.nh; c->fmax = hm.nf; c->bmax = hm.words;
    c->T = (C + best - 1) / best;
    // the count arrays hold the accepted tile size's values (the loop stops at the first fit)
    int64_t *cnt[4] = {tsize, xcnt, icnt, n2cnt}, *off[4] = {boff, xoff, ibase, k2base};
    for (int a = 0; a < 4; a++) {
      size_t b = cub_bytes;
      RT_CUDA(c, cudaMemsetAsync(cnt[a] + c->T, 0, 8, st));
      RT_CUDA(c, cub::DeviceScan::ExclusiveSum(cub_tmp, b, cnt[a], off[a], c->T + 1, st));
    }
    // blobs at a fixed stride, so that a kernel finds a tile's blob without reading its descriptor first
    c->bstride = (hm.words + RT_BLOB_HEAD + 3) & ~3;
    c->blob_words = (int64_t)c->bstride * c->T;
    RT_CUDA(c, cudaMemcpyAsync(&c->ninc, xoff + c->T, 8, cudaMemcpyDeviceToHost, st));
    RT_CUDA(c, cudaMemcpyAsync(&c->n2, k2base + c->T, 8, cudaMemcpyDeviceToHost, st));
    RT_CUDA(c, cudaStreamSynchronize(st));
    if ((size_t)c->blob_words * 4 > lay.blob_bytes)
      return rt_fail(c, RT_ENOMEM, "tile tables need %lld bytes, the workspace holds %zu", (long long)c->blob_words * 4,
                     lay.blob_bytes);
    if (c->ninc > lay.xcap)
      return rt_fail(c, RT_ENOMEM, "%lld faces cross tile boundaries, the workspace holds the fluxes of %lld: "
                     "size it with rt_workspace_bytes(..., flags | RT_WS_ALL_FACES_CROSS)",
                     (long long)c->ninc, (long long)lay.xcap);
    rt_tile *tiles = rt_ptr<rt_tile>(c, lay.tiles);
    uint32_t *blob = rt_ptr<uint32_t>(c, lay.blob);
    k_tile_build<1><<<(unsigned)c->T, TILE_BT, 0, st>>>(C, best, fo, ro, R, rl, rn, nullptr, nullptr, nullptr, nullptr, mx, c->bstride,
                                                       xoff, ibase, k2base, tiles, blob, faceX,
                                                       rt_ptr<int32_t>(c, lay.k2cell), rt_ptr<int32_t>(c, lay.k2off));
    k_tile_rows<<<(unsigned)c->T, TILE_BT, 0, st>>>(best, tiles, blob, ibase, faceX, rt_ptr<int32_t>(c, lay.k2row));
    // (tsize is dead after the scan: reuse its first words for the halo total)
    RT_CUDA(c, cudaMemsetAsync(tsize, 0, 16, st));
    k_tile_totals<<<nblk(c->T), SETUP_BLOCK, 0, st>>>(c->T, tiles, (unsigned long long *)tsize);
    int64_t tot[2] = {0, 0};
    RT_CUDA(c, cudaMemcpyAsync(tot, tsize, 16, cudaMemcpyDeviceToHost, st));
    RT_CUDA(c, cudaStreamSynchronize(st));
    c->nhalo = tot[1];
    // tile classes: most tiles are much smaller than the largest one, so the kernels run them with
    // smaller shared-memory capacities (a quantile of the sizes) and more blocks per SM; the few
    // others run in a second launch with the maxima
    {
      const int64_t T = c->T;
      int32_t *sz[4], *sorted[4];
      for (int a = 0; a < 4; a++) { sz[a] = (int32_t *)k0 + a * T; sorted[a] = (int32_t *)k1 + a * T; }
      k_tile_sizes<<<nblk(T), SETUP_BLOCK, 0, st>>>(T, tiles, sz[0], sz[1], sz[2], sz[3]);
      std::vector<int32_t> hs[4];
      for (int a = 0; a < 4; a++) {
        size_t b = cub_bytes;
        RT_CUDA(c, cub::DeviceRadixSort::SortKeys(cub_tmp, b, sz[a], sorted[a], (int)T, 0, 32, st));
        hs[a].resize((size_t)T);
        RT_CUDA(c, cudaMemcpyAsync(hs[a].data(), sorted[a], 4 * (size_t)T, cudaMemcpyDeviceToHost, st));
      }
      RT_CUDA(c, cudaStreamSynchronize(st));
      const double qs[] = {1.0, 0.9995, 0.999, 0.998, 0.995, 0.99, 0.985, 0.98, 0.97, 0.96, 0.95, 0.93, 0.9, 0.87, 0.84, 0.8, 0.75, 0.7};
      auto quant = [&](const std::vector<int32_t> &v, double q) {
        int64_t k = (int64_t)(q * (double)T + 0.999999) - 1;
        if (k < 0) k = 0;
        if (k >= T) k = T - 1;
        return (int)v[(size_t)k];
      };
      const bool classes = c->tun.tile_classes != 1;
      // k_flux: three blocks of 256 threads per SM is what its registers allow
      c->omaxA = c->omax; c->fmaxA = c->fmax;
      const size_t lim_flux = 233472 / 3 - 1024 - 512;
      if (classes && rt_smem_flux(best, c->G, c->omax, c->fmax, c->bstride) > lim_flux)
        for (double q : qs) {
          const int o = quant(hs[0], q), f = quant(hs[1], q);
          if (rt_smem_flux(best, c->G, o, f, c->bstride) <= lim_flux) { c->omaxA = o; c->fmaxA = f; break; }
        }
      // k_grad: six blocks, else five (off by default: measured no gain, its registers and the
      // shared-memory pipeline bound it before occupancy does); RT_GRAD_CLASSES=1 turns it on
      c->smaxA = c->smax; c->hmaxA = c->hmax;
      bool done = false;
      const bool gclasses = classes && (c->tun.variant & 1);
      for (int nb = 6; gclasses && nb >= 5 && !done; nb--) {
        const size_t lim = 233472 / nb - 1024 - 64;
        if (rt_smem_grad(best, c->G, c->smax, c->hmax, c->bstride) <= lim) break;
        for (double q : qs) {
          if (q < 0.95) break;
          const int s2 = quant(hs[2], q), h2 = quant(hs[3], q);
          if (rt_smem_grad(best, c->G, s2, h2, c->bstride) <= lim) { c->smaxA = s2; c->hmaxA = h2; done = true; break; }
        }
      }
      // lists: class-A tiles in ascending order, then the class-B tiles
      uint8_t *flag = (uint8_t *)v1;
      int *cnt = (int *)flags + 16;
      int32_t *lists[2] = {rt_ptr<int32_t>(c, lay.tlistF), rt_ptr<int32_t>(c, lay.tlistG)};
      const int32_t *sa[2] = {sz[0], sz[2]}, *sb[2] = {sz[1], sz[3]};
      const int capa[2] = {c->omaxA, c->smaxA}, capb[2] = {c->fmaxA, c->hmaxA};
      int64_t *nA[2] = {&c->nFA, &c->nGA};
      for (int k = 0; k < 2; k++) {
        int hcnt = 0;
        size_t b = cub_bytes;
        k_tile_fits<<<nblk(T), SETUP_BLOCK, 0, st>>>(T, sa[k], sb[k], capa[k], capb[k], 0, flag);
        RT_CUDA(c, cub::DeviceSelect::Flagged(cub_tmp, b, cub::CountingInputIterator<int32_t>(0), flag, lists[k], cnt, (int)T, st));
        RT_CUDA(c, cudaMemcpyAsync(&hcnt, cnt, sizeof(int), cudaMemcpyDeviceToHost, st));
        RT_CUDA(c, cudaStreamSynchronize(st));
        *nA[k] = hcnt;
        if (hcnt < T) {
          b = cub_bytes;
          k_tile_fits<<<nblk(T), SETUP_BLOCK, 0, st>>>(T, sa[k], sb[k], capa[k], capb[k], 1, flag);
          RT_CUDA(c, cub::DeviceSelect::Flagged(cub_tmp, b, cub::CountingInputIterator<int32_t>(0), flag, lists[k] + hcnt, cnt, (int)T, st));
        }
      }
      RT_CUDA(c, cudaStreamSynchronize(st));
    }
  }
  if (m->nghost > 0)
    RT_CUDA(c, cudaMemcpyAsync(rt_ptr<double>(c, lay.ghost), m->ghost_state, sizeof(double) * m->nghost * 4 * c->G,
                               cudaMemcpyHostToDevice, st));
  RT_CUDA(c, cudaStreamSynchronize(st));
  RT_CUDA(c, cudaGetLastError());
  if (hflags)
    return rt_fail(c, RT_EMESH, "mesh validation failed:%s%s",
                   hflags & E_CLOSURE ? " a cell is not closed (|sum s A n| > 1e-10 sum A);" : "",
                   hflags & E_MATRIX ? " singular gradient matrix;" : "");
  return RT_OK;
}

rt_layout rt_make_layout(int64_t C, int64_t F, int G, int flags) {
  rt_layout l;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o = align256(o + bytes); return r; };
  l.nbc = (C + RT_BLOCK - 1) / RT_BLOCK;
  l.max_tiles = (C + RT_MIN_TILE - 1) / RT_MIN_TILE;
  l.perm = take(4 * C); l.iperm = take(4 * C);
  l.cellV = take(8 * C + 64); l.Minv = take(48 * C);
  l.faceC = take(32 * F); l.faceN = take(32 * F); l.faceW = take(32 * F);
  l.fo = take(8 * (C + 1)); l.ro = take(8 * (C + 1));
  // tile tables: descriptors for the smallest tile size; blobs bounded by
  // sum_t (TC + 4) + half-faces (<= 2F) + slots (<= 2F) + halo (<= 2F) + incoming (<= F) words
  l.tiles = take(sizeof(rt_tile) * (size_t)(l.max_tiles + 1));
  l.blob_bytes = 4 * ((size_t)(6.5 * (double)F) + 2 * (size_t)C + 5 * (size_t)l.max_tiles + 2048);
  l.blob = take(l.blob_bytes);
  l.tlistG = take(4 * (size_t)(l.max_tiles + 1)); l.tlistF = take(4 * (size_t)(l.max_tiles + 1));
  // fluxes of the faces that cross tile boundaries, written by the owner tile (<= 56 % of the
  // faces; rt_mesh_upload fails with RT_ENOMEM on a mesh whose tiles need more)
  l.xcap = (flags & RT_WS_ALL_FACES_CROSS) ? F : (int64_t)(0.56 * (double)F) + 1024;
  l.xphi = take(32 * (size_t)G * (size_t)l.xcap);
  // cells with incoming faces and the xphi rows of those faces (k_finish)
  l.k2cell = take(4 * (size_t)C); l.k2off = take(4 * ((size_t)C + 1)); l.k2row = take(4 * (size_t)l.xcap);
  l.ghost = take(8 * 4 * RT_MAXG * 64);
  l.led = take(sizeof(rt_dev_ledger));
  l.temp = o;
  l.Ua = take(32 * (size_t)G * C); l.Ub = take(32 * (size_t)G * C);
  l.grad = take(96 * (size_t)G * C);
  l.pacc = take(32 * (size_t)G * C);  // partial flux sums of the cells with incoming faces
  l.xHII = take(8 * C); l.xHeII = take(8 * C); l.xHeIII = take(8 * C); l.eth = take(8 * C); l.nH = take(8 * C);
  l.kappa = take(8 * C);
  l.srcidx = take(4 * C + 64);  // (+ padding: the tile kernels copy whole 16-byte chunks)
  l.srcrate = take(8 * (size_t)G * 65536);
  // partial sums: chem absorbed [<= 4 nbc + 1][G]; per tile: floor, outflow, inflow [max_tiles][G] each
  l.part = take(8 * (size_t)G * ((4 * RT_CHEM_MAXPASS + 1) * l.nbc + 3 * l.max_tiles + (size_t)G * l.nbc + 64));
  // sub-stepping passes of the chemistry: carried (t, h, attempts), flags, two index lists, cub scratch
  l.cact = take((size_t)C + 64); l.tact = take((size_t)l.max_tiles + 64);  // active / touched flags per cell, per tile
  l.chem_t = take(8 * (size_t)C); l.chem_h = take(8 * (size_t)C); l.chem_att = take(4 * (size_t)C);
  l.chem_flag = take((size_t)C + 64); l.chem_list = take(8 * (size_t)C); l.chem_count = take(256);
  l.chem_cub_bytes = rt_chem_cub_bytes(C);
  l.chem_cub = take(l.chem_cub_bytes);
  l.scratch_end = o;
  // setup scratch aliases the state region; make sure it fits (incl. staging of a host mesh)
  int64_t NM = C > F ? C : F;
  const size_t staging = (flags & RT_WS_DEVICE_MESH) ? 0 : 88 * (size_t)F + 32 * (size_t)C;
  size_t need = 24 * (size_t)NM + 4096 + (size_t)(64 << 20) + 16 * (size_t)F + 32 * (size_t)C + staging + 32 * 256;
  if (l.temp + need > o) o = align256(l.temp + need);
  l.total = o;
  return l;
}
