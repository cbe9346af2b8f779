// Internal declarations of librt.so (not part of the ABI; see include/rt.h).
//
// Device data layout (all inside the caller's workspace, fp64, 256-byte aligned blocks).
//   cells in Peano-Hilbert order p = 0..C-1:   perm[p] = caller's id, iperm = inverse
//     cellS[C][4] = (sx, sy, sz, V); Minv[C][6] (symmetric inverse of sum_f A n n^T, eq (15))
//   faces sorted by owner (= left cell, the lower new id), then by right id, boundary faces last;
//   every face array is [F][4] doubles = one aligned 32-byte sector per face:
//     faceC = (cx, cy, cz, A)     centroid in the left cell's frame and area
//     faceN = (nx, ny, nz, L|R)   unit normal L -> R; the fourth slot holds the two int32 ids
//     faceW = (wx, wy, wz, L|R)   w = A d/|d|^2, d = s_R - s_L: prefactor of eq (15)'s second
//                                 term
//   cell -> faces: owned faces are the contiguous range fo[i]..fo[i+1]; the faces
//     where the cell is the right one are r-list entries ro[i]..ro[i+1] (ascending face id)
//   tiles: TC consecutive cells (a compact blob of the Hilbert curve) are one thread block's
//     work.  A tile's "slots" are its owned faces (slot s = face - fo[c0]) followed by its
//     incoming faces (right cell in the tile, owner in an earlier tile), listed in
//     incf[inco[t]..inco[t+1]].  hl[fo[i]+ro[i] ..] is cell i's half-face list: the slot of each of
//     its faces inside its tile (owned faces first; bit 15 set where the cell is the right one),
//     so a cell finds every one of its faces in the tile's shared-memory slot arrays.
//   state, cell-major so that a tile is one contiguous run:
//     Ua, Ub [C][G][4] = (N, Fx, Fy, Fz); grad [C][G][12] (field-major, then direction);
//     xHII, xHeII, xHeIII, eth, nH, kappa [C]
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <vector>
#include "rt.h"

#ifndef RT_BLOCK
#define RT_BLOCK 128
#endif
#define RT_CHEM_BLOCK 32  // one warp per block: a slow cell holds back 31 others, not 127
#define RT_REC 18        // doubles per (cell, group) row of U + gradients in shared memory (16 + 2 pad: bank spread)
#define RT_MIN_TILE 8     // smallest tile size rt_mesh_upload will fall back to

struct rt_dev_ledger {  // accumulators on the device (value + compensation)
  double acc[5][RT_MAXG][2];  // 0 absorbed, 1 outflow, 2 inflow_bc, 3 floor_added, 4 stored (value only)
  unsigned long long substeps_total, substeps_max, cells_hit_cap;
};

struct rt_layout {
  size_t perm, iperm, cellS, Minv, faceC, faceN, faceW, L, R, fo, ro, rl, rn, hl, incf, inco, ghost, led;
  size_t Ua, Ub, grad, xHII, xHeII, xHeIII, eth, nH, kappa, srcidx, srcrate, part, scratch_end;
  size_t temp;        // start of the setup-time scratch (aliases the state region)
  size_t total;
  int64_t nbc;        // blocks of RT_BLOCK cells (partial-sum rows of k_stored)
  int64_t max_tiles;  // tiles at the smallest tile size (sizes inco and the partial sums)
};

struct rt_ctx {
  int device;
  cudaStream_t stream;
  char err[512];
  int64_t C, F, NR;
  int G;
  int TC;             // cells per tile
  int64_t T;          // number of tiles
  int smax;           // largest slot count of any tile
  int hmax;           // largest half-face count of any tile
  int64_t ninc;       // total incoming faces over all tiles
  double box[3];
  int per[3];
  int nghost;
  char *ws;
  size_t ws_bytes;
  rt_layout lay;
  bool have_mesh, have_state;
  rt_params par;
  int nsrc;
  double src_total[RT_MAXG];
  double injected[RT_MAXG][2];  // host-side compensated sum
  int64_t nsub_done;
  int64_t launches;
  // optional per-kernel timing with CUDA events on the context's stream (rt_profile)
  bool prof_on;
  std::vector<cudaEvent_t> prof_ev;   // pairs (start, stop)
  std::vector<int> prof_cls;
  size_t prof_used;
};

enum { RT_K_CHEM = 0, RT_K_GRAD = 1, RT_K_FLUX = 2, RT_K_UPDATE = 3, RT_K_REDUCE = 4, RT_K_OTHER = 5, RT_K_NCLS = 6 };
void rt_prof_begin(rt_ctx *c, int cls);
void rt_prof_end(rt_ctx *c);

// dynamic shared memory of the two tile kernels (rt_transport.cu) for a tile of TC cells whose
// slot count is at most smax
// (hmax: most half-faces of any tile; the face-list tables are int[TC+1] and uint16[hmax])
static inline size_t rt_smem_tables(int TC, int hmax) { return ((size_t)4 * (TC + 1) + (size_t)2 * hmax + 15) & ~(size_t)15; }
static inline size_t rt_smem_grad(int TC, int G, int smax, int hmax) {
  return (size_t)64 * smax + (size_t)32 * TC * G + rt_smem_tables(TC, hmax);
}
static inline size_t rt_smem_stage(int TC, int G, int smax, int hmax) {
  const int per_slot = 32 * G > 64 ? 32 * G : 64;  // A*Phi of every group, or the staged face record before it
  return (size_t)per_slot * smax + (size_t)RT_REC * 8 * TC * G + (size_t)32 * TC + rt_smem_tables(TC, hmax);
}
#define RT_SMEM_MAX 232448     // 227 KB: the most one block may have on sm_100
#define RT_SMEM_TARGET 110000  // two blocks per SM

template <class T>
static inline T *rt_ptr(const rt_ctx *c, size_t off) { return (T *)(c->ws + off); }

rt_layout rt_make_layout(int64_t C, int64_t F, int G);

int rt_fail(rt_ctx *c, int code, const char *fmt, ...);
#define RT_CUDA(c, call)                                                                          \
  do {                                                                                            \
    cudaError_t e_ = (call);                                                                      \
    if (e_ != cudaSuccess) return rt_fail((c), RT_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

// rt_setup.cu
int rt_setup_mesh(rt_ctx *c, const rt_mesh *m);
// rt_kernels.cu
int rt_transport_configure(rt_ctx *c);  // after rt_setup_mesh: shared-memory opt-in of the tile kernels
int rt_launch_step(rt_ctx *c, double dt);
int rt_launch_gradients(rt_ctx *c, const double *U);
// dst[p*stride + r] = src[r*C + perm[p]]  /  dst[r*C + perm[p]] = src[p*stride + r], r < rows
int rt_launch_permute_in(rt_ctx *c, const double *src, double *dst, int rows, int stride);
int rt_launch_permute_out(rt_ctx *c, const double *src, double *dst, int rows, int stride);
int rt_launch_init_sources(rt_ctx *c, const int32_t *cell_dev, int nsrc);
int rt_launch_stored(rt_ctx *c);

// min-image of a difference (periodic dims only)
__host__ __device__ inline double rt_wrap(double d, double L, int per) { return per ? d - L * rint(d / L) : d; }
