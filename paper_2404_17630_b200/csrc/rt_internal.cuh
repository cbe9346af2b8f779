// Internal declarations of librt.so (not part of the ABI; see include/rt.h).
//
// Device data layout (all inside the caller's workspace, fp64, 256-byte aligned blocks).  Arrays
// that are gathered through an index (neighbour states, gradients, face fluxes, cell geometry) are
// packed so that one gather is one or a few 32-byte sectors ("array of small structs"); arrays
// that are only streamed are plain.
//   cells in Peano-Hilbert order p = 0..C-1:   perm[p] = caller's id, iperm = inverse
//     cellS[C][4] = (sx, sy, sz, V); Minv[C][6] (symmetric inverse of sum_f A n n^T, eq (15))
//   faces sorted by owner (= left cell, the lower new id), then by right id, boundary faces last:
//     faceC[F][4] = (cx, cy, cz, A)  centroid in the left cell's frame and area
//     faceN[F][3] = unit normal L -> R
//     faceW[F][3] = A d/|d|^2, d = s_R - s_L: prefactor of eq (15)'s second term
//     L[F], R[F]
//   cell -> faces: owned faces are the contiguous range fo[i]..fo[i+1]; faces where
//     the cell is the right one are listed in rl[ro[i]..ro[i+1]] (ascending face id), with the
//     cell across each of them (= L[rl[k]]) in rn[k]
//   state: Ua, Ub [G][C][4] = (N, Fx, Fy, Fz); grad [G][C][12] (field-major, then direction);
//     phi [G][F][4] = A * (Phi_N, Phi_F); xHII, xHeII, xHeIII, eth, nH, kappa [C]
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

struct rt_dev_ledger {  // accumulators on the device (value + compensation)
  double acc[5][RT_MAXG][2];  // 0 absorbed, 1 outflow, 2 inflow_bc, 3 floor_added, 4 stored (value only)
  unsigned long long substeps_total, substeps_max, cells_hit_cap;
};

struct rt_layout {
  size_t perm, iperm, cellS, Minv, faceC, faceN, faceW, L, R, fo, ro, rl, rn, ghost, led;
  size_t Ua, Ub, grad, phi, xHII, xHeII, xHeIII, eth, nH, kappa, srcidx, srcrate, part, scratch_end;
  size_t temp;        // start of the setup-time scratch (aliases the state region)
  size_t total;
  int64_t nbc, nbf;   // blocks over cells / faces (partial-sum rows)
};

struct rt_ctx {
  int device;
  cudaStream_t stream;
  char err[512];
  int64_t C, F, NR;
  int G;
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
int rt_launch_step(rt_ctx *c, double dt);
int rt_launch_gradients(rt_ctx *c, const double *U);
// dst[p*stride + r] = src[r*C + perm[p]]  /  dst[r*C + perm[p]] = src[p*stride + r], r < rows
int rt_launch_permute_in(rt_ctx *c, const double *src, double *dst, int rows, int stride);
int rt_launch_permute_out(rt_ctx *c, const double *src, double *dst, int rows, int stride);
int rt_launch_init_sources(rt_ctx *c, const int32_t *cell_dev, int nsrc);
int rt_launch_stored(rt_ctx *c);

// min-image of a difference (periodic dims only)
__host__ __device__ inline double rt_wrap(double d, double L, int per) { return per ? d - L * rint(d / L) : d; }
