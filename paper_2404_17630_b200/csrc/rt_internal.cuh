// Internal declarations of librt.so (not part of the ABI; see include/rt.h).
//
// Device data layout (all inside the caller's workspace, SoA, fp64, 256-byte aligned blocks):
//   cells in Peano-Hilbert order p = 0..C-1:   perm[p] = caller's id, iperm = inverse
//     vol[C], s[3][C], Minv[6][C] (symmetric inverse of sum_f A n n^T, eq (15))
//   faces sorted by owner (= left cell, the lower new id), then by right id, boundary faces last:
//     A[F], nrm[3][F], cf[3][F] (left frame), w[3][F] = A d/|d|^2 with d = s_R - s_L,
//     L[F], R[F]
//   cell -> faces: owned faces are the contiguous range fo[i]..fo[i+1]; faces where
//     the cell is the right one are listed in rl[ro[i]..ro[i+1]] (ascending face id)
//   state: Ua, Ub [G][4][C] (N, Fx, Fy, Fz), grad [G][12][C], phi [G][4][F], x*, eth, nH, kappa
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <vector>
#include "rt.h"

#define RT_BLOCK 128

struct rt_dev_ledger {  // accumulators on the device (value + compensation)
  double acc[5][RT_MAXG][2];  // 0 absorbed, 1 outflow, 2 inflow_bc, 3 floor_added, 4 stored (value only)
  unsigned long long substeps_total, substeps_max, cells_hit_cap;
};

struct rt_layout {
  size_t perm, iperm, vol, s, Minv, A, nrm, cf, w, L, R, fo, ro, rl, ghost, led;
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
int rt_launch_permute_in(rt_ctx *c, const double *src, double *dst, int rows);   // dst[r][p] = src[r][perm[p]]
int rt_launch_permute_out(rt_ctx *c, const double *src, double *dst, int rows);  // dst[r][perm[p]] = src[r][p]
int rt_launch_init_sources(rt_ctx *c, const int32_t *cell_dev, int nsrc);
int rt_launch_stored(rt_ctx *c);

// min-image of a difference (periodic dims only)
__host__ __device__ inline double rt_wrap(double d, double L, int per) { return per ? d - L * rint(d / L) : d; }
