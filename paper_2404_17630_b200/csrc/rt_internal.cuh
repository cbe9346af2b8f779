// Internal declarations of librt.so (not part of the ABI; see include/rt.h).
//
// Device data layout (all inside the caller's workspace, fp64, 256-byte aligned blocks).
//   cells in Peano-Hilbert order p = 0..C-1:   perm[p] = caller's id, iperm = inverse
//     cellV[C] = V; Minv[C][6] (symmetric inverse of sum_f A n n^T, eq (15))
//   faces sorted by owner (= left cell, the lower new id), then by right id, boundary faces last;
//   every face array holds 4 doubles per face, stored as two halves: [F][2] = components 0-1, then
//   [F][2] = components 2-3, so that consecutive faces (and scattered ones) are read as 16-byte
//   chunks at a 16-byte stride, which spread over all shared-memory banks (32-byte records read by
//   one lane each collide two-way at best):
//     faceC = (cx, cy | cz, A)     centroid relative to the left cell's centroid (min-image) and area
//     faceN = (nx, ny | nz, 0)     unit normal L -> R
//     faceW = (wx, wy | wz, kappa) w = A d/|d|^2, d = s_R - s_L: prefactor of eq (15)'s second
//                                  term; kappa = |d|^2/A, so the face centroid relative
//                                  to the right cell is c - kappa w
//   cell -> faces: owned faces are the contiguous range fo[i]..fo[i+1]; the faces
//     where the cell is the right one are r-list entries ro[i]..ro[i+1] (ascending face id)
//   tiles: TC consecutive cells (a compact blob of the Hilbert curve) are one thread block's
//     work.  A tile's "slots" are its owned faces (slot s = face - fo[c0]) followed by its
//     incoming faces (right cell in the tile, owner in an earlier tile).  Its "halo" is the sorted
//     list of the cells outside the tile that touch one of its slots; a cell of the tile has the
//     local id x = i - c0, halo cell k the local id TC + k.  Per tile one descriptor (rt_tile) and
//     one contiguous blob of 32-bit words (16-byte aligned, a whole number of 16-byte chunks):
//       ho[TC+1]   offset of each cell's half-face list inside hl
//       hl[nhf]    half-faces, cell by cell, owned faces first:
//                    bits 0-14 slot, bit 15 set where the cell is the face's right cell,
//                    bits 16-31 local id of the cell across the face or a boundary code
//       slr[nown]  per owned slot: bits 0-15 local id of the left cell, bits 16-31 local id of the
//                    right cell or a boundary code (0x10000 + right, i.e. 0xFFFF outflow, 0xFFFE
//                    reflective, 0xFFFD - k Dirichlet ghost k); local ids stay below 0xFF00
//       halo[nh]   global ids of the halo cells, ascending: the first nb lie before the tile
//                  ("backward"), the others after it ("forward")
//       incf[ninc] global face ids of the incoming slots
//       outs[nout] the owned slots whose right cell lies in a later tile ("outgoing"), ascending;
//                  the tile writes their fluxes to rows xbase .. xbase + nout of xphi
//     so a thread block stages everything its tile touches in shared memory with asynchronous
//     copies and then computes from shared memory alone.  Every face's flux is evaluated once, by
//     the tile of its left cell (k_flux), which also updates the cells all of whose faces it has.
//     The other cells ("incomplete": k2cell[n2]) get the fluxes of their incoming faces from
//     xphi[ninc][G][4] in k_finish: rows k2row[k2off[k] .. k2off[k+1]] for cell k2cell[k].
//   state, cell-major so that a tile is one contiguous run:
//     Ua, Ub [C][G][4] = (N, Fx, Fy, Fz); grad [C][G][12] (field-major, then direction; with rt_params.mixed
//     the same region holds [C][G][12] floats: the gradients times the length unit l0, reading S28);
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
#define RT_CHEM_MAXPASS 8  // sub-stepping passes (rt_chem.cu): partial-sum rows are reserved for each
#define RT_RED_BLOCKS 64   // blocks per (job, group) of k_reduce
#define RT_CHEM_BLOCK 32  // one warp per block: a slow cell holds back 31 others, not 127
#define RT_REC 18        // doubles per (cell, group) row of U + gradients in shared memory (16 + 2 pad: bank spread)
#define RT_MIN_TILE 8     // smallest tile size rt_mesh_upload will fall back to

struct rt_dev_ledger {  // accumulators on the device (value + compensation)
  double acc[5][RT_MAXG][2];  // 0 absorbed, 1 outflow, 2 inflow_bc, 3 floor_added, 4 stored (value only)
  unsigned long long substeps_total, substeps_max, cells_hit_cap;
  // scratch of k_reduce: per (job, group) the chunk sums of its blocks and the count of blocks done
  double red_tmp[2][RT_MAXG][RT_RED_BLOCKS];
  unsigned red_cnt[2][RT_MAXG];
};

struct rt_layout {
  size_t perm, iperm, cellV, Minv, faceC, faceN, faceW, fo, ro, tiles, blob, tlistG, tlistF, xphi, k2cell, k2off, k2row, ghost, led;
  size_t chem_t, chem_h, chem_att, chem_flag, chem_list, chem_count, chem_cub, chem_cub_bytes;
  size_t Ua, Ub, grad, pacc, xHII, xHeII, xHeIII, eth, nH, kappa, srcidx, srcrate, part, cact, tact, scratch_end;
  size_t blob_bytes;  // capacity of the blob region
  int64_t xcap;       // rows [G][4] of xphi
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
  int hmax;           // largest halo (cells outside the tile touching it) of any tile
  int fmax;           // largest forward halo of any tile
  int omax;           // most owned faces of any tile
  int nsm;            // multiprocessors of the device (0 until first needed)
  // tiles in two classes per kernel: class A = the tiles that fit smaller shared-memory capacities
  // (more blocks per SM), class B = the others, sized by the maxima above.  tlist*: A tiles first.
  int64_t nGA, nFA;   // class-A tiles of k_grad / k_flux
  int smaxA, hmaxA;   // class-A capacities of k_grad
  int omaxA, fmaxA;   // class-A capacities of k_flux
  int64_t n2;         // cells with at least one incoming face
  int bmax;           // largest blob of any tile, in 32-bit words (without the header)
  int bstride;        // words between the blobs of consecutive tiles
  int64_t ninc;       // total incoming faces over all tiles
  int64_t nhalo;      // total halo cells over all tiles
  int64_t blob_words; // total blob size
  double box[3];
  int per[3];
  int nghost;
  double l0;          // mixed precision: length unit, the power of two next above the mean cell size cbrt(box volume / C)
  char *ws;
  size_t ws_bytes;
  rt_layout lay;
  bool have_mesh, have_state;
  rt_params par;
  rt_tuning tun;      // rt_set_tuning (zeros = defaults)
  bool has_active;    // rt_set_active gave a proper subset: cact / tact are valid
  int phase_next;     // rt_step_phase: the phase of the running subcycle that comes next (0 between subcycles)
  std::vector<int32_t> src_cell;  // host copies of the sources (rt_set_active recomputes the injection rate)
  std::vector<double> src_rate;
  unsigned long long *dbg_tl;  // device buffer of rt_debug_tile_timeline while it runs, else null
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

// one tile's descriptor (56 bytes)
struct rt_tile {
  int64_t fbase;  // first owned face = fo[c0]
  int64_t blob;   // first word of the tile's blob
  int64_t xbase;  // first row of xphi the tile publishes
  int32_t nown, ninc, nh, nhf;  // owned faces, incoming faces, halo cells, half-faces
  int32_t nb, nout, n2, pad;    // backward halo cells, outgoing faces, cells with incoming faces; pad: bit 0 = the tile has boundary faces
};
#define RT_BLOB_HEAD 16     // 32-bit words reserved for the descriptor copy at the start of a blob
static_assert(sizeof(rt_tile) <= 4 * RT_BLOB_HEAD, "the blob header must hold a whole descriptor");
#define RT_TILE_LIMIT 2048  // most owned faces / r-list entries / halo candidates of a tile the builder handles
__host__ __device__ static inline int rt_blob_words(int TC, int nhf, int nown, int nh, int ninc, int nout) {
  return (TC + 1 + nhf + nown + nh + ninc + nout + 3) & ~3;
}

// dynamic shared memory of the two tile kernels (rt_transport.cu) for tiles of TC cells with at
// most smax slots, hmax halo cells (k_grad) / forward halo cells (k_stage) and bmax blob words
static inline size_t rt_smem_grad(int TC, int G, int smax, int hmax, int bmax) {
  return (size_t)4 * bmax + (size_t)64 * smax + (size_t)(32 * G + 16) * (TC + hmax) + (size_t)48 * TC;  // cell rows padded by 16 bytes
}
static inline size_t rt_smem_flux(int TC, int G, int omax, int fmax, int bmax, bool mixed = false) {
  const int planes = G > 3 ? G : 3;  // three face records per slot, overwritten by A*Phi of every group
  const int NE = (TC + fmax + 1) & ~1;
  // per cell: U [G][4] doubles, gradients [G][12] doubles (floats in mixed precision), the volume
  return (size_t)4 * bmax + (size_t)32 * planes * omax + (size_t)((mixed ? 80 : 128) * G + 8) * NE + (size_t)16 * ((TC + 3) / 4) +
         (size_t)((NE + 15) & ~15);  // + the active / touched flags
}
#define RT_SMEM_MAX 232448     // 227 KB: the most one block may have on sm_100
#define RT_SMEM_TARGET 115000  // two blocks per SM (228 KB per SM, 1 KB reserved per block)

template <class T>
static inline T *rt_ptr(const rt_ctx *c, size_t off) { return (T *)(c->ws + off); }

rt_layout rt_make_layout(int64_t C, int64_t F, int G, int flags);

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
int rt_launch_phase(rt_ctx *c, double dt, int phase);  // one phase of a subcycle (rt_step_phase)
// buf[k][:] = field[iperm[cells[k]]][:] (pack) or the reverse; rows of row_bytes (a multiple of 16)
int rt_launch_halo(rt_ctx *c, bool pack, void *field, int row_bytes, int64_t n, const int32_t *cells_dev, void *buf_dev);
int rt_launch_gradients(rt_ctx *c, const double *U);
// dst[p*stride + r] = src[r*C + perm[p]]  /  dst[r*C + perm[p]] = src[p*stride + r], r < rows
int rt_launch_permute_in(rt_ctx *c, const double *src, double *dst, int rows, int stride);
int rt_launch_permute_out(rt_ctx *c, const double *src, double *dst, int rows, int stride);
int rt_launch_init_sources(rt_ctx *c, const int32_t *cell_dev, int nsrc);
int rt_launch_stored(rt_ctx *c);
// cact[p] = bit 0 active, bit 1 touched (active or sharing a face with an active cell); tact[t] = OR over the tile's cells
int rt_launch_active(rt_ctx *c, const uint8_t *active_dev);

// min-image of a difference (periodic dims only)
__host__ __device__ inline double rt_wrap(double d, double L, int per) { return per ? d - L * rint(d / L) : d; }
