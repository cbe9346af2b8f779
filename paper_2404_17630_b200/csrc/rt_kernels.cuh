// Kernel-side parameter blocks and launch wrappers shared by the .cu files of librt.so.
#pragma once
#include "rt_internal.cuh"

struct rt_chem_par {
  double ctilde, y_he, T_fixed, alphaB_override, f_accept, f_target, x_floor_rel;
  long long max_substeps;
  double sigma[RT_MAXG][3], eps[RT_MAXG][3];
};

// geometry + tile tables passed by value to the transport kernels (layout: rt_internal.cuh)
struct rt_geom {
  int64_t C, F;
  const double *cellV, *Minv, *faceC, *faceN, *faceW;
  const rt_tile *tiles;
  const uint32_t *blob;
  double *xphi;          // [ninc][G][4] fluxes of the faces that cross tile boundaries
  const double *ghost;
  const uint8_t *cact, *tact;  // active / touched flags per cell and per tile (rt_set_active), or null: all active
  double box[3];
  int per[3];
  int G, TC, smax, omax, hmax, fmax, bmax, bstride;
  const int32_t *tlist;  // the launch works on tiles tlist[tbase + blockIdx.x]
  int64_t tbase;
  int prefetch_tiles;    // the tile kernels ask L2 for the data of tile t + prefetch_tiles
  int variant;           // rt_tuning.variant
  unsigned long long *tl; // rt_debug_tile_timeline: 8 time stamps (ns) per tile of the flux kernel, or null
  // mixed precision (rt_params.mixed): the length unit l0, a power of two near the mean cell size
  double il0, l0sq;      // 1 / l0, l0^2 (products with them are formed in double, then rounded: exact, and safe in range)
};

void rt_launch_chem(rt_ctx *c, const rt_chem_par &P, double dt, double *U);  // all passes + their ledger reductions
size_t rt_chem_cub_bytes(int64_t C);
// acc[slot][g] += weight * sum_rows part[row][g]; nrows = ceil(*ncount / 32) if ncount is given
struct reduce_job { const double *part; int64_t nrows; double weight; int slot; const int *ncount; };
void rt_reduce2(rt_ctx *c, reduce_job a, reduce_job b, int njobs);
rt_geom rt_geom_of(const rt_ctx *c);
