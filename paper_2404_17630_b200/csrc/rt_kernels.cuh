// Kernel-side parameter blocks and launch wrappers shared by the .cu files of librt.so.
#pragma once
#include "rt_internal.cuh"

struct rt_chem_par {
  double ctilde, y_he, T_fixed, alphaB_override, f_accept, f_target, x_floor_rel;
  long long max_substeps;
  double sigma[RT_MAXG][3], eps[RT_MAXG][3];
};

// geometry + box block passed by value to the transport kernels
struct rt_geom {
  int64_t C, F;
  const double *cellS, *Minv, *faceC, *faceN, *faceW;
  const int32_t *L, *R, *rl, *rn;
  const int64_t *fo, *ro;
  const double *ghost;
  double box[3];
  int per[3];
  int G;
};

void rt_launch_chem(rt_ctx *c, const rt_chem_par &P, double dt, double *U);
rt_geom rt_geom_of(const rt_ctx *c);
