// a1: per-cell thermochemistry over one subcycle (PAPER.md:125-127 semi-implicit scheme,
// PAPER.md:236-238 adaptive sub-stepping on the GPU).  One thread per cell; the whole sub-step
// loop runs in registers with no main-memory access inside the iterations.
// Formulas: readings S17-S24 of DESIGN.md (the paper defers them to Kannan+19); rate fits:
// DESIGN.md appendix A.
#include <cub/cub.cuh>
#include <stdlib.h>
#include "rt_internal.cuh"
#include "rt_kernels.cuh"

#define KB_CGS 1.380649e-16
#define T_FLOOR 10.0

// 1/x for positive normal x: MUFU.RCP64H seed + two Newton steps (relative error ~1e-16), a sixth
// of the instructions of an IEEE division.  Used where the quotient feeds a controller decision or
// a quantity compared at 1e-10; the abundances themselves (x = n / n_H) keep the exact division so
// that x = 1 stays exactly 1.
__device__ __forceinline__ double rcp_pos(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  return fma(r, e, r);
}

struct rate_set {
  double aHII, aHeII, aHeIII;      // case-B recombination
  double bHI, bHeI, bHeII;         // collisional ionisation
  double cool_ion[3];              // cooling per n_e n_X for X = HII, HeII, HeIII (recombination + brems)
  double cool_neu[3];              // cooling per n_e n_X for X = HI, HeI, HeII (coll. ionisation + excitation)
};

// The fits are products of powers of T; every power is taken as exp(c log x) from ONE log T
// (log lambda_i = log(2 T_i) - log T), which costs a third of pow() and agrees with it to ~1e-14
// relative (|c log x| <= 40): far inside the parity tolerance, and the sub-step controller's
// decisions only differ where f sits within 1e-14 of its threshold.
// 2.753e-14 lam^1.5 / (1 + (lam/2.74)^0.407)^2.242
__device__ inline double recomb_fit(double loglam) {
  const double u = exp(0.407 * (loglam - 1.007957920399979));  // log 2.74
  return 2.753e-14 * exp(1.5 * loglam - 2.242 * log(1.0 + u));
}
// 3.435e-30 T lam^1.970 / (1 + (lam/2.250)^0.376)^3.720
__device__ inline double recomb_cool_fit(double T, double loglam) {
  const double u = exp(0.376 * (loglam - 0.8109302162163288));  // log 2.25
  return 3.435e-30 * T * exp(1.970 * loglam - 3.720 * log(1.0 + u));
}

template <bool THERMAL>
__device__ inline void eval_rates(double T, double aB_override, rate_set &r) {
  const double iT = rcp_pos(T), logT = log(T);
  // log(2 T_i) for T_HI = 157807, T_HeI = 285335, T_HeII = 631515 K
  const double llHI = 12.662275226919286 - logT, llHeI = 13.254566388120152 - logT, llHeII = 14.049024154019651 - logT;
  const double sq = sqrt(T), q = rcp_pos(1.0 + sqrt(T * 1.0e-5));
  const double eHI = exp(-157809.1 * iT), eHeI = exp(-285335.4 * iT), eHeII = exp(-631515.0 * iT);
  const double sqq = sq * q;
  r.aHII = aB_override > 0.0 ? aB_override : recomb_fit(llHI);
  r.aHeII = 1.26e-14 * exp(0.75 * llHeI);
  r.aHeIII = 2.0 * recomb_fit(llHeII);
  r.bHI = 5.85e-11 * sqq * eHI;
  r.bHeI = 2.38e-11 * sqq * eHeI;
  r.bHeII = 5.68e-12 * sqq * eHeII;
  if (THERMAL) {
    const double lt = logT * 0.43429448190325176;  // log10 T
    const double brem = 1.42e-27 * (1.1 + 0.34 * exp(-(5.5 - lt) * (5.5 - lt) * (1.0 / 3.0))) * sq;
    r.cool_ion[0] = recomb_cool_fit(T, llHI) + brem;
    r.cool_ion[1] = KB_CGS * T * r.aHeII + brem;
    r.cool_ion[2] = 8.0 * recomb_cool_fit(T, llHeII) + 4.0 * brem;
    r.cool_neu[0] = 1.27e-21 * sqq * eHI + 7.50e-19 * exp(-118348.0 * iT) * q;
    r.cool_neu[1] = 9.38e-22 * sqq * eHeI;
    r.cool_neu[2] = 4.95e-22 * sqq * eHeII + 5.54e-17 * exp(-0.397 * logT - 473638.0 * iT) * q;
  }
}

template <int G>
struct cell_state {
  double N[G], Fx[G], Fy[G], Fz[G], xHII, xHeII, xHeIII, e;
};
// what a trial sub-step proposes: the photon attenuation factors and the new chemistry state
template <int G>
struct trial_out {
  double inv[G], xHII, xHeII, xHeIII, e;
};

// one trial sub-step of size h from s into o; returns the controller's f (C1-C7)
template <int G, bool THERMAL>
__device__ inline double trial(const rt_chem_par &P, const cell_state<G> &s, double nH, double h, const rate_set &r,
                               trial_out<G> &o) {
  const double y = P.y_he, nHe = y * nH;
  const double xe = s.xHII + y * (s.xHeII + 2.0 * s.xHeIII);
  const double ne = nH * xe;
  const double nHI = nH * (1.0 - s.xHII), nHeI = nHe * (1.0 - s.xHeII - s.xHeIII), nHeII = nHe * s.xHeII;
  double pHI = 0.0, pHeI = 0.0, pHeII = 0.0, heat = 0.0;
#pragma unroll
  for (int g = 0; g < G; g++) {
    const double k0 = P.sigma[g][0] * nHI, k1 = P.sigma[g][1] * nHeI, k2 = P.sigma[g][2] * nHeII;
    const double k = k0 + k1 + k2;
    const double inv = rcp_pos(1.0 + h * P.ctilde * k);
    o.inv[g] = inv;
    if (k > 0.0) {
      const double dNk = (s.N[g] - s.N[g] * inv) * rcp_pos(k);
      const double a0 = dNk * k0, a1 = dNk * k1, a2 = dNk * k2;
      pHI += a0; pHeI += a1; pHeII += a2;
      if (THERMAL) heat += a0 * P.eps[g][0] + a1 * P.eps[g][1] + a2 * P.eps[g][2];
    }
  }
  // hydrogen: backward Euler, n_e frozen
  double nHIIn = (nH * s.xHII + pHI + h * r.bHI * ne * nH) * rcp_pos(1.0 + h * ne * (r.bHI + r.aHII));
  nHIIn = fmin(fmax(nHIIn, 0.0), nH);
  o.xHII = nHIIn / nH;
  double nHeIn = 0.0, nHeIIn = 0.0, nHeIIIn = 0.0;
  if (nHe > 0.0) {
    const double hn = h * ne;
    const double a11 = 1.0 + hn * (r.bHeI + r.aHeII), a12 = hn * r.aHeII;
    const double a21 = hn * r.bHeII, a22 = 1.0 + hn * (r.aHeIII + r.bHeII);
    const double b1 = nHeI - pHeI + hn * r.aHeII * nHe;
    const double b2 = nHe * s.xHeIII + pHeII + hn * r.bHeII * nHe;
    const double idet = rcp_pos(a11 * a22 - a12 * a21);
    double a = (b1 * a22 - a12 * b2) * idet, c = (a11 * b2 - a21 * b1) * idet;
    a = fmin(fmax(a, 0.0), nHe);
    c = fmin(fmax(c, 0.0), nHe - a);
    nHeIn = a; nHeIIIn = c; nHeIIn = nHe - a - c;
    o.xHeII = nHeIIn / nHe; o.xHeIII = nHeIIIn / nHe;
  } else { o.xHeII = s.xHeII; o.xHeIII = s.xHeIII; }
  double f = 0.0;
  if (THERMAL) {
    const double xen = o.xHII + y * (o.xHeII + 2.0 * o.xHeIII);
    const double nen = nH * xen;
    const double lam = nen * (r.cool_ion[0] * nHIIn + r.cool_ion[1] * nHeIIn + r.cool_ion[2] * nHeIIIn +
                              r.cool_neu[0] * (nH - nHIIn) + r.cool_neu[1] * nHeIn + r.cool_neu[2] * nHeIIn);
    double en = s.e + heat - h * lam;
    en = fmax(en, 1.5 * nH * (1.0 + y + xen) * KB_CGS * T_FLOOR);
    o.e = en;
    f = fabs(en - s.e) * rcp_pos(s.e);
  } else o.e = s.e;
  const double fl = P.x_floor_rel;
  f = fmax(f, fabs(o.xHII - s.xHII) * rcp_pos(fmax(s.xHII, fl)));
  f = fmax(f, fabs((1.0 - o.xHII) - (1.0 - s.xHII)) * rcp_pos(fmax(1.0 - s.xHII, fl)));
  if (nHe > 0.0) {
    f = fmax(f, fabs(o.xHeII - s.xHeII) * rcp_pos(fmax(s.xHeII, fl)));
    f = fmax(f, fabs(o.xHeIII - s.xHeIII) * rcp_pos(fmax(s.xHeIII, fl)));
    f = fmax(f, fabs((1.0 - o.xHeII - o.xHeIII) - (1.0 - s.xHeII - s.xHeIII)) * rcp_pos(fmax(1.0 - s.xHeII - s.xHeIII, fl)));
  }
  return f;
}

// deterministic sum over the block's single warp (fixed tree), result valid in thread 0
__device__ inline double block_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}

// what a cell whose sub-stepping is not finished carries to the next pass (the cells
// that need many sub-steps are compacted and continued by later passes, so that a few slow cells
// do not hold back the warps of the fast ones)
struct chem_carry {
  double *t, *h;      // time reached, next sub-step (negative: it is the clipped last one)
  int32_t *attempts;  // trials so far
};

// One pass of the sub-stepping.  FIRST: every cell, starting at t = 0, h = dt; otherwise the cells
// list[0 .. *count) with the carried (t, h).  A cell stops after `cap` trials in this pass
// (cap <= 0: no limit) and is flagged for the next pass.  One warp per block; warps stride over the
// cells; part_abs has one row per 32 consecutive entries (fixed order: deterministic ledger).
template <int G, int MODE, bool FIRST>
__global__ void __launch_bounds__(RT_CHEM_BLOCK, 16) k_chem(rt_chem_par P, int64_t C, double dt, double *__restrict__ U,
                                                   double *__restrict__ xHII, double *__restrict__ xHeII,
                                                   double *__restrict__ xHeIII, double *__restrict__ eth,
                                                   const double *__restrict__ nHv, const double *__restrict__ cellV,
                                                   const double *__restrict__ kappa, double *__restrict__ part_abs,
                                                   rt_dev_ledger *led, const int32_t *__restrict__ list,
                                                   const int *__restrict__ count, int cap, chem_carry carry,
                                                   uint8_t *__restrict__ flag, const uint8_t *__restrict__ cact) {
  constexpr bool THERMAL = (MODE == RT_CHEM_HHE_THERMAL);
  static_assert(RT_CHEM_BLOCK == 32, "block_sum assumes one warp");
  const int64_t n = FIRST ? C : (int64_t)*count;
  unsigned long long wsum_att = 0, wmax_att = 0;
  int wcap = 0;
  for (int64_t row = blockIdx.x; row * RT_CHEM_BLOCK < n; row += gridDim.x) {
    const int64_t idx = row * RT_CHEM_BLOCK + threadIdx.x;
    // (individual time steps: a passive cell does no chemistry; only the first pass sees such cells)
    const bool live = idx < n && !(FIRST && cact && (cact[idx] & 5) != 1);  // (passive cells and ghosts do no chemistry)
    if (FIRST && flag && idx < n && !live) flag[idx] = 0;
    double absd[G];
#pragma unroll
    for (int g = 0; g < G; g++) absd[g] = 0.0;
    if (live) {
      const int64_t i = FIRST ? idx : (int64_t)list[idx];
      cell_state<G> s;
#pragma unroll
      for (int g = 0; g < G; g++) {
        const double4 u = *reinterpret_cast<const double4 *>(U + ((size_t)i * G + g) * 4);
        s.N[g] = u.x; s.Fx[g] = u.y; s.Fy[g] = u.z; s.Fz[g] = u.w;
        absd[g] = s.N[g];
      }
      bool unfinished = false;
      if (MODE == RT_CHEM_FIXED_OPACITY) {
        // one implicit step of the absorption terms of eqs (6)-(7): N' = N/(1 + dt c kappa)
        const double den = 1.0 + dt * P.ctilde * kappa[i];
#pragma unroll
        for (int g = 0; g < G; g++) { s.N[g] /= den; s.Fx[g] /= den; s.Fy[g] /= den; s.Fz[g] /= den; }
      } else {
        const double nH = nHv[i];
        s.xHII = xHII[i]; s.xHeII = xHeII[i]; s.xHeIII = xHeIII[i]; s.e = eth[i];
        rate_set r;
        if (!THERMAL) eval_rates<false>(P.T_fixed, P.alphaB_override, r);
        // controller of PAPER.md:238: start with h = dt; reject if f > 0.1 and shrink by f_s/f; on
        // accept scale by f_s/f but at most double; the last step is clipped to end at dt
        double t = 0.0, h = dt;
        bool last = true, stale = true;  // rates depend on the state only: a retry reuses them
        long long attempts = 0;
        if (!FIRST) {
          t = carry.t[i];
          h = carry.h[i];
          last = h < 0.0;
          h = fabs(h);
          attempts = carry.attempts[i];
        }
        int here = 0, capped = 0;
        bool done = false;
        while (true) {
          if (attempts >= P.max_substeps) { capped = 1; done = true; break; }
          if (cap > 0 && here >= cap) break;
          if (THERMAL && stale) {
            stale = false;
            const double xe = s.xHII + P.y_he * (s.xHeII + 2.0 * s.xHeIII);
            const double T = (2.0 / 3.0) * s.e * rcp_pos(KB_CGS * (nH * (1.0 + P.y_he + xe)));
            eval_rates<true>(T, P.alphaB_override, r);
          }
          trial_out<G> o;
          const double f = trial<G, THERMAL>(P, s, nH, h, r, o);
          attempts++; here++;
          if (!(f <= P.f_accept)) { h = h * P.f_target / f; last = false; continue; }  // (a NaN change is a reject: the cell then runs into the cap)
#pragma unroll
          for (int g = 0; g < G; g++) { s.N[g] *= o.inv[g]; s.Fx[g] *= o.inv[g]; s.Fy[g] *= o.inv[g]; s.Fz[g] *= o.inv[g]; }
          s.xHII = o.xHII; s.xHeII = o.xHeII; s.xHeIII = o.xHeIII; s.e = o.e;
          stale = true;
          if (last) { done = true; break; }
          t += h;
          h = h * fmin(2.0, P.f_target / fmax(f, 1e-300));
          if (h >= dt - t) { h = dt - t; last = true; }
        }
        xHII[i] = s.xHII; xHeII[i] = s.xHeII; xHeIII[i] = s.xHeIII;
        if (THERMAL) eth[i] = s.e;
        wsum_att += (unsigned long long)here;
        if (done) {
          wmax_att = (unsigned long long)attempts > wmax_att ? (unsigned long long)attempts : wmax_att;
          wcap += capped;
        } else {
          unfinished = true;
          carry.t[i] = t; carry.h[i] = last ? -h : h; carry.attempts[i] = (int32_t)attempts;
        }
      }
      if (flag) flag[idx] = unfinished ? 1 : 0;
      const double V = cellV[i];
#pragma unroll
      for (int g = 0; g < G; g++) {
        *reinterpret_cast<double4 *>(U + ((size_t)i * G + g) * 4) = make_double4(s.N[g], s.Fx[g], s.Fy[g], s.Fz[g]);
        absd[g] = V * (absd[g] - s.N[g]);
      }
    }
#pragma unroll
    for (int g = 0; g < G; g++) {
      const double tsum = block_sum(absd[g]);
      if (threadIdx.x == 0) part_abs[(size_t)row * G + g] = tsum;
    }
  }
  if (MODE != RT_CHEM_FIXED_OPACITY) {
    // integer counters: order-independent, so atomics keep the result deterministic
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      wsum_att += __shfl_down_sync(0xffffffffu, wsum_att, o);
      unsigned long long mm = __shfl_down_sync(0xffffffffu, wmax_att, o);
      wmax_att = mm > wmax_att ? mm : wmax_att;
      wcap += __shfl_down_sync(0xffffffffu, wcap, o);
    }
    if ((threadIdx.x & 31) == 0) {
      if (wsum_att) atomicAdd(&led->substeps_total, wsum_att);
      if (wmax_att) atomicMax(&led->substeps_max, wmax_att);
      if (wcap) atomicAdd(&led->cells_hit_cap, (unsigned long long)wcap);
    }
  }
}

// caps of the passes: rt_tuning.chem_caps = {1, 8} means pass 0 makes one trial per cell, pass 1 up to
// 8 more for the cells still unfinished, and a last pass finishes the rest (the default)
static int chem_caps(const rt_ctx *c, int *caps, int maxn) {
  int n = 0;
  for (; n < 6 && n < maxn && c->tun.chem_caps[n] > 0; n++) caps[n] = c->tun.chem_caps[n];
  if (n == 0) { caps[0] = 1; caps[1] = 8; n = 2; }
  return n;
}

template <int G, int MODE>
static void launch_chem_mode(rt_ctx *c, const rt_chem_par &P, double dt, double *U) {
  const rt_layout &l = c->lay;
  const int64_t C = c->C;
  const unsigned nrows = (unsigned)((C + RT_CHEM_BLOCK - 1) / RT_CHEM_BLOCK);
  double *part = rt_ptr<double>(c, l.part);
  rt_dev_ledger *led = rt_ptr<rt_dev_ledger>(c, l.led);
  chem_carry carry = {rt_ptr<double>(c, l.chem_t), rt_ptr<double>(c, l.chem_h), rt_ptr<int32_t>(c, l.chem_att)};
  uint8_t *flags = rt_ptr<uint8_t>(c, l.chem_flag);
  int32_t *lists[2] = {rt_ptr<int32_t>(c, l.chem_list), rt_ptr<int32_t>(c, l.chem_list) + C};
  int *count = rt_ptr<int>(c, l.chem_count);
#define CHEM_ARGS P, C, dt, U, rt_ptr<double>(c, l.xHII), rt_ptr<double>(c, l.xHeII), rt_ptr<double>(c, l.xHeIII), \
      rt_ptr<double>(c, l.eth), rt_ptr<double>(c, l.nH), rt_ptr<double>(c, l.cellV), rt_ptr<double>(c, l.kappa)
  int caps[8];
  const int ncap = MODE == RT_CHEM_FIXED_OPACITY ? 0 : chem_caps(c, caps, 8);
  // pass 0: every cell
  rt_prof_begin(c, RT_K_CHEM);
  const uint8_t *cact = c->has_active ? rt_ptr<uint8_t>(c, l.cact) : nullptr;
  k_chem<G, MODE, true><<<nrows, RT_CHEM_BLOCK, 0, c->stream>>>(CHEM_ARGS, part, led, nullptr, nullptr, ncap > 0 ? caps[0] : 0, carry,
                                                              ncap > 0 ? flags : nullptr, cact);
  rt_prof_end(c);
  c->launches++;
  rt_reduce2(c, {part, nrows, 1.0, 0, nullptr}, {part, nrows, 1.0, 0, nullptr}, 1);
  // later passes: compact the unfinished cells (order kept: deterministic), continue them
  unsigned grid = (unsigned)(c->nsm > 0 ? c->nsm : 148) * 32u;
  if (grid > nrows) grid = nrows;
  for (int p = 1; p <= ncap; p++) {
    size_t bytes = l.chem_cub_bytes;
    rt_prof_begin(c, RT_K_CHEM);
    if (p == 1)
      cub::DeviceSelect::Flagged(rt_ptr<void>(c, l.chem_cub), bytes, cub::CountingInputIterator<int32_t>(0), flags, lists[1], count,
                                 (int)C, c->stream);
    else
      cub::DeviceSelect::Flagged(rt_ptr<void>(c, l.chem_cub), bytes, lists[(p - 1) & 1], flags, lists[p & 1], count, (int)C,
                                 c->stream);
    cudaMemsetAsync(flags, 0, (size_t)C, c->stream);  // entries beyond the new count must not be selected again
    double *part_p = part + (size_t)p * G * nrows;
    k_chem<G, MODE, false><<<grid, RT_CHEM_BLOCK, 0, c->stream>>>(CHEM_ARGS, part_p, led, lists[p & 1], count, p < ncap ? caps[p] : 0,
                                                               carry, flags, nullptr);
    rt_prof_end(c);
    c->launches += 3;  // two kernels of the compaction + the pass
    rt_reduce2(c, {part_p, 0, 1.0, 0, count}, {part_p, 0, 1.0, 0, count}, 1);
  }
#undef CHEM_ARGS
}

template <int G>
static void launch_chem_g(rt_ctx *c, const rt_chem_par &P, double dt, double *U) {
  switch (c->par.chem_mode) {
    case RT_CHEM_FIXED_OPACITY: launch_chem_mode<G, RT_CHEM_FIXED_OPACITY>(c, P, dt, U); break;
    case RT_CHEM_H_ISOTHERMAL: launch_chem_mode<G, RT_CHEM_H_ISOTHERMAL>(c, P, dt, U); break;
    default: launch_chem_mode<G, RT_CHEM_HHE_THERMAL>(c, P, dt, U); break;
  }
}

size_t rt_chem_cub_bytes(int64_t C) {
  size_t bytes = 0;
  cub::DeviceSelect::Flagged(nullptr, bytes, (const int32_t *)nullptr, (const uint8_t *)nullptr, (int32_t *)nullptr, (int *)nullptr,
                             (int)C);
  return bytes + 256;
}

void rt_launch_chem(rt_ctx *c, const rt_chem_par &P, double dt, double *U) {
  if (c->nsm <= 0) {
    int n = 0;
    cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, c->device);
    c->nsm = n > 0 ? n : 1;
  }
  switch (c->G) {
    case 1: launch_chem_g<1>(c, P, dt, U); break;
    case 2: launch_chem_g<2>(c, P, dt, U); break;
    case 3: launch_chem_g<3>(c, P, dt, U); break;
    case 4: launch_chem_g<4>(c, P, dt, U); break;
    case 5: launch_chem_g<5>(c, P, dt, U); break;
    case 6: launch_chem_g<6>(c, P, dt, U); break;
    case 7: launch_chem_g<7>(c, P, dt, U); break;
    default: launch_chem_g<8>(c, P, dt, U); break;
  }
}
