// a2-a4: the transport kernels of one Heun stage.
//   k_grad    LPC lanes per (cell, group): second term of eq (15) over the cell's faces with the
//             stored per-face prefactors, lane-reduced by warp shuffles, multiplied by the stored
//             inverse matrix; second pass over the faces for the slope limiter
//
//   k_flux    one thread per (face, group): extrapolate both cells to the face centre, M1 closure,
//             global Lax-Friedrichs flux with signal speed c~, donor cap; the flux (times the face
//             area) is saved to memory, not scattered
//   k_update  LPC lanes per (cell, group): sum the saved fluxes over the cell's face list, add the
//             source, Heun combine, floor and |F| <= c~ N (S3, S11, S12)
// Packed layouts (rt_internal.cuh): U[g][C][4], grad[g][C][12], phi[g][F][4], cellS[C][4],
// faceC[F][4], faceN[F][3], faceW[F][3]: one gather = one or a few whole 32-byte sectors.
#include "rt_internal.cuh"
#include "rt_kernels.cuh"

#include <stdlib.h>
// lanes per (cell, group) in k_grad / k_update: tuned on config 3/4 (profiles/); RT_LPC_GRAD and
// RT_LPC_UPD in the environment override them for experiments
static int lpc_of(const char *name, int dflt) {
  const char *e = getenv(name);
  int v = e ? atoi(e) : dflt;
  return (v == 1 || v == 2 || v == 4 || v == 8) ? v : dflt;
}
static int lpc_grad() { static int v = lpc_of("RT_LPC_GRAD", 1); return v; }
static int lpc_upd() { static int v = lpc_of("RT_LPC_UPD", 1); return v; }

__device__ __forceinline__ double4 ld4(const double *p) { return *reinterpret_cast<const double4 *>(p); }
__device__ __forceinline__ void st4(double *p, double a, double b, double c, double d) {
  *reinterpret_cast<double4 *>(p) = make_double4(a, b, c, d);
}

template <int W>
__device__ __forceinline__ double lanes_sum(double v) {
#pragma unroll
  for (int o = W / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o, W);
  return v;
}
template <int W>
__device__ __forceinline__ double lanes_max(double v) {
#pragma unroll
  for (int o = W / 2; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o, W));
  return v;
}
template <int W>
__device__ __forceinline__ double lanes_min(double v) {
#pragma unroll
  for (int o = W / 2; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o, W));
  return v;
}

// neighbour or ghost state seen across a boundary face with right code `code` (S13)
__device__ __forceinline__ double4 ghost_for_gradient(int code, const double4 Ui, const double *n3,
                                                      const double *ghost, int G, int g) {
  if (code == RT_BC_OUTFLOW) return Ui;
  if (code == RT_BC_REFLECT) {
    const double p = 2.0 * (Ui.y * n3[0] + Ui.z * n3[1] + Ui.w * n3[2]);
    return make_double4(Ui.x, Ui.y - p * n3[0], Ui.z - p * n3[1], Ui.w - p * n3[2]);
  }
  return ld4(ghost + ((size_t)(RT_BC_DIRICHLET0 - code) * G + g) * 4);
}

template <int GG, int LPC>
__global__ void __launch_bounds__(RT_BLOCK *GG) k_grad(rt_geom m, const double *__restrict__ U,
                                                        double *__restrict__ grad) {
  constexpr int CPB = RT_BLOCK / LPC;  // cells per block
  const int64_t C = m.C;
  const int lane = threadIdx.x % LPC;
  const int64_t i = (int64_t)blockIdx.x * CPB + threadIdx.x / LPC;
  const int g = threadIdx.y;
  const bool live = i < C;
  const int64_t ic = live ? i : C - 1;  // dead lanes shadow the last cell (keeps shuffles uniform)
  const double *Ug = U + (size_t)4 * g * C;
  const double4 Ui = ld4(Ug + 4 * ic);
  double b[4][3], hi[4] = {Ui.x, Ui.y, Ui.z, Ui.w}, lo[4] = {Ui.x, Ui.y, Ui.z, Ui.w};
#pragma unroll
  for (int v = 0; v < 4; v++) b[v][0] = b[v][1] = b[v][2] = 0.0;
  const int64_t f0 = m.fo[ic], r0 = m.ro[ic];
  const int nown = (int)(m.fo[ic + 1] - f0), nr = (int)(m.ro[ic + 1] - r0);

  auto accumulate = [&](const double4 Uj, double wx, double wy, double wz) {
    const double d0 = Uj.x - Ui.x, d1 = Uj.y - Ui.y, d2 = Uj.z - Ui.z, d3 = Uj.w - Ui.w;
    b[0][0] += wx * d0; b[0][1] += wy * d0; b[0][2] += wz * d0;
    b[1][0] += wx * d1; b[1][1] += wy * d1; b[1][2] += wz * d1;
    b[2][0] += wx * d2; b[2][1] += wy * d2; b[2][2] += wz * d2;
    b[3][0] += wx * d3; b[3][1] += wy * d3; b[3][2] += wz * d3;
    hi[0] = fmax(hi[0], Uj.x); hi[1] = fmax(hi[1], Uj.y); hi[2] = fmax(hi[2], Uj.z); hi[3] = fmax(hi[3], Uj.w);
    lo[0] = fmin(lo[0], Uj.x); lo[1] = fmin(lo[1], Uj.y); lo[2] = fmin(lo[2], Uj.z); lo[3] = fmin(lo[3], Uj.w);
  };
  // first pass: sum_f w_f (phi_j - phi_i), min/max.  Owned faces: the cell is the left one.
#pragma unroll 2
  for (int k = lane; k < nown; k += LPC) {
    const int64_t q = f0 + k;
    const int32_t j = m.R[q];
    const double *w = m.faceW + 3 * q;
    const double wx = w[0], wy = w[1], wz = w[2];
    const double4 Uj = j >= 0 ? ld4(Ug + 4 * (int64_t)j) : ghost_for_gradient(j, Ui, m.faceN + 3 * q, m.ghost, m.G, g);
    accumulate(Uj, wx, wy, wz);
  }
  // faces where the cell is the right one: d = s_L - s_R, so the prefactor changes sign
#pragma unroll 2
  for (int k = lane; k < nr; k += LPC) {
    const int64_t q = m.rl[r0 + k];
    const int32_t j = m.rn[r0 + k];
    const double *w = m.faceW + 3 * q;
    const double wx = -w[0], wy = -w[1], wz = -w[2];
    accumulate(ld4(Ug + 4 * (int64_t)j), wx, wy, wz);
  }
#pragma unroll
  for (int v = 0; v < 4; v++) {
    b[v][0] = lanes_sum<LPC>(b[v][0]); b[v][1] = lanes_sum<LPC>(b[v][1]); b[v][2] = lanes_sum<LPC>(b[v][2]);
    hi[v] = lanes_max<LPC>(hi[v]); lo[v] = lanes_min<LPC>(lo[v]);
  }
  const double *Mi = m.Minv + 6 * ic;
  const double m00 = Mi[0], m01 = Mi[1], m02 = Mi[2], m11 = Mi[3], m12 = Mi[4], m22 = Mi[5];
  double gr[4][3];
#pragma unroll
  for (int v = 0; v < 4; v++) {
    gr[v][0] = m00 * b[v][0] + m01 * b[v][1] + m02 * b[v][2];
    gr[v][1] = m01 * b[v][0] + m11 * b[v][1] + m12 * b[v][2];
    gr[v][2] = m02 * b[v][0] + m12 * b[v][1] + m22 * b[v][2];
  }
  // second pass: extreme extrapolated increments at the face centres.  min_f (hi-phi)/D_f is
  // attained at the largest D_f (division is monotone), so only the extremes are kept.
  const double4 si = ld4(m.cellS + 4 * ic);
  double dmax[4] = {0, 0, 0, 0}, dmin[4] = {0, 0, 0, 0};
  auto extremes = [&](double rx, double ry, double rz) {
#pragma unroll
    for (int v = 0; v < 4; v++) {
      const double d = gr[v][0] * rx + gr[v][1] * ry + gr[v][2] * rz;
      dmax[v] = fmax(dmax[v], d); dmin[v] = fmin(dmin[v], d);
    }
  };
#pragma unroll 2
  for (int k = lane; k < nown; k += LPC) {
    const double4 c = ld4(m.faceC + 4 * (f0 + k));  // already in this cell's frame
    extremes(c.x - si.x, c.y - si.y, c.z - si.z);
  }
#pragma unroll 2
  for (int k = lane; k < nr; k += LPC) {
    const double4 c = ld4(m.faceC + 4 * (int64_t)m.rl[r0 + k]);
    extremes(rt_wrap(c.x - si.x, m.box[0], m.per[0]), rt_wrap(c.y - si.y, m.box[1], m.per[1]),
             rt_wrap(c.z - si.z, m.box[2], m.per[2]));
  }
#pragma unroll
  for (int v = 0; v < 4; v++) { dmax[v] = lanes_max<LPC>(dmax[v]); dmin[v] = lanes_min<LPC>(dmin[v]); }
  if (!live) return;
  // lane v scales and writes field v (3 doubles each: the cell's 96 bytes leave as one run)
  double *out = grad + ((size_t)g * C + i) * 12;
  const double Uiv[4] = {Ui.x, Ui.y, Ui.z, Ui.w};
#pragma unroll
  for (int v = 0; v < 4; v++) {
    if (v % LPC != lane) continue;
    double a = 1.0;
    if (dmax[v] > 0.0) a = fmin(a, (hi[v] - Uiv[v]) / dmax[v]);
    if (dmin[v] < 0.0) a = fmin(a, (lo[v] - Uiv[v]) / dmin[v]);
    out[3 * v] = a * gr[v][0]; out[3 * v + 1] = a * gr[v][1]; out[3 * v + 2] = a * gr[v][2];
  }
}

// N D.n for the M1 closure (S1), lab frame: D = (1-chi)/2 I + (3 chi - 1)/2 nF nF^T
__device__ __forceinline__ void pressure_dot_n(const double U[4], const double n[3], double ct, double out[3]) {
  const double f2n = U[1] * U[1] + U[2] * U[2] + U[3] * U[3];
  const double fn = sqrt(f2n);
  const double f = fmin(1.0, fn / fmax(ct * U[0], 1e-300));
  const double chi = (3.0 + 4.0 * f * f) / (5.0 + 2.0 * sqrt(4.0 - 3.0 * f * f));
  const double a = 0.5 * (1.0 - chi) * U[0];
  double bb = 0.0;
  if (f2n > 0.0) bb = 0.5 * (3.0 * chi - 1.0) * U[0] * (U[1] * n[0] + U[2] * n[1] + U[3] * n[2]) / f2n;
  out[0] = a * n[0] + bb * U[1]; out[1] = a * n[1] + bb * U[2]; out[2] = a * n[2] + bb * U[3];
}

// U_face = U_i + grad U_i . r  (linear extrapolation to the centre of the interface)
__device__ __forceinline__ void extrapolate(const double *__restrict__ Ug, const double *__restrict__ gg, int64_t i,
                                            double rx, double ry, double rz, bool second_order, double Uo[4]) {
  const double4 u = ld4(Ug + 4 * i);
  Uo[0] = u.x; Uo[1] = u.y; Uo[2] = u.z; Uo[3] = u.w;
  if (second_order) {
    const double *p = gg + 12 * i;
    const double4 a = ld4(p), b = ld4(p + 4), c = ld4(p + 8);
    Uo[0] += a.x * rx + a.y * ry + a.z * rz;
    Uo[1] += a.w * rx + b.x * ry + b.y * rz;
    Uo[2] += b.z * rx + b.w * ry + c.x * rz;
    Uo[3] += c.y * rx + c.z * ry + c.w * rz;
  }
}

template <int GG>
__global__ void __launch_bounds__(RT_BLOCK *GG) k_flux(rt_geom m, const double *__restrict__ U,
                                                        const double *__restrict__ grad, double *__restrict__ phi,
                                                        double ct, double dt, int second_order,
                                                        double *__restrict__ part_out, double *__restrict__ part_in) {
  __shared__ double sm_out[GG][RT_BLOCK / 32], sm_in[GG][RT_BLOCK / 32];
  const int64_t C = m.C, F = m.F;
  const int64_t q = (int64_t)blockIdx.x * RT_BLOCK + threadIdx.x;
  const int g = threadIdx.y;
  double b_out = 0.0, b_in = 0.0;
  if (q < F) {
    const double *Ug = U + (size_t)4 * g * C, *gg = grad + (size_t)12 * g * C;
    const int32_t l = m.L[q], r = m.R[q];
    const double4 fc = ld4(m.faceC + 4 * q);
    const double n[3] = {m.faceN[3 * q], m.faceN[3 * q + 1], m.faceN[3 * q + 2]};
    const double A = fc.w;
    const double4 sl = ld4(m.cellS + 4 * (int64_t)l);
    double UL[4], UR[4];
    double Vr = 0.0, Nr = 0.0;
    extrapolate(Ug, gg, l, fc.x - sl.x, fc.y - sl.y, fc.z - sl.z, second_order, UL);
    if (r >= 0) {
      const double4 sr = ld4(m.cellS + 4 * (int64_t)r);
      Vr = sr.w;
      extrapolate(Ug, gg, r, rt_wrap(fc.x - sr.x, m.box[0], m.per[0]), rt_wrap(fc.y - sr.y, m.box[1], m.per[1]),
                  rt_wrap(fc.z - sr.z, m.box[2], m.per[2]), second_order, UR);
      Nr = Ug[4 * (int64_t)r];
    } else if (r == RT_BC_OUTFLOW) { UR[0] = UR[1] = UR[2] = UR[3] = 0.0; }  // vacuum ghost
    else if (r == RT_BC_REFLECT) {
      const double p = 2.0 * (UL[1] * n[0] + UL[2] * n[1] + UL[3] * n[2]);
      UR[0] = UL[0]; UR[1] = UL[1] - p * n[0]; UR[2] = UL[2] - p * n[1]; UR[3] = UL[3] - p * n[2];
    } else {
      const double4 gs = ld4(m.ghost + ((size_t)(RT_BC_DIRICHLET0 - r) * m.G + g) * 4);
      UR[0] = gs.x; UR[1] = gs.y; UR[2] = gs.z; UR[3] = gs.w;
    }
    double PL[3], PR[3];
    pressure_dot_n(UL, n, ct, PL);
    pressure_dot_n(UR, n, ct, PR);
    double ph[4];
    ph[0] = 0.5 * ((UL[1] + UR[1]) * n[0] + (UL[2] + UR[2]) * n[1] + (UL[3] + UR[3]) * n[2]) - 0.5 * ct * (UR[0] - UL[0]);
    const double hc2 = 0.5 * ct * ct, hc = 0.5 * ct;
#pragma unroll
    for (int a = 0; a < 3; a++) ph[1 + a] = hc2 * (PL[a] + PR[a]) - hc * (UR[1 + a] - UL[1 + a]);
    // donor cap (S11): the donor cannot lose more photons than it holds through this face in dt;
    // only the number flux is clamped (continuous in the state; Phi_F is left alone)
    if (ph[0] > 0.0) {
      const double lim = Ug[4 * (int64_t)l] * sl.w / (dt * A);
      if (ph[0] > lim) ph[0] = lim;
    } else if (ph[0] < 0.0 && r >= 0) {
      const double lim = Nr * Vr / (dt * A);
      if (-ph[0] > lim) ph[0] = -lim;
    }
    st4(phi + ((size_t)g * F + q) * 4, A * ph[0], A * ph[1], A * ph[2], A * ph[3]);
    if (r == RT_BC_OUTFLOW) b_out = A * ph[0];
    else if (r <= RT_BC_DIRICHLET0) b_in = -A * ph[0];
  }
  // boundary ledgers: fixed-order block sums, one row per block
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    b_out += __shfl_down_sync(0xffffffffu, b_out, o);
    b_in += __shfl_down_sync(0xffffffffu, b_in, o);
  }
  if ((threadIdx.x & 31) == 0) { sm_out[g][threadIdx.x >> 5] = b_out; sm_in[g][threadIdx.x >> 5] = b_in; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double so = 0.0, si = 0.0;
    for (int k = 0; k < RT_BLOCK / 32; k++) { so += sm_out[g][k]; si += sm_in[g][k]; }
    part_out[(size_t)blockIdx.x * m.G + g] = so;
    part_in[(size_t)blockIdx.x * m.G + g] = si;
  }
}

template <int GG, int LPC>
__global__ void __launch_bounds__(RT_BLOCK *GG) k_update(rt_geom m, const double *Ucur, const double *U0,
                                                          const double *__restrict__ phi, double *Uout,
                                                          const int32_t *__restrict__ srcidx,
                                                          const double *__restrict__ srcrate, int nsrc, double ca,
                                                          double cb, double dt, double ct, double n_floor,
                                                          double *__restrict__ part_floor) {
  constexpr int CPB = RT_BLOCK / LPC;
  __shared__ double sm[GG][RT_BLOCK / 32];
  const int64_t C = m.C, F = m.F;
  const int lane = threadIdx.x % LPC;
  const int64_t i = (int64_t)blockIdx.x * CPB + threadIdx.x / LPC;
  const int g = threadIdx.y;
  const bool live = i < C;
  const int64_t ic = live ? i : C - 1;
  const double *pg = phi + (size_t)4 * g * F;
  double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
  const int64_t f0 = m.fo[ic], r0 = m.ro[ic];
  const int nown = (int)(m.fo[ic + 1] - f0), nr = (int)(m.ro[ic + 1] - r0);
#pragma unroll 2
  for (int k = lane; k < nown; k += LPC) {
    const double4 p = ld4(pg + 4 * (f0 + k));
    s0 += p.x; s1 += p.y; s2 += p.z; s3 += p.w;
  }
#pragma unroll 2
  for (int k = lane; k < nr; k += LPC) {
    const double4 p = ld4(pg + 4 * (int64_t)m.rl[r0 + k]);
    s0 -= p.x; s1 -= p.y; s2 -= p.z; s3 -= p.w;
  }
  s0 = lanes_sum<LPC>(s0); s1 = lanes_sum<LPC>(s1); s2 = lanes_sum<LPC>(s2); s3 = lanes_sum<LPC>(s3);
  double fl = 0.0;
  if (live && lane == 0) {
    const double V = m.cellS[4 * i + 3];
    double R[4] = {-s0 / V, -s1 / V, -s2 / V, -s3 / V};
    const int32_t si = srcidx[i];
    if (si >= 0) R[0] += srcrate[(size_t)g * nsrc + si] / V;  // isotropic source (S5)
    const size_t o = ((size_t)g * C + i) * 4;
    const double4 uc = ld4(Ucur + o), u0 = ld4(U0 + o);
    double Un[4] = {ca * u0.x + cb * (uc.x + dt * R[0]), ca * u0.y + cb * (uc.y + dt * R[1]),
                    ca * u0.z + cb * (uc.z + dt * R[2]), ca * u0.w + cb * (uc.w + dt * R[3])};
    if (Un[0] < n_floor) { fl = V * (n_floor - Un[0]); Un[0] = n_floor; }
    const double fn = sqrt(Un[1] * Un[1] + Un[2] * Un[2] + Un[3] * Un[3]), lim = ct * Un[0];
    if (fn > lim) { const double sc = lim / fn; Un[1] *= sc; Un[2] *= sc; Un[3] *= sc; }
    st4(Uout + o, Un[0], Un[1], Un[2], Un[3]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) fl += __shfl_down_sync(0xffffffffu, fl, o);
  if ((threadIdx.x & 31) == 0) sm[g][threadIdx.x >> 5] = fl;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int k = 0; k < RT_BLOCK / 32; k++) t += sm[g][k];
    part_floor[(size_t)blockIdx.x * m.G + g] = t;
  }
}

// acc[slot][g] += weight * sum_rows part[row][g]; one block per (array, g); fixed order.
struct reduce_job { const double *part; int64_t nrows; double weight; int slot; };
__global__ void __launch_bounds__(1024) k_reduce(reduce_job j0, reduce_job j1, int G, rt_dev_ledger *led) {
  __shared__ double sm[1024];
  const reduce_job j = blockIdx.y == 0 ? j0 : j1;
  const int g = blockIdx.x;
  double s = 0.0, c = 0.0;
  for (int64_t r = threadIdx.x; r < j.nrows; r += 1024) {  // Neumaier per thread
    const double x = j.part[(size_t)r * G + g];
    const double t = s + x;
    c += fabs(s) >= fabs(x) ? (s - t) + x : (x - t) + s;
    s = t;
  }
  sm[threadIdx.x] = s + c;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) sm[threadIdx.x] += sm[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    double *a = led->acc[j.slot][g];
    if (j.slot == 4) { a[0] = j.weight * sm[0]; a[1] = 0.0; }
    else {
      const double x = j.weight * sm[0], t = a[0] + x;
      a[1] += fabs(a[0]) >= fabs(x) ? (a[0] - t) + x : (x - t) + a[0];
      a[0] = t;
    }
  }
}

// stored photons per block: part[row][g] = sum_cells V N
template <int GG>
__global__ void __launch_bounds__(RT_BLOCK *GG) k_stored(int64_t C, int G, const double *__restrict__ U,
                                                          const double *__restrict__ cellS, double *__restrict__ part) {
  __shared__ double sm[GG][RT_BLOCK / 32];
  const int64_t i = (int64_t)blockIdx.x * RT_BLOCK + threadIdx.x;
  const int g = threadIdx.y;
  double v = i < C ? cellS[4 * i + 3] * U[((size_t)g * C + i) * 4] : 0.0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) sm[g][threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int k = 0; k < RT_BLOCK / 32; k++) t += sm[g][k];
    part[(size_t)blockIdx.x * G + g] = t;
  }
}

// caller's SoA rows <-> internal packed rows
__global__ void k_permute_in(int64_t C, int rows, int stride, const int32_t *__restrict__ perm,
                             const double *__restrict__ src, double *__restrict__ dst) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= C) return;
  const int32_t o = perm[p];
  for (int r = 0; r < rows; r++) dst[(size_t)p * stride + r] = src[(size_t)r * C + o];
}
__global__ void k_permute_out(int64_t C, int rows, int stride, const int32_t *__restrict__ perm,
                              const double *__restrict__ src, double *__restrict__ dst) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= C) return;
  const int32_t o = perm[p];
  for (int r = 0; r < rows; r++) dst[(size_t)r * C + o] = src[(size_t)p * stride + r];
}
__global__ void k_fill_i32(int64_t n, int32_t v, int32_t *a) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p < n) a[p] = v;
}
__global__ void k_set_sources(int nsrc, const int32_t *__restrict__ cell, const int32_t *__restrict__ iperm,
                              int32_t *__restrict__ srcidx) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k < nsrc) srcidx[iperm[cell[k]]] = k;
}

// ------------------------------------------------------------------ host-side launchers
static inline unsigned blocks_for(int64_t n, int per_block) { return (unsigned)((n + per_block - 1) / per_block); }
#define DISPATCH_G(Gv, KERNEL, grid, block, stream, ...)                                  \
  switch (Gv) {                                                                           \
    case 1: KERNEL(1)<<<grid, block, 0, stream>>>(__VA_ARGS__); break;                    \
    case 2: KERNEL(2)<<<grid, block, 0, stream>>>(__VA_ARGS__); break;                    \
    case 3: KERNEL(3)<<<grid, block, 0, stream>>>(__VA_ARGS__); break;                    \
    case 4: KERNEL(4)<<<grid, block, 0, stream>>>(__VA_ARGS__); break;                    \
    case 5: KERNEL(5)<<<grid, block, 0, stream>>>(__VA_ARGS__); break;                    \
    case 6: KERNEL(6)<<<grid, block, 0, stream>>>(__VA_ARGS__); break;                    \
    case 7: KERNEL(7)<<<grid, block, 0, stream>>>(__VA_ARGS__); break;                    \
    default: KERNEL(8)<<<grid, block, 0, stream>>>(__VA_ARGS__); break;                   \
  }
#define K_GRAD1(g) k_grad<g, 1>
#define K_GRAD2(g) k_grad<g, 2>
#define K_GRAD4(g) k_grad<g, 4>
#define K_GRAD8(g) k_grad<g, 8>
#define K_FLUX(g) k_flux<g>
#define K_UPD1(g) k_update<g, 1>
#define K_UPD2(g) k_update<g, 2>
#define K_UPD4(g) k_update<g, 4>
#define K_UPD8(g) k_update<g, 8>
#define K_STORED(g) k_stored<g>
#define DISPATCH_LPC(lpc, Gv, K1, K2, K4, K8, cells, block, stream, ...)                               \
  switch (lpc) {                                                                                       \
    case 1: DISPATCH_G(Gv, K1, blocks_for(cells, RT_BLOCK), block, stream, __VA_ARGS__); break;        \
    case 2: DISPATCH_G(Gv, K2, blocks_for(cells, RT_BLOCK / 2), block, stream, __VA_ARGS__); break;    \
    case 4: DISPATCH_G(Gv, K4, blocks_for(cells, RT_BLOCK / 4), block, stream, __VA_ARGS__); break;    \
    default: DISPATCH_G(Gv, K8, blocks_for(cells, RT_BLOCK / 8), block, stream, __VA_ARGS__); break;   \
  }

rt_geom rt_geom_of(const rt_ctx *c) {
  const rt_layout &l = c->lay;
  rt_geom m;
  m.C = c->C; m.F = c->F; m.G = c->G;
  m.cellS = rt_ptr<double>(c, l.cellS); m.Minv = rt_ptr<double>(c, l.Minv);
  m.faceC = rt_ptr<double>(c, l.faceC); m.faceN = rt_ptr<double>(c, l.faceN); m.faceW = rt_ptr<double>(c, l.faceW);
  m.L = rt_ptr<int32_t>(c, l.L); m.R = rt_ptr<int32_t>(c, l.R);
  m.rl = rt_ptr<int32_t>(c, l.rl); m.rn = rt_ptr<int32_t>(c, l.rn); m.fo = rt_ptr<int64_t>(c, l.fo); m.ro = rt_ptr<int64_t>(c, l.ro);
  m.ghost = rt_ptr<double>(c, l.ghost);
  for (int a = 0; a < 3; a++) { m.box[a] = c->box[a]; m.per[a] = c->per[a]; }
  return m;
}

int rt_launch_gradients(rt_ctx *c, const double *U) {
  DISPATCH_LPC(lpc_grad(), c->G, K_GRAD1, K_GRAD2, K_GRAD4, K_GRAD8, c->C, dim3(RT_BLOCK, c->G), c->stream, rt_geom_of(c),
               U, rt_ptr<double>(c, c->lay.grad));
  c->launches++;
  return RT_OK;
}

static void reduce2(rt_ctx *c, reduce_job a, reduce_job b, int njobs) {
  rt_prof_begin(c, RT_K_REDUCE);
  k_reduce<<<dim3(c->G, njobs), 1024, 0, c->stream>>>(a, b, c->G, rt_ptr<rt_dev_ledger>(c, c->lay.led));
  rt_prof_end(c);
  c->launches++;
}

// one Heun stage: Uout = ca*U0 + cb*(Uin + dt R(Uin)); ledger weights wl (fluxes), wf (floor)
static void stage(rt_ctx *c, const double *Uin, const double *U0, double *Uout, double ca, double cb, double dt,
                  double wl, double wf) {
  const rt_layout &l = c->lay;
  const rt_geom m = rt_geom_of(c);
  const int G = c->G;
  double *grad = rt_ptr<double>(c, l.grad), *phi = rt_ptr<double>(c, l.phi);
  double *part = rt_ptr<double>(c, l.part);
  const int64_t nbu = blocks_for(c->C, RT_BLOCK / lpc_upd());
  const int64_t nchem = blocks_for(c->C, RT_CHEM_BLOCK);
  double *p_floor = part + (size_t)G * nchem, *p_out = p_floor + (size_t)G * nbu, *p_in = p_out + (size_t)G * l.nbf;
  const int second = c->par.order >= 2;
  if (second) {
    rt_prof_begin(c, RT_K_GRAD);
    DISPATCH_LPC(lpc_grad(), G, K_GRAD1, K_GRAD2, K_GRAD4, K_GRAD8, c->C, dim3(RT_BLOCK, G), c->stream, m, Uin, grad);
    rt_prof_end(c);
    c->launches++;
  }
  rt_prof_begin(c, RT_K_FLUX);
  DISPATCH_G(G, K_FLUX, (unsigned)l.nbf, dim3(RT_BLOCK, G), c->stream, m, Uin, grad, phi, c->par.ctilde, dt, second, p_out,
             p_in);
  rt_prof_end(c);
  c->launches++;
  reduce2(c, {p_out, l.nbf, wl * dt, 1}, {p_in, l.nbf, wl * dt, 2}, 2);
  rt_prof_begin(c, RT_K_UPDATE);
  DISPATCH_LPC(lpc_upd(), G, K_UPD1, K_UPD2, K_UPD4, K_UPD8, c->C, dim3(RT_BLOCK, G), c->stream, m, Uin, U0, phi, Uout,
               rt_ptr<int32_t>(c, l.srcidx), rt_ptr<double>(c, l.srcrate), c->nsrc, ca, cb, dt, c->par.ctilde,
               c->par.n_floor, p_floor);
  rt_prof_end(c);
  c->launches++;
  reduce2(c, {p_floor, nbu, wf, 3}, {p_floor, nbu, wf, 3}, 1);
}

int rt_launch_step(rt_ctx *c, double dt) {
  rt_layout &l = c->lay;
  double *Ua = rt_ptr<double>(c, l.Ua), *Ub = rt_ptr<double>(c, l.Ub);
  if (c->par.chem_mode != RT_CHEM_NONE) {
    rt_chem_par P;
    P.ctilde = c->par.ctilde; P.y_he = c->par.y_he; P.T_fixed = c->par.T_fixed;
    P.alphaB_override = c->par.alphaB_override; P.f_accept = c->par.f_accept; P.f_target = c->par.f_target;
    P.x_floor_rel = c->par.x_floor_rel; P.max_substeps = c->par.max_substeps;
    for (int g = 0; g < RT_MAXG; g++)
      for (int j = 0; j < 3; j++) { P.sigma[g][j] = c->par.sigma[g][j]; P.eps[g][j] = c->par.eps_heat[g][j]; }
    rt_launch_chem(c, P, dt, Ua);
    const int64_t nchem = blocks_for(c->C, RT_CHEM_BLOCK);
    reduce2(c, {rt_ptr<double>(c, l.part), nchem, 1.0, 0}, {rt_ptr<double>(c, l.part), nchem, 1.0, 0}, 1);
  }
  double tot[RT_MAXG];
  for (int g = 0; g < c->G; g++) tot[g] = dt * c->src_total[g];
  if (c->par.heun) {
    stage(c, Ua, Ua, Ub, 0.0, 1.0, dt, 0.5, 0.5);  // U1 = enforce(Un + dt R(Un))
    stage(c, Ub, Ua, Ua, 0.5, 0.5, dt, 0.5, 1.0);  // Un+1 = enforce(Un/2 + (U1 + dt R(U1))/2)
  } else {
    stage(c, Ua, Ua, Ub, 0.0, 1.0, dt, 1.0, 1.0);
    size_t t = l.Ua; l.Ua = l.Ub; l.Ub = t;  // the new state lives in the other buffer
  }
  for (int g = 0; g < c->G; g++) {  // injected photons: host-side compensated sum
    double *a = c->injected[g];
    const double x = tot[g], t = a[0] + x;
    a[1] += fabs(a[0]) >= fabs(x) ? (a[0] - t) + x : (x - t) + a[0];
    a[0] = t;
  }
  c->nsub_done++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return rt_fail(c, RT_ECUDA, "kernel launch: %s", cudaGetErrorString(e));
  return RT_OK;
}

int rt_launch_stored(rt_ctx *c) {
  const rt_layout &l = c->lay;
  double *part = rt_ptr<double>(c, l.part);
  DISPATCH_G(c->G, K_STORED, (unsigned)l.nbc, dim3(RT_BLOCK, c->G), c->stream, c->C, c->G, rt_ptr<double>(c, l.Ua),
             rt_ptr<double>(c, l.cellS), part);
  c->launches++;
  reduce2(c, {part, l.nbc, 1.0, 4}, {part, l.nbc, 1.0, 4}, 1);
  return RT_OK;
}

int rt_launch_permute_in(rt_ctx *c, const double *src, double *dst, int rows, int stride) {
  k_permute_in<<<blocks_for(c->C, 256), 256, 0, c->stream>>>(c->C, rows, stride, rt_ptr<int32_t>(c, c->lay.perm), src, dst);
  c->launches++;
  return RT_OK;
}
int rt_launch_permute_out(rt_ctx *c, const double *src, double *dst, int rows, int stride) {
  k_permute_out<<<blocks_for(c->C, 256), 256, 0, c->stream>>>(c->C, rows, stride, rt_ptr<int32_t>(c, c->lay.perm), src, dst);
  c->launches++;
  return RT_OK;
}
int rt_launch_init_sources(rt_ctx *c, const int32_t *cell_dev, int nsrc) {
  int32_t *srcidx = rt_ptr<int32_t>(c, c->lay.srcidx);
  k_fill_i32<<<blocks_for(c->C, 256), 256, 0, c->stream>>>(c->C, -1, srcidx);
  if (nsrc > 0)
    k_set_sources<<<(nsrc + 255) / 256, 256, 0, c->stream>>>(nsrc, cell_dev, rt_ptr<int32_t>(c, c->lay.iperm), srcidx);
  c->launches += 2;
  return RT_OK;
}
