// a2-a4: the transport kernels of one Heun stage.
//   k_grad    one thread per (cell, group): second term of eq (15) over the cell's faces with the
//             stored per-face prefactors, multiply by the stored inverse matrix, second loop over
//             the faces for the slope limiter
//   k_flux    one thread per (face, group): extrapolate both cells to the face centre, M1 closure,
//             global Lax-Friedrichs flux with signal speed c~, donor cap; the flux is saved to
//             memory, not scattered
//   k_update  one thread per (cell, group): sum the saved fluxes over the cell's face list, add
//             the source, Heun combine, floor and |F| <= c~ N (S3, S11, S12)
// State layout U[g][4][C] (N, Fx, Fy, Fz), grad[g][12][C] (field-major, then direction).
#include "rt_internal.cuh"
#include "rt_kernels.cuh"

// neighbour or ghost state seen across a boundary face with right code `code` (S13)
__device__ inline void ghost_for_gradient(int code, const double Ui[4], const double n[3], const double *ghost, int G,
                                          int g, double Uj[4]) {
  if (code == RT_BC_OUTFLOW) { Uj[0] = Ui[0]; Uj[1] = Ui[1]; Uj[2] = Ui[2]; Uj[3] = Ui[3]; }
  else if (code == RT_BC_REFLECT) {
    const double p = 2.0 * (Ui[1] * n[0] + Ui[2] * n[1] + Ui[3] * n[2]);
    Uj[0] = Ui[0]; Uj[1] = Ui[1] - p * n[0]; Uj[2] = Ui[2] - p * n[1]; Uj[3] = Ui[3] - p * n[2];
  } else {
    const double *gs = ghost + ((size_t)(RT_BC_DIRICHLET0 - code) * G + g) * 4;
    Uj[0] = gs[0]; Uj[1] = gs[1]; Uj[2] = gs[2]; Uj[3] = gs[3];
  }
}

template <int GG>
__global__ void __launch_bounds__(RT_BLOCK * GG) k_grad(rt_geom m, const double *__restrict__ U,
                                                           double *__restrict__ grad) {
  const int64_t C = m.C, F = m.F;
  const int64_t i = (int64_t)blockIdx.x * RT_BLOCK + threadIdx.x;
  const int g = threadIdx.y;
  if (i >= C) return;
  const double *Ug = U + (size_t)4 * g * C;
  double Ui[4] = {Ug[i], Ug[C + i], Ug[2 * C + i], Ug[3 * C + i]};
  double b[4][3], hi[4], lo[4];
#pragma unroll
  for (int q = 0; q < 4; q++) { b[q][0] = b[q][1] = b[q][2] = 0.0; hi[q] = lo[q] = Ui[q]; }
  const int64_t f0 = m.fo[i], f1 = m.fo[i + 1], r0 = m.ro[i], r1 = m.ro[i + 1];
  const int64_t nown = f1 - f0, ntot = nown + (r1 - r0);
  // first loop: sum_f w_f (phi_j - phi_i), min/max
  for (int64_t k = 0; k < ntot; k++) {
    const bool own = k < nown;
    const int64_t q = own ? f0 + k : m.rl[r0 + (k - nown)];
    const int32_t j = own ? m.R[q] : m.L[q];
    const double sg = own ? 1.0 : -1.0;
    const double wx = sg * m.w[q], wy = sg * m.w[F + q], wz = sg * m.w[2 * F + q];
    double Uj[4];
    if (j >= 0) { Uj[0] = Ug[j]; Uj[1] = Ug[C + j]; Uj[2] = Ug[2 * C + j]; Uj[3] = Ug[3 * C + j]; }
    else {
      const double n[3] = {m.nrm[q], m.nrm[F + q], m.nrm[2 * F + q]};
      ghost_for_gradient(j, Ui, n, m.ghost, m.G, g, Uj);
    }
#pragma unroll
    for (int v = 0; v < 4; v++) {
      const double d = Uj[v] - Ui[v];
      b[v][0] += wx * d; b[v][1] += wy * d; b[v][2] += wz * d;
      hi[v] = fmax(hi[v], Uj[v]); lo[v] = fmin(lo[v], Uj[v]);
    }
  }
  const double m00 = m.Minv[i], m01 = m.Minv[C + i], m02 = m.Minv[2 * C + i], m11 = m.Minv[3 * C + i],
               m12 = m.Minv[4 * C + i], m22 = m.Minv[5 * C + i];
  double gr[4][3];
#pragma unroll
  for (int v = 0; v < 4; v++) {
    gr[v][0] = m00 * b[v][0] + m01 * b[v][1] + m02 * b[v][2];
    gr[v][1] = m01 * b[v][0] + m11 * b[v][1] + m12 * b[v][2];
    gr[v][2] = m02 * b[v][0] + m12 * b[v][1] + m22 * b[v][2];
  }
  // second loop: extreme extrapolated increments at the face centres.  min_f (hi-phi)/D_f is
  // attained at the largest D_f (division is monotone), so only the extremes are kept.
  const double sx = m.s[i], sy = m.s[C + i], sz = m.s[2 * C + i];
  double dmax[4] = {0, 0, 0, 0}, dmin[4] = {0, 0, 0, 0};
  for (int64_t k = 0; k < ntot; k++) {
    const bool own = k < nown;
    const int64_t q = own ? f0 + k : m.rl[r0 + (k - nown)];
    double rx = m.cf[q] - sx, ry = m.cf[F + q] - sy, rz = m.cf[2 * F + q] - sz;
    if (!own) { rx = rt_wrap(rx, m.box[0], m.per[0]); ry = rt_wrap(ry, m.box[1], m.per[1]); rz = rt_wrap(rz, m.box[2], m.per[2]); }
#pragma unroll
    for (int v = 0; v < 4; v++) {
      const double d = gr[v][0] * rx + gr[v][1] * ry + gr[v][2] * rz;
      dmax[v] = fmax(dmax[v], d); dmin[v] = fmin(dmin[v], d);
    }
  }
  double *out = grad + (size_t)12 * g * C;
#pragma unroll
  for (int v = 0; v < 4; v++) {
    double a = 1.0;
    if (dmax[v] > 0.0) a = fmin(a, (hi[v] - Ui[v]) / dmax[v]);
    if (dmin[v] < 0.0) a = fmin(a, (lo[v] - Ui[v]) / dmin[v]);
    out[(size_t)(3 * v) * C + i] = a * gr[v][0];
    out[(size_t)(3 * v + 1) * C + i] = a * gr[v][1];
    out[(size_t)(3 * v + 2) * C + i] = a * gr[v][2];
  }
}

// c~^2 P.n / c~^2 = N D.n for the M1 closure (S1), lab frame
__device__ inline void pressure_dot_n(const double U[4], const double n[3], double ct, double out[3]) {
  const double f2n = U[1] * U[1] + U[2] * U[2] + U[3] * U[3];
  const double fn = sqrt(f2n);
  const double f = fmin(1.0, fn / fmax(ct * U[0], 1e-300));
  const double chi = (3.0 + 4.0 * f * f) / (5.0 + 2.0 * sqrt(4.0 - 3.0 * f * f));
  const double a = 0.5 * (1.0 - chi) * U[0];
  double bb = 0.0;
  if (f2n > 0.0) bb = 0.5 * (3.0 * chi - 1.0) * U[0] * (U[1] * n[0] + U[2] * n[1] + U[3] * n[2]) / f2n;
  out[0] = a * n[0] + bb * U[1]; out[1] = a * n[1] + bb * U[2]; out[2] = a * n[2] + bb * U[3];
}

__device__ inline void extrapolate(const double *__restrict__ Ug, const double *__restrict__ gg, int64_t C, int64_t i,
                                   double rx, double ry, double rz, bool second_order, double Uo[4]) {
#pragma unroll
  for (int v = 0; v < 4; v++) {
    double x = Ug[(size_t)v * C + i];
    if (second_order)
      x += gg[(size_t)(3 * v) * C + i] * rx + gg[(size_t)(3 * v + 1) * C + i] * ry + gg[(size_t)(3 * v + 2) * C + i] * rz;
    Uo[v] = x;
  }
}

template <int GG>
__global__ void __launch_bounds__(RT_BLOCK * GG) k_flux(rt_geom m, const double *__restrict__ U,
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
    const double n[3] = {m.nrm[q], m.nrm[F + q], m.nrm[2 * F + q]};
    const double cx = m.cf[q], cy = m.cf[F + q], cz = m.cf[2 * F + q];
    const double A = m.A[q];
    double UL[4], UR[4];
    extrapolate(Ug, gg, C, l, cx - m.s[l], cy - m.s[C + l], cz - m.s[2 * C + l], second_order, UL);
    if (r >= 0) {
      extrapolate(Ug, gg, C, r, rt_wrap(cx - m.s[r], m.box[0], m.per[0]), rt_wrap(cy - m.s[C + r], m.box[1], m.per[1]),
                  rt_wrap(cz - m.s[2 * C + r], m.box[2], m.per[2]), second_order, UR);
    } else if (r == RT_BC_OUTFLOW) { UR[0] = UR[1] = UR[2] = UR[3] = 0.0; }  // vacuum ghost
    else if (r == RT_BC_REFLECT) {
      const double p = 2.0 * (UL[1] * n[0] + UL[2] * n[1] + UL[3] * n[2]);
      UR[0] = UL[0]; UR[1] = UL[1] - p * n[0]; UR[2] = UL[2] - p * n[1]; UR[3] = UL[3] - p * n[2];
    } else {
      const double *gs = m.ghost + ((size_t)(RT_BC_DIRICHLET0 - r) * m.G + g) * 4;
      UR[0] = gs[0]; UR[1] = gs[1]; UR[2] = gs[2]; UR[3] = gs[3];
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
    const int32_t d = ph[0] > 0.0 ? l : (ph[0] < 0.0 ? r : -1);
    if (d >= 0) {
      const double lim = Ug[d] * m.vol[d] / (dt * A);
      if (fabs(ph[0]) > lim) ph[0] = ph[0] > 0.0 ? lim : -lim;
    }
    double *po = phi + (size_t)4 * g * F;
    po[q] = ph[0]; po[F + q] = ph[1]; po[2 * F + q] = ph[2]; po[3 * F + q] = ph[3];
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

template <int GG>
__global__ void __launch_bounds__(RT_BLOCK * GG) k_update(rt_geom m, const double *Ucur,
                                                             const double *U0,
                                                             const double *__restrict__ phi, double *Uout,
                                                             const int32_t *__restrict__ srcidx,
                                                             const double *__restrict__ srcrate, int nsrc, double ca,
                                                             double cb, double dt, double ct, double n_floor,
                                                             double *__restrict__ part_floor) {
  __shared__ double sm[GG][RT_BLOCK / 32];
  const int64_t C = m.C, F = m.F;
  const int64_t i = (int64_t)blockIdx.x * RT_BLOCK + threadIdx.x;
  const int g = threadIdx.y;
  double fl = 0.0;
  if (i < C) {
    const double *pg = phi + (size_t)4 * g * F;
    double sum[4] = {0, 0, 0, 0};
    const int64_t f0 = m.fo[i], f1 = m.fo[i + 1], r0 = m.ro[i], r1 = m.ro[i + 1];
    for (int64_t q = f0; q < f1; q++) {
      const double A = m.A[q];
      sum[0] += A * pg[q]; sum[1] += A * pg[F + q]; sum[2] += A * pg[2 * F + q]; sum[3] += A * pg[3 * F + q];
    }
    for (int64_t k = r0; k < r1; k++) {
      const int64_t q = m.rl[k];
      const double A = m.A[q];
      sum[0] -= A * pg[q]; sum[1] -= A * pg[F + q]; sum[2] -= A * pg[2 * F + q]; sum[3] -= A * pg[3 * F + q];
    }
    const double V = m.vol[i];
    double R[4] = {-sum[0] / V, -sum[1] / V, -sum[2] / V, -sum[3] / V};
    const int32_t si = srcidx[i];
    if (si >= 0) R[0] += srcrate[(size_t)g * nsrc + si] / V;  // isotropic source (S5)
    const size_t o = (size_t)4 * g * C + i;
    double Un[4];
#pragma unroll
    for (int v = 0; v < 4; v++) Un[v] = ca * U0[o + (size_t)v * C] + cb * (Ucur[o + (size_t)v * C] + dt * R[v]);
    if (Un[0] < n_floor) { fl = V * (n_floor - Un[0]); Un[0] = n_floor; }
    const double fn = sqrt(Un[1] * Un[1] + Un[2] * Un[2] + Un[3] * Un[3]), lim = ct * Un[0];
    if (fn > lim) { const double sc = lim / fn; Un[1] *= sc; Un[2] *= sc; Un[3] *= sc; }
#pragma unroll
    for (int v = 0; v < 4; v++) Uout[o + (size_t)v * C] = Un[v];
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
__global__ void __launch_bounds__(RT_BLOCK * GG) k_stored(int64_t C, int G, const double *__restrict__ U,
                                                             const double *__restrict__ vol, double *__restrict__ part) {
  __shared__ double sm[GG][RT_BLOCK / 32];
  const int64_t i = (int64_t)blockIdx.x * RT_BLOCK + threadIdx.x;
  const int g = threadIdx.y;
  double v = i < C ? vol[i] * U[(size_t)4 * g * C + i] : 0.0;
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

__global__ void k_permute_in(int64_t C, int rows, const int32_t *__restrict__ perm, const double *__restrict__ src,
                             double *__restrict__ dst) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= C) return;
  const int32_t o = perm[p];
  for (int r = 0; r < rows; r++) dst[(size_t)r * C + p] = src[(size_t)r * C + o];
}
__global__ void k_permute_out(int64_t C, int rows, const int32_t *__restrict__ perm, const double *__restrict__ src,
                              double *__restrict__ dst) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= C) return;
  const int32_t o = perm[p];
  for (int r = 0; r < rows; r++) dst[(size_t)r * C + o] = src[(size_t)r * C + p];
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
#define DISPATCH_G(Gv, KERNEL, grid, block, stream, ...)                                  \
  switch (Gv) {                                                                           \
    case 1: KERNEL<1><<<grid, block, 0, stream>>>(__VA_ARGS__); break;                    \
    case 2: KERNEL<2><<<grid, block, 0, stream>>>(__VA_ARGS__); break;                    \
    case 3: KERNEL<3><<<grid, block, 0, stream>>>(__VA_ARGS__); break;                    \
    case 4: KERNEL<4><<<grid, block, 0, stream>>>(__VA_ARGS__); break;                    \
    case 5: KERNEL<5><<<grid, block, 0, stream>>>(__VA_ARGS__); break;                    \
    case 6: KERNEL<6><<<grid, block, 0, stream>>>(__VA_ARGS__); break;                    \
    case 7: KERNEL<7><<<grid, block, 0, stream>>>(__VA_ARGS__); break;                    \
    default: KERNEL<8><<<grid, block, 0, stream>>>(__VA_ARGS__); break;                   \
  }
rt_geom rt_geom_of(const rt_ctx *c) {
  const rt_layout &l = c->lay;
  rt_geom m;
  m.C = c->C; m.F = c->F; m.G = c->G;
  m.vol = rt_ptr<double>(c, l.vol); m.s = rt_ptr<double>(c, l.s); m.Minv = rt_ptr<double>(c, l.Minv);
  m.A = rt_ptr<double>(c, l.A); m.nrm = rt_ptr<double>(c, l.nrm); m.cf = rt_ptr<double>(c, l.cf);
  m.w = rt_ptr<double>(c, l.w); m.L = rt_ptr<int32_t>(c, l.L); m.R = rt_ptr<int32_t>(c, l.R);
  m.rl = rt_ptr<int32_t>(c, l.rl); m.fo = rt_ptr<int64_t>(c, l.fo); m.ro = rt_ptr<int64_t>(c, l.ro);
  m.ghost = rt_ptr<double>(c, l.ghost);
  for (int a = 0; a < 3; a++) { m.box[a] = c->box[a]; m.per[a] = c->per[a]; }
  return m;
}

int rt_launch_gradients(rt_ctx *c, const double *U) {
  DISPATCH_G(c->G, k_grad, (unsigned)c->lay.nbc, dim3(RT_BLOCK, c->G), c->stream, rt_geom_of(c), U,
             rt_ptr<double>(c, c->lay.grad));
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
  double *p_floor = part + (size_t)G * l.nbc, *p_out = part + (size_t)G * 3 * l.nbc, *p_in = p_out + (size_t)G * l.nbf;
  const int second = c->par.order >= 2;
  if (second) {
    rt_prof_begin(c, RT_K_GRAD);
    DISPATCH_G(G, k_grad, (unsigned)l.nbc, dim3(RT_BLOCK, G), c->stream, m, Uin, grad);
    rt_prof_end(c);
    c->launches++;
  }
  rt_prof_begin(c, RT_K_FLUX);
  DISPATCH_G(G, k_flux, (unsigned)l.nbf, dim3(RT_BLOCK, G), c->stream, m, Uin, grad, phi, c->par.ctilde, dt, second, p_out,
             p_in);
  rt_prof_end(c);
  c->launches++;
  reduce2(c, {p_out, l.nbf, wl * dt, 1}, {p_in, l.nbf, wl * dt, 2}, 2);
  rt_prof_begin(c, RT_K_UPDATE);
  DISPATCH_G(G, k_update, (unsigned)l.nbc, dim3(RT_BLOCK, G), c->stream, m, Uin, U0, phi, Uout,
             rt_ptr<int32_t>(c, l.srcidx), rt_ptr<double>(c, l.srcrate), c->nsrc, ca, cb, dt, c->par.ctilde,
             c->par.n_floor, p_floor);
  rt_prof_end(c);
  c->launches++;
  reduce2(c, {p_floor, l.nbc, wf, 3}, {p_floor, l.nbc, wf, 3}, 1);
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
    reduce2(c, {rt_ptr<double>(c, l.part), l.nbc, 1.0, 0}, {rt_ptr<double>(c, l.part), l.nbc, 1.0, 0}, 1);
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
  DISPATCH_G(c->G, k_stored, (unsigned)l.nbc, dim3(RT_BLOCK, c->G), c->stream, c->C, c->G, rt_ptr<double>(c, l.Ua),
             rt_ptr<double>(c, l.vol), part);
  c->launches++;
  reduce2(c, {part, l.nbc, 1.0, 4}, {part, l.nbc, 1.0, 4}, 1);
  return RT_OK;
}

int rt_launch_permute_in(rt_ctx *c, const double *src, double *dst, int rows) {
  k_permute_in<<<(unsigned)((c->C + 255) / 256), 256, 0, c->stream>>>(c->C, rows, rt_ptr<int32_t>(c, c->lay.perm), src, dst);
  c->launches++;
  return RT_OK;
}
int rt_launch_permute_out(rt_ctx *c, const double *src, double *dst, int rows) {
  k_permute_out<<<(unsigned)((c->C + 255) / 256), 256, 0, c->stream>>>(c->C, rows, rt_ptr<int32_t>(c, c->lay.perm), src, dst);
  c->launches++;
  return RT_OK;
}
int rt_launch_init_sources(rt_ctx *c, const int32_t *cell_dev, int nsrc) {
  int32_t *srcidx = rt_ptr<int32_t>(c, c->lay.srcidx);
  k_fill_i32<<<(unsigned)((c->C + 255) / 256), 256, 0, c->stream>>>(c->C, -1, srcidx);
  if (nsrc > 0)
    k_set_sources<<<(nsrc + 255) / 256, 256, 0, c->stream>>>(nsrc, cell_dev, rt_ptr<int32_t>(c, c->lay.iperm), srcidx);
  c->launches += 2;
  return RT_OK;
}
