// a2-a4: the transport kernels of one Heun stage, one thread block per tile of TC consecutive
// cells of the Peano-Hilbert order (layout and tile tables: rt_internal.cuh).
//   k_grad   stages the tile's face records (eq (15) prefactors, face centres, neighbour ids), its
//            cells' U and its face-list tables in shared memory with coalesced loads; then one
//            thread per (cell, group) sums the second term of eq (15) over the cell's faces,
//            multiplies by the stored inverse matrix and runs the slope limiter
//
//   k_stage  stages the tile's U and gradients in shared memory; one thread per face slot
//            extrapolates both cells to the face centre, evaluates the M1 closure and the global
//            Lax-Friedrichs flux with signal speed c~ and the donor cap for every group, and
//            leaves A*Phi in shared memory; after a barrier one thread per
//            (cell, group) sums the cell's face list in fixed order, adds the source, does the Heun
//            combine, the floor and |F| <= c~ N (S3, S11, S12).  The fluxes
//            never go to HBM; a face shared by two tiles is evaluated by both.
// fp64 throughout.  Reciprocals and the closure's square root use MUFU seeds + two Newton steps
// (relative error ~1e-16, no special-case branches: all arguments are positive and normal).
#include <stdlib.h>
#include "rt_internal.cuh"
#include "rt_kernels.cuh"

__device__ __forceinline__ double4 ld4(const double *p) { return *reinterpret_cast<const double4 *>(p); }
__device__ __forceinline__ void st4(double *p, double a, double b, double c, double d) {
  *reinterpret_cast<double4 *>(p) = make_double4(a, b, c, d);
}
__device__ __forceinline__ double dmax2(double a, double b) { return a > b ? a : b; }
__device__ __forceinline__ double dmin2(double a, double b) { return a < b ? a : b; }

// 1/x for positive normal x: MUFU.RCP64H seed, two Newton steps
__device__ __forceinline__ double fast_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  return fma(r, e, r);
}
// sqrt(x) for positive normal x: MUFU.RSQ64H seed, two coupled Newton steps (g -> sqrt x, h -> 1/(2 sqrt x))
__device__ __forceinline__ double fast_sqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double g = x * y, h = 0.5 * y;
  double r = fma(-h, g, 0.5);
  g = fma(g, r, g); h = fma(h, r, h);
  r = fma(-h, g, 0.5);
  return fma(g, r, g);
}

// neighbour or ghost state seen across a boundary face with right code `code` (S13)
__device__ __forceinline__ double4 ghost_for_gradient(int code, const double4 Ui, const double *faceN, int64_t q,
                                                      const double *ghost, int G, int g) {
  if (code == RT_BC_OUTFLOW) return Ui;
  if (code == RT_BC_REFLECT) {
    const double4 n = ld4(faceN + 4 * q);
    const double p = 2.0 * (Ui.y * n.x + Ui.z * n.y + Ui.w * n.z);
    return make_double4(Ui.x, Ui.y - p * n.x, Ui.z - p * n.y, Ui.w - p * n.z);
  }
  return ld4(ghost + ((size_t)(RT_BC_DIRICHLET0 - code) * G + g) * 4);
}

// fixed-order block sum of v over the block's threads; result valid in thread 0.
// red: shared scratch of >= 32 doubles.
__device__ __forceinline__ double block_sum(double v, double *red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[w] = v;
  __syncthreads();
  double t = 0.0;
  if (threadIdx.x == 0)
    for (int k = 0; k < nw; k++) t += red[k];
  return t;
}

// per-tile face-list tables staged in shared memory: local cell x has the half-faces
// hl[ho[x]..ho[x+1]]: slot number, bit 15 set where the cell is the face's right cell
struct tile_tables { int *ho; uint16_t *hl; };
__device__ __forceinline__ tile_tables stage_tables(const rt_geom &m, unsigned char *base, int64_t c0, int ncell) {
  tile_tables t;
  t.ho = reinterpret_cast<int *>(base);
  t.hl = reinterpret_cast<uint16_t *>(t.ho + (m.TC + 1));
  const int64_t hbase = m.fo[c0] + m.ro[c0];
  for (int x = threadIdx.x; x <= ncell; x += blockDim.x) t.ho[x] = (int)(m.fo[c0 + x] + m.ro[c0 + x] - hbase);
  const int nh = (int)(m.fo[c0 + ncell] + m.ro[c0 + ncell] - hbase);
  const uint16_t *src = m.hl + hbase;
  for (int k = threadIdx.x; k < nh; k += blockDim.x) t.hl[k] = src[k];
  return t;
}

// min-image of a face-centre offset: |d| < 1.5 L always (the face touches the cell)
__device__ __forceinline__ double wrap1(double d, double L, int per) {
  const double h = 0.5 * L;
  const double w = d > h ? d - L : (d < -h ? d + L : d);
  return per ? w : d;
}

// ------------------------------------------------------------------ a2: gradients + limiter
template <int G>
__global__ void __launch_bounds__(256) k_grad(rt_geom m, const double *__restrict__ U, double *__restrict__ grad) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double *sW = reinterpret_cast<double *>(smem_raw);  // [smax][4]  (w, L|R)
  double *sC = sW + 4 * m.smax;                       // [smax][4]  (c, A)
  double *sU = sC + 4 * m.smax;                       // [TC][G][4]
  const int64_t C = m.C;
  const int64_t c0 = (int64_t)blockIdx.x * m.TC;
  const int ncell = (int)(c0 + m.TC < C ? m.TC : C - c0);
  const int64_t fbase = m.fo[c0];
  const int nown = (int)(m.fo[c0 + ncell] - fbase);
  const int64_t ib = m.inco[blockIdx.x];
  const int ns = nown + (int)(m.inco[blockIdx.x + 1] - ib);
  // stage the slot records, the tile's U and the face-list tables
  for (int s = threadIdx.x; s < ns; s += blockDim.x) {
    const int64_t q = s < nown ? fbase + s : (int64_t)m.incf[ib + (s - nown)];
    *reinterpret_cast<double4 *>(sW + 4 * s) = ld4(m.faceW + 4 * q);
    *reinterpret_cast<double4 *>(sC + 4 * s) = ld4(m.faceC + 4 * q);
  }
  {
    const double *Ut = U + 4 * c0 * G;
    for (int x = threadIdx.x; x < ncell * G; x += blockDim.x) *reinterpret_cast<double4 *>(sU + 4 * x) = ld4(Ut + 4 * x);
  }
  const tile_tables tt = stage_tables(m, reinterpret_cast<unsigned char *>(sU + 4 * m.TC * G), c0, ncell);
  __syncthreads();

  const int32_t c0i = (int32_t)c0;
  for (int item = threadIdx.x; item < ncell * G; item += blockDim.x) {
    const int il = item / G, g = item - il * G;
    const int64_t i = c0 + il;
    const double4 Ui = ld4(sU + 4 * item);
    double b[4][3], hi[4] = {Ui.x, Ui.y, Ui.z, Ui.w}, lo[4] = {Ui.x, Ui.y, Ui.z, Ui.w};
#pragma unroll
    for (int v = 0; v < 4; v++) b[v][0] = b[v][1] = b[v][2] = 0.0;
    const int h0 = tt.ho[il], h1 = tt.ho[il + 1];
    const double *Ug = U + 4 * g;  // neighbour j outside the tile: Ug + 4 G j

    // first pass over the cell's half-faces: sum_f w_f (phi_j - phi_i), min/max.  Where the cell is
    // the face's right cell, d = s_L - s_R: the stored prefactor changes sign, the neighbour is L.
#pragma unroll 2
    for (int k = h0; k < h1; k++) {
      const unsigned e = tt.hl[k];
      const int s = (int)(e & 0x7fffu);
      const bool right = e >= 0x8000u;
      const double4 w = ld4(sW + 4 * s);
      int32_t l, r;
      rt_unpack_lr(w.w, l, r);
      const int32_t j = right ? l : r;
      const double sg = right ? -1.0 : 1.0;
      double4 Uj;
      if (j >= 0) {
        const unsigned jl = (unsigned)(j - c0i);
        Uj = ld4(jl < (unsigned)ncell ? sU + 4 * ((int)jl * G + g) : Ug + (int64_t)(4 * G) * j);
      } else Uj = ghost_for_gradient(j, Ui, m.faceN, fbase + s, m.ghost, G, g);
      const double wx = sg * w.x, wy = sg * w.y, wz = sg * w.z;
      const double d0 = Uj.x - Ui.x, d1 = Uj.y - Ui.y, d2 = Uj.z - Ui.z, d3 = Uj.w - Ui.w;
      b[0][0] += wx * d0; b[0][1] += wy * d0; b[0][2] += wz * d0;
      b[1][0] += wx * d1; b[1][1] += wy * d1; b[1][2] += wz * d1;
      b[2][0] += wx * d2; b[2][1] += wy * d2; b[2][2] += wz * d2;
      b[3][0] += wx * d3; b[3][1] += wy * d3; b[3][2] += wz * d3;
      hi[0] = dmax2(hi[0], Uj.x); hi[1] = dmax2(hi[1], Uj.y); hi[2] = dmax2(hi[2], Uj.z); hi[3] = dmax2(hi[3], Uj.w);
      lo[0] = dmin2(lo[0], Uj.x); lo[1] = dmin2(lo[1], Uj.y); lo[2] = dmin2(lo[2], Uj.z); lo[3] = dmin2(lo[3], Uj.w);
    }
    const double *Mi = m.Minv + 6 * i;
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
    const double4 si = ld4(m.cellS + 4 * i);
    double dmax[4] = {0, 0, 0, 0}, dmin[4] = {0, 0, 0, 0};
    // (the stored face centre is in the left cell's frame: min-image it for the right cell;
    // for the left cell the wrap is the identity)
#pragma unroll 2
    for (int k = h0; k < h1; k++) {
      const double4 c = ld4(sC + 4 * (int)(tt.hl[k] & 0x7fffu));
      const double rx = wrap1(c.x - si.x, m.box[0], m.per[0]), ry = wrap1(c.y - si.y, m.box[1], m.per[1]),
                   rz = wrap1(c.z - si.z, m.box[2], m.per[2]);
#pragma unroll
      for (int v = 0; v < 4; v++) {
        const double d = gr[v][0] * rx + gr[v][1] * ry + gr[v][2] * rz;
        dmax[v] = dmax2(dmax[v], d); dmin[v] = dmin2(dmin[v], d);
      }
    }
    double *out = grad + 12 * (i * G + g);
    const double Uiv[4] = {Ui.x, Ui.y, Ui.z, Ui.w};
    double o[12];
#pragma unroll
    for (int v = 0; v < 4; v++) {
      double a = 1.0;
      if (dmax[v] > 0.0) a = dmin2(a, (hi[v] - Uiv[v]) / dmax[v]);
      if (dmin[v] < 0.0) a = dmin2(a, (lo[v] - Uiv[v]) / dmin[v]);
      o[3 * v] = a * gr[v][0]; o[3 * v + 1] = a * gr[v][1]; o[3 * v + 2] = a * gr[v][2];
    }
    st4(out, o[0], o[1], o[2], o[3]); st4(out + 4, o[4], o[5], o[6], o[7]); st4(out + 8, o[8], o[9], o[10], o[11]);
  }
}

// ------------------------------------------------------------------ a3 + a4: fluxes and update
// N D.n for the M1 closure (S1), lab frame, D = (1-chi)/2 I + (3 chi - 1)/2 nF nF^T with
// chi = (3+4f^2)/(5+2s), s = sqrt(4-3f^2), f = min(1, |F|/(c~ N)).  Written with one square root and
// two reciprocals: with m = max(|F|^2, (c~N)^2), f^2 = |F|^2/m, and since
// 3 chi - 1 = 6 f^2/(2+s):  (1-chi)/2 = 1/3 - f^2/(2+s),  (3chi-1)/2 N /|F|^2 = 3 N/((2+s) m).
__device__ __forceinline__ void pressure_dot_n(const double U[4], const double n[3], double ct, double out[3]) {
  const double f2n = U[1] * U[1] + U[2] * U[2] + U[3] * U[3];
  const double cN = ct * U[0];
  const double mm = dmax2(dmax2(f2n, cN * cN), 1e-290);
  const double rm = fast_rcp(mm);
  const double f2 = f2n * rm;
  const double r2 = fast_rcp(2.0 + fast_sqrt(fma(-3.0, f2, 4.0)));
  const double a = fma(-f2, r2, 1.0 / 3.0) * U[0];
  const double bb = 3.0 * U[0] * (U[1] * n[0] + U[2] * n[1] + U[3] * n[2]) * (rm * r2);
  out[0] = a * n[0] + bb * U[1]; out[1] = a * n[1] + bb * U[2]; out[2] = a * n[2] + bb * U[3];
}

// U_face = U_i + grad U_i . r  (linear extrapolation to the centre of the interface)
// pu: the cell's (N, Fx, Fy, Fz); pg: its 12 gradient components (field-major); shared or global
template <bool SECOND>
__device__ __forceinline__ void extrapolate(const double *pu, const double *pg, double rx, double ry, double rz,
                                            double Uo[4], double &Ncentre) {
  const double4 u = ld4(pu);
  Ncentre = u.x;
  Uo[0] = u.x; Uo[1] = u.y; Uo[2] = u.z; Uo[3] = u.w;
  if (SECOND) {
    const double4 a = ld4(pg), b = ld4(pg + 4), c = ld4(pg + 8);
    Uo[0] += a.x * rx + a.y * ry + a.z * rz;
    Uo[1] += a.w * rx + b.x * ry + b.y * rz;
    Uo[2] += b.z * rx + b.w * ry + c.x * rz;
    Uo[3] += c.y * rx + c.z * ry + c.w * rz;
  }
}

template <int G, bool SECOND>
__global__ void __launch_bounds__(256) k_stage(rt_geom m, const double *__restrict__ Uin, const double *__restrict__ grad,
                                               const double *U0, double *Uout, const int32_t *__restrict__ srcidx,
                                               const double *__restrict__ srcrate, int nsrc, double ca, double cb, double dt,
                                               double ct, double n_floor, double *__restrict__ part_floor,
                                               double *__restrict__ part_out, double *__restrict__ part_in) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ double red[32];
  constexpr int PS = 4 * G > 8 ? 4 * G : 8;             // doubles per slot
  double *sPhi = reinterpret_cast<double *>(smem_raw);  // [smax][PS]: the staged face record (c, A), (n, L|R),
                                                        // overwritten by its owner thread with A * (Phi_N, Phi_F)[G]
  double *sR = sPhi + PS * m.smax;                      // [TC][G][RT_REC]  U (4) + gradients (12)
  double *sS = sR + RT_REC * G * m.TC;                  // [TC][4]  (s, V)
  const int64_t C = m.C;
  const int64_t c0 = (int64_t)blockIdx.x * m.TC;
  const int ncell = (int)(c0 + m.TC < C ? m.TC : C - c0);
  const int64_t fbase = m.fo[c0];
  const int nown = (int)(m.fo[c0 + ncell] - fbase);
  const int64_t ib = m.inco[blockIdx.x];
  const int ns = nown + (int)(m.inco[blockIdx.x + 1] - ib);
  // stage the face records, the tile's cells and the face-list tables
  for (int s = threadIdx.x; s < ns; s += blockDim.x) {
    const int64_t q = s < nown ? fbase + s : (int64_t)m.incf[ib + (s - nown)];
    *reinterpret_cast<double4 *>(sPhi + PS * s) = ld4(m.faceC + 4 * q);
    *reinterpret_cast<double4 *>(sPhi + PS * s + 4) = ld4(m.faceN + 4 * q);
  }
  {
    const double *Ut = Uin + 4 * c0 * G, *gt = grad + 12 * c0 * G;
    for (int x = threadIdx.x; x < ncell * G; x += blockDim.x) *reinterpret_cast<double4 *>(sR + RT_REC * x) = ld4(Ut + 4 * x);
    if (SECOND)
      for (int u = threadIdx.x; u < ncell * G * 3; u += blockDim.x) {
        const int x = u / 3, part = u - 3 * x;
        *reinterpret_cast<double4 *>(sR + RT_REC * x + 4 + 4 * part) = ld4(gt + 4 * u);
      }
    const double *St = m.cellS + 4 * c0;
    for (int x = threadIdx.x; x < ncell; x += blockDim.x) *reinterpret_cast<double4 *>(sS + 4 * x) = ld4(St + 4 * x);
  }
  const tile_tables tt = stage_tables(m, reinterpret_cast<unsigned char *>(sS + 4 * m.TC), c0, ncell);
  __syncthreads();

  // ---- a3: one thread per face slot, all groups
  double b_out[G], b_in[G];
#pragma unroll
  for (int g = 0; g < G; g++) b_out[g] = b_in[g] = 0.0;
  int bnd = 0;
  const double hc2 = 0.5 * ct * ct, hc = 0.5 * ct;
  const int32_t c0i = (int32_t)c0;
  for (int s = threadIdx.x; s < ns; s += blockDim.x) {
    const double4 fc = ld4(sPhi + PS * s), fn = ld4(sPhi + PS * s + 4);
    int32_t l, r;
    rt_unpack_lr(fn.w, l, r);
    const double n[3] = {fn.x, fn.y, fn.z};
    const double A = fc.w;
    const unsigned ll = (unsigned)(l - c0i), rl = (unsigned)(r - c0i);
    const bool l_in = ll < (unsigned)ncell, r_in = rl < (unsigned)ncell;  // r < 0 gives a huge rl
    // per-group rows of the two cells: shared memory for tile cells, global memory for the halo
    const double *puL = l_in ? sR + RT_REC * G * (int)ll : Uin + (int64_t)(4 * G) * l;
    const double *pgL = l_in ? puL + 4 : grad + (int64_t)(12 * G) * l;
    const int suL = l_in ? RT_REC : 4, sgL = l_in ? RT_REC : 12;
    const double4 sl = ld4(l_in ? sS + 4 * (int)ll : m.cellS + 4 * (int64_t)l);
    const double rLx = fc.x - sl.x, rLy = fc.y - sl.y, rLz = fc.z - sl.z;
    const int rr = r >= 0 ? r : 0;
    const double *puR = r_in ? sR + RT_REC * G * (int)rl : Uin + (int64_t)(4 * G) * rr;
    const double *pgR = r_in ? puR + 4 : grad + (int64_t)(12 * G) * rr;
    const int suR = r_in ? RT_REC : 4, sgR = r_in ? RT_REC : 12;
    double rRx = 0.0, rRy = 0.0, rRz = 0.0, Vr = 0.0;
    if (r >= 0) {
      const double4 sr = ld4(r_in ? sS + 4 * (int)rl : m.cellS + 4 * (int64_t)r);
      Vr = sr.w;
      rRx = wrap1(fc.x - sr.x, m.box[0], m.per[0]); rRy = wrap1(fc.y - sr.y, m.box[1], m.per[1]);
      rRz = wrap1(fc.z - sr.z, m.box[2], m.per[2]);
    }
    const double rdtA = fast_rcp(dt * A);
    const double capL = sl.w * rdtA, capR = Vr * rdtA;
#pragma unroll
    for (int g = 0; g < G; g++) {
      double UL[4], UR[4], NL, NR = 0.0;
      extrapolate<SECOND>(puL + suL * g, pgL + sgL * g, rLx, rLy, rLz, UL, NL);
      if (r >= 0) extrapolate<SECOND>(puR + suR * g, pgR + sgR * g, rRx, rRy, rRz, UR, NR);
      else if (r == RT_BC_OUTFLOW) { UR[0] = UR[1] = UR[2] = UR[3] = 0.0; }  // vacuum ghost
      else if (r == RT_BC_REFLECT) {
        const double p = 2.0 * (UL[1] * n[0] + UL[2] * n[1] + UL[3] * n[2]);
        UR[0] = UL[0]; UR[1] = UL[1] - p * n[0]; UR[2] = UL[2] - p * n[1]; UR[3] = UL[3] - p * n[2];
      } else {
        const double4 gs = ld4(m.ghost + ((size_t)(RT_BC_DIRICHLET0 - r) * G + g) * 4);
        UR[0] = gs.x; UR[1] = gs.y; UR[2] = gs.z; UR[3] = gs.w;
      }
      double PL[3], PR[3], ph[4];
      pressure_dot_n(UL, n, ct, PL);
      pressure_dot_n(UR, n, ct, PR);
      ph[0] = 0.5 * ((UL[1] + UR[1]) * n[0] + (UL[2] + UR[2]) * n[1] + (UL[3] + UR[3]) * n[2]) - hc * (UR[0] - UL[0]);
#pragma unroll
      for (int a = 0; a < 3; a++) ph[1 + a] = hc2 * (PL[a] + PR[a]) - hc * (UR[1 + a] - UL[1 + a]);
      // donor cap (S11): the donor cannot lose more photons than it holds through this face in dt;
      // only the number flux is clamped (continuous in the state; Phi_F is left alone)
      if (ph[0] > 0.0) ph[0] = dmin2(ph[0], NL * capL);
      else if (r >= 0) ph[0] = -dmin2(-ph[0], NR * capR);
      st4(sPhi + PS * s + 4 * g, A * ph[0], A * ph[1], A * ph[2], A * ph[3]);
      if (r == RT_BC_OUTFLOW) { b_out[g] += A * ph[0]; bnd = 1; }
      else if (r <= RT_BC_DIRICHLET0) { b_in[g] -= A * ph[0]; bnd = 1; }
    }
  }
  // boundary ledgers: fixed-order block sums, one row per tile (the barrier also ends phase a3)
  if (__syncthreads_or(bnd)) {
#pragma unroll
    for (int g = 0; g < G; g++) {
      const double so = block_sum(b_out[g], red), si = block_sum(b_in[g], red);
      if (threadIdx.x == 0) { part_out[(size_t)blockIdx.x * G + g] = so; part_in[(size_t)blockIdx.x * G + g] = si; }
    }
  } else if (threadIdx.x < G) {
    part_out[(size_t)blockIdx.x * G + threadIdx.x] = 0.0;
    part_in[(size_t)blockIdx.x * G + threadIdx.x] = 0.0;
  }

  // ---- a4: one thread per (cell, group): gather the cell's faces in list order, update
  double fl[G];
#pragma unroll
  for (int g = 0; g < G; g++) fl[g] = 0.0;
  int floored = 0;
  for (int item = threadIdx.x; item < ncell * G; item += blockDim.x) {
    const int il = item / G, g = item - il * G;
    const int64_t i = c0 + il;
    const int h0 = tt.ho[il], h1 = tt.ho[il + 1];
    const double *pg = sPhi + 4 * g;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
#pragma unroll 4
    for (int k = h0; k < h1; k++) {
      const unsigned e = tt.hl[k];
      const double4 p = ld4(pg + PS * (int)(e & 0x7fffu));
      const double sg = e >= 0x8000u ? -1.0 : 1.0;  // the flux leaves the left cell and enters the right one
      a0 = fma(sg, p.x, a0); a1 = fma(sg, p.y, a1); a2 = fma(sg, p.z, a2); a3 = fma(sg, p.w, a3);
    }
    const double V = sS[4 * il + 3];
    const double kk = dt * fast_rcp(V);  // dt / V
    const int32_t si = srcidx[i];
    if (si >= 0) a0 -= srcrate[(size_t)g * nsrc + si];  // isotropic source (S5): + dt Ndot / V on N
    const int64_t o = 4 * (i * G + g);
    const double4 uc = ld4(sR + RT_REC * item), u0 = ld4(U0 + o);
    double Un[4] = {ca * u0.x + cb * fma(-kk, a0, uc.x), ca * u0.y + cb * fma(-kk, a1, uc.y),
                    ca * u0.z + cb * fma(-kk, a2, uc.z), ca * u0.w + cb * fma(-kk, a3, uc.w)};
    if (Un[0] < n_floor) {
      const double add = V * (n_floor - Un[0]);
#pragma unroll
      for (int gg = 0; gg < G; gg++) if (gg == g) fl[gg] += add;
      Un[0] = n_floor; floored = 1;
    }
    const double f2 = Un[1] * Un[1] + Un[2] * Un[2] + Un[3] * Un[3], lim = ct * Un[0];
    if (f2 > lim * lim) { const double sc = lim / sqrt(f2); Un[1] *= sc; Un[2] *= sc; Un[3] *= sc; }
    st4(Uout + o, Un[0], Un[1], Un[2], Un[3]);
  }
  if (__syncthreads_or(floored)) {
#pragma unroll
    for (int g = 0; g < G; g++) {
      const double t = block_sum(fl[g], red);
      if (threadIdx.x == 0) part_floor[(size_t)blockIdx.x * G + g] = t;
    }
  } else if (threadIdx.x < G) part_floor[(size_t)blockIdx.x * G + threadIdx.x] = 0.0;
}

// ------------------------------------------------------------------ ledgers
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
__global__ void __launch_bounds__(RT_BLOCK *GG) k_stored(int64_t C, const double *__restrict__ U,
                                                          const double *__restrict__ cellS, double *__restrict__ part) {
  __shared__ double sm[GG][RT_BLOCK / 32];
  const int64_t i = (int64_t)blockIdx.x * RT_BLOCK + threadIdx.x;
  const int g = threadIdx.y;
  double v = i < C ? cellS[4 * i + 3] * U[((size_t)i * GG + g) * 4] : 0.0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) sm[g][threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int k = 0; k < RT_BLOCK / 32; k++) t += sm[g][k];
    part[(size_t)blockIdx.x * GG + g] = t;
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
#define DISPATCH_G(Gv, KERNEL, grid, block, smem, stream, ...)                            \
  switch (Gv) {                                                                           \
    case 1: KERNEL(1)<<<grid, block, smem, stream>>>(__VA_ARGS__); break;                 \
    case 2: KERNEL(2)<<<grid, block, smem, stream>>>(__VA_ARGS__); break;                 \
    case 3: KERNEL(3)<<<grid, block, smem, stream>>>(__VA_ARGS__); break;                 \
    case 4: KERNEL(4)<<<grid, block, smem, stream>>>(__VA_ARGS__); break;                 \
    case 5: KERNEL(5)<<<grid, block, smem, stream>>>(__VA_ARGS__); break;                 \
    case 6: KERNEL(6)<<<grid, block, smem, stream>>>(__VA_ARGS__); break;                 \
    case 7: KERNEL(7)<<<grid, block, smem, stream>>>(__VA_ARGS__); break;                 \
    default: KERNEL(8)<<<grid, block, smem, stream>>>(__VA_ARGS__); break;                \
  }
#define K_GRAD(g) k_grad<g>
#define K_STAGE2(g) k_stage<g, true>
#define K_STAGE1(g) k_stage<g, false>
#define K_STORED(g) k_stored<g>

// the tile kernels need more than the default 48 KB of dynamic shared memory
template <class K>
static cudaError_t allow_smem(K kernel, size_t bytes) {
  cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  if (e != cudaSuccess) return e;
  // as many blocks per SM as shared memory allows: take the largest carve-out
  return cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
}
#define SET_SMEM_G(Gv, KERNEL, bytes, err)                      \
  switch (Gv) {                                                 \
    case 1: err = allow_smem(KERNEL(1), bytes); break;          \
    case 2: err = allow_smem(KERNEL(2), bytes); break;          \
    case 3: err = allow_smem(KERNEL(3), bytes); break;          \
    case 4: err = allow_smem(KERNEL(4), bytes); break;          \
    case 5: err = allow_smem(KERNEL(5), bytes); break;          \
    case 6: err = allow_smem(KERNEL(6), bytes); break;          \
    case 7: err = allow_smem(KERNEL(7), bytes); break;          \
    default: err = allow_smem(KERNEL(8), bytes); break;         \
  }

int rt_transport_configure(rt_ctx *c) {
  cudaError_t e = cudaSuccess;
  const size_t sg = rt_smem_grad(c->TC, c->G, c->smax, c->hmax), ss = rt_smem_stage(c->TC, c->G, c->smax, c->hmax);
  SET_SMEM_G(c->G, K_GRAD, sg, e);
  if (e == cudaSuccess) SET_SMEM_G(c->G, K_STAGE2, ss, e);
  if (e == cudaSuccess) SET_SMEM_G(c->G, K_STAGE1, ss, e);
  if (e != cudaSuccess) return rt_fail(c, RT_ECUDA, "cudaFuncSetAttribute(shared memory): %s", cudaGetErrorString(e));
  return RT_OK;
}

// threads per tile block: a whole number of warps, at most 256 (the kernels' launch bound);
// RT_TILE_THREADS in the environment overrides the default for experiments
static int tile_threads(const rt_ctx *c) {
  static int env = -1;
  if (env < 0) { const char *e = getenv("RT_TILE_THREADS"); env = e ? atoi(e) : 0; }
  int n = env > 0 ? env : 256;
  n = ((n + 31) / 32) * 32;
  return n > 256 ? 256 : (n < 32 ? 32 : n);
}

rt_geom rt_geom_of(const rt_ctx *c) {
  const rt_layout &l = c->lay;
  rt_geom m;
  m.C = c->C; m.F = c->F; m.G = c->G; m.TC = c->TC; m.smax = c->smax;
  m.cellS = rt_ptr<double>(c, l.cellS); m.Minv = rt_ptr<double>(c, l.Minv);
  m.faceC = rt_ptr<double>(c, l.faceC); m.faceN = rt_ptr<double>(c, l.faceN); m.faceW = rt_ptr<double>(c, l.faceW);
  m.fo = rt_ptr<int64_t>(c, l.fo); m.ro = rt_ptr<int64_t>(c, l.ro); m.inco = rt_ptr<int64_t>(c, l.inco);
  m.incf = rt_ptr<int32_t>(c, l.incf); m.hl = rt_ptr<uint16_t>(c, l.hl);
  m.ghost = rt_ptr<double>(c, l.ghost);
  for (int a = 0; a < 3; a++) { m.box[a] = c->box[a]; m.per[a] = c->per[a]; }
  return m;
}

int rt_launch_gradients(rt_ctx *c, const double *U) {
  DISPATCH_G(c->G, K_GRAD, (unsigned)c->T, tile_threads(c), rt_smem_grad(c->TC, c->G, c->smax, c->hmax), c->stream, rt_geom_of(c), U,
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
  double *grad = rt_ptr<double>(c, l.grad);
  double *part = rt_ptr<double>(c, l.part);
  const int64_t nchem = blocks_for(c->C, RT_CHEM_BLOCK);
  double *p_floor = part + (size_t)G * nchem, *p_out = p_floor + (size_t)G * c->T, *p_in = p_out + (size_t)G * c->T;
  const int nt = tile_threads(c);
  const size_t ss = rt_smem_stage(c->TC, G, c->smax, c->hmax);
  if (c->par.order >= 2) {
    rt_prof_begin(c, RT_K_GRAD);
    DISPATCH_G(G, K_GRAD, (unsigned)c->T, nt, rt_smem_grad(c->TC, G, c->smax, c->hmax), c->stream, m, Uin, grad);
    rt_prof_end(c);
    c->launches++;
    rt_prof_begin(c, RT_K_UPDATE);
    DISPATCH_G(G, K_STAGE2, (unsigned)c->T, nt, ss, c->stream, m, Uin, grad, U0, Uout, rt_ptr<int32_t>(c, l.srcidx),
               rt_ptr<double>(c, l.srcrate), c->nsrc, ca, cb, dt, c->par.ctilde, c->par.n_floor, p_floor, p_out, p_in);
    rt_prof_end(c);
  } else {
    rt_prof_begin(c, RT_K_UPDATE);
    DISPATCH_G(G, K_STAGE1, (unsigned)c->T, nt, ss, c->stream, m, Uin, grad, U0, Uout, rt_ptr<int32_t>(c, l.srcidx),
               rt_ptr<double>(c, l.srcrate), c->nsrc, ca, cb, dt, c->par.ctilde, c->par.n_floor, p_floor, p_out, p_in);
    rt_prof_end(c);
  }
  c->launches++;
  reduce2(c, {p_out, c->T, wl * dt, 1}, {p_in, c->T, wl * dt, 2}, 2);
  reduce2(c, {p_floor, c->T, wf, 3}, {p_floor, c->T, wf, 3}, 1);
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
  DISPATCH_G(c->G, K_STORED, (unsigned)l.nbc, dim3(RT_BLOCK, c->G), 0, c->stream, c->C, rt_ptr<double>(c, l.Ua),
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
