// a2-a4: the transport kernels of one Heun stage.  A thread block works on one tile of TC consecutive
// cells of the Peano-Hilbert order; everything the tile touches (its cells, its faces, the cells
// across its faces, its index tables: layout in rt_internal.cuh) is staged in shared memory with
// asynchronous copies (TMA bulk copies for the contiguous runs, 16-byte LDGSTS for the gathers)
// and the arithmetic then runs from shared memory alone.
//   k_grad    one thread per (cell, group): the second term of eq (15) summed over the cell's
//             faces, times the stored inverse matrix, then the slope limiter
//   k_flux    a3: one lane per (owned face, group) extrapolates both cells to the face centre,
//             evaluates the M1 closure, the global Lax-Friedrichs flux with signal speed c~ and the
//             donor cap, and leaves A*Phi in shared memory.  Every face is
//             evaluated once, by the tile of its left cell; fluxes of faces whose right cell lies in
//             a later tile also go to xphi.  a4: the tile's cells sum their faces in list order; a
//             cell all of whose faces are the tile's gets the source, the Heun combine, the floor
//             and |F| <= c~ N here (S3, S11, S12)
//   k_finish  a4 for the other cells: adds the fluxes of the faces owned by earlier tiles (xphi)
// fp64 throughout.  Reciprocals and the closure's square root use MUFU seeds + two Newton steps
// (relative error ~1e-16, no special-case branches: all arguments are positive and normal).
#include "rt_internal.cuh"
#include "rt_kernels.cuh"

__device__ __forceinline__ unsigned long long now_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
  return t;
}
__device__ __forceinline__ double4 ld4(const double *p) { return *reinterpret_cast<const double4 *>(p); }
__device__ __forceinline__ double2 ld2(const double *p) { return *reinterpret_cast<const double2 *>(p); }
__device__ __forceinline__ void st2(double *p, double a, double b) { *reinterpret_cast<double2 *>(p) = make_double2(a, b); }
__device__ __forceinline__ void st4(double *p, double a, double b, double c, double d) {
  *reinterpret_cast<double4 *>(p) = make_double4(a, b, c, d);
}
// x with its sign bit xor-ed with sgn (0 or 0x80000000): an integer operation, not an fp64 multiply
__device__ __forceinline__ double flip_sign(double x, int sgn) { return __hiloint2double(__double2hiint(x) ^ sgn, __double2loint(x)); }
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

// 1/sqrt(x) for positive normal x: MUFU.RSQ64H seed, two Newton steps
__device__ __forceinline__ double fast_rsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double hx = 0.5 * x;
  y = y * fma(-hx * y, y, 1.5);
  return y * fma(-hx * y, y, 1.5);
}

// neighbour or ghost state seen across a boundary face with right code `code` (S13)
__device__ __forceinline__ double4 ghost_for_gradient(int code, const double4 Ui, const double *faceN, int64_t F, int64_t q,
                                                      const double *ghost, int G, int g) {
  if (code == RT_BC_OUTFLOW) return Ui;
  if (code == RT_BC_REFLECT) {
    const double2 n01 = ld2(faceN + 2 * q);
    const double4 n = make_double4(n01.x, n01.y, faceN[2 * F + 2 * q], 0.0);
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

// asynchronous 16-byte global -> shared copies (LDGSTS) for the gathers: the data never passes
// through registers, so one thread keeps many copies in flight; they bypass L1
__device__ __forceinline__ void cp16(void *dst, const void *src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp8(void *dst, const void *src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
// n consecutive 16-byte chunks
template <int N>
__device__ __forceinline__ void cp_run(double *dst, const double *src) {
#pragma unroll
  for (int c = 0; c < N; c++) cp16(dst + 2 * c, src + 2 * c);
}

// bulk asynchronous global -> shared copies (TMA, cp.async.bulk) for the long contiguous runs: one instruction moves a whole
// contiguous run (16-byte aligned, a multiple of 16 bytes) and reports to an mbarrier, so staging a
// tile costs a handful of instructions instead of one per 16 bytes
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
// one arrival that also announces `bytes` of bulk copies still to land in this phase
__device__ __forceinline__ void mbar_expect(uint64_t *bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@!p bra WAIT_%=;\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, uint64_t *bar) {
  if (bytes == 0) return;
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// asks L2 to fetch a contiguous run (a tile that a later block will stage)
__device__ __forceinline__ void bulk_prefetch_l2(const void *src, unsigned bytes) {
  if (bytes == 0) return;
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}

// a tile's blob in shared memory (layout: rt_internal.cuh)
struct tile_view {
  int64_t c0, fbase, xbase;
  int ncell, nown, ninc, ns, nh, nhf, nb, nout, words, bnd;
  const uint32_t *ho, *hl, *slr, *halo, *incf, *outs;  // in shared memory
  const uint32_t *blob;                                // in global memory
};
// the view of a tile whose blob (header + tables) has landed in shared memory at sB
__device__ __forceinline__ tile_view view_tile(const rt_geom &m, const uint32_t *sB, unsigned tile) {
  const rt_tile d = *reinterpret_cast<const rt_tile *>(sB);
  tile_view v;
  v.c0 = (int64_t)tile * m.TC;
  v.ncell = (int)(v.c0 + m.TC < m.C ? m.TC : m.C - v.c0);
  v.fbase = d.fbase; v.xbase = d.xbase; v.nown = d.nown; v.ninc = d.ninc; v.ns = d.nown + d.ninc; v.nh = d.nh; v.nhf = d.nhf;
  v.nb = d.nb; v.nout = d.nout; v.bnd = d.pad & 1;
  v.words = rt_blob_words(m.TC, v.nhf, v.nown, v.nh, v.ninc, v.nout);
  v.ho = sB + RT_BLOB_HEAD; v.hl = v.ho + m.TC + 1; v.slr = v.hl + v.nhf; v.halo = v.slr + v.nown; v.incf = v.halo + v.nh;
  v.outs = v.incf + v.ninc;
  v.blob = m.blob + (size_t)tile * m.bstride;
  return v;
}

// ------------------------------------------------------------------ a2: gradients + limiter
// Four lanes per cell.  Lane (h, p) of a cell keeps the fields {2h, 2h + 1} of (N, Fx, Fy, Fz) of a block of up
// to three groups in registers and takes the entries p, p + 2, ... of the cell's half-face list; the partial
// sums, minima and maxima of the two lanes p are combined by shuffles (a fixed order: deterministic).  A
// face's geometry is thereby loaded once for three groups and two fields: shared-memory loads cost the
// same whether the lanes of a warp ask for distinct words or for the same one (profiles/r2_alu_peak.md),
// so one lane per (cell, group) spent two thirds of its geometry loads on copies.
// Cell rows in shared memory are padded to an odd number of 16-byte chunks (bank spread of the gathers).
__device__ __forceinline__ double shx(double v, int lane_mask) { return __shfl_xor_sync(0xffffffffu, v, lane_mask); }

struct grad_smem { const double *Wl, *Wh, *Cl, *Ch, *U, *M; };

// the gradients of groups g0 .. g0 + GB - 1 of the tile's cells.  BND: the tile has boundary half-faces
template <int G, int GB, bool BND>
__device__ __forceinline__ void grad_cells(const rt_geom &m, const tile_view &v, const grad_smem &sm, const int g0,
                                           double *__restrict__ grad, const int tid, const int nt) {
  constexpr int US = 4 * G + 2;  // doubles per cell row
  const int h = (tid >> 1) & 1, p = tid & 1;
  for (int xb = 0; xb < v.ncell; xb += nt >> 2) {  // (whole warps iterate together: the shuffles need every lane)
    const int x = xb + (tid >> 2);
    // (a passive cell is skipped: its face state is its cell value; a ghost's gradient is imported: rt_halo_unpack)
    const bool on = x < v.ncell && (!m.cact || (m.cact[v.c0 + x] & 5) == 1);
    const int xx = on ? x : 0;
    const int h0 = on ? (int)v.ho[xx] : 0, h1 = on ? (int)v.ho[xx + 1] : 0;
    const double *ui_p = sm.U + US * xx + 4 * g0 + 2 * h;
    double ui[GB][2], b[GB][2][3], hi[GB][2], lo[GB][2];
#pragma unroll
    for (int g = 0; g < GB; g++) {
      const double2 t = ld2(ui_p + 4 * g);
      ui[g][0] = hi[g][0] = lo[g][0] = t.x; ui[g][1] = hi[g][1] = lo[g][1] = t.y;
#pragma unroll
      for (int f = 0; f < 2; f++) b[g][f][0] = b[g][f][1] = b[g][f][2] = 0.0;
    }
    // first pass over the cell's half-faces: sum_f w_f (phi_j - phi_i), min/max.  Where the cell is
    // the face's right cell, d = s_L - s_R: the stored prefactor changes sign.
#pragma unroll 2
    for (int k = h0 + p; k < h1; k += 2) {
      const uint32_t e = v.hl[k];
      const int s = (int)(e & 0x7fffu);
      const uint32_t nb = e >> 16;
      const int sgn = (int)((e & 0x8000u) << 16);  // sign bit where the cell is the right one
      const double2 wl = ld2(sm.Wl + 2 * s);
      const double wzz = sm.Wh[2 * s];
      const double wx = flip_sign(wl.x, sgn), wy = flip_sign(wl.y, sgn), wz = flip_sign(wzz, sgn);
      double2 uj[GB];
      if (!BND || nb < 0xFF00u) {
        const double *q = sm.U + US * (int)nb + 4 * g0 + 2 * h;
#pragma unroll
        for (int g = 0; g < GB; g++) uj[g] = ld2(q + 4 * g);
      } else {  // ghost state across a boundary face (S13)
        const int code = (int)nb - 0x10000;
#pragma unroll
        for (int g = 0; g < GB; g++) {
          const double4 Ui = ld4(sm.U + US * xx + 4 * (g0 + g));
          const double4 gh = ghost_for_gradient(code, Ui, m.faceN, m.F, v.fbase + s, m.ghost, G, g0 + g);
          uj[g] = h ? make_double2(gh.z, gh.w) : make_double2(gh.x, gh.y);
        }
      }
#pragma unroll
      for (int g = 0; g < GB; g++) {
        const double d0 = uj[g].x - ui[g][0], d1 = uj[g].y - ui[g][1];
        b[g][0][0] += wx * d0; b[g][0][1] += wy * d0; b[g][0][2] += wz * d0;
        b[g][1][0] += wx * d1; b[g][1][1] += wy * d1; b[g][1][2] += wz * d1;
        hi[g][0] = dmax2(hi[g][0], uj[g].x); hi[g][1] = dmax2(hi[g][1], uj[g].y);
        lo[g][0] = dmin2(lo[g][0], uj[g].x); lo[g][1] = dmin2(lo[g][1], uj[g].y);
      }
    }
    const double *Mi = sm.M + 6 * xx;
    const double2 ma = ld2(Mi), mb = ld2(Mi + 2), mc = ld2(Mi + 4);
    const double m00 = ma.x, m01 = ma.y, m02 = mb.x, m11 = mb.y, m12 = mc.x, m22 = mc.y;
    double gr[GB][2][3];
#pragma unroll
    for (int g = 0; g < GB; g++)
#pragma unroll
      for (int f = 0; f < 2; f++) {
        // (the two lanes of a pair add their partial sums: both get the same bits)
        const double b0 = b[g][f][0] + shx(b[g][f][0], 1), b1 = b[g][f][1] + shx(b[g][f][1], 1), b2 = b[g][f][2] + shx(b[g][f][2], 1);
        hi[g][f] = dmax2(hi[g][f], shx(hi[g][f], 1));
        lo[g][f] = dmin2(lo[g][f], shx(lo[g][f], 1));
        gr[g][f][0] = m00 * b0 + m01 * b1 + m02 * b2;
        gr[g][f][1] = m01 * b0 + m11 * b1 + m12 * b2;
        gr[g][f][2] = m02 * b0 + m12 * b1 + m22 * b2;
      }
    // second pass: extreme extrapolated increments at the face centres.  min_f (hi-phi)/D_f is
    // attained at the largest D_f (division is monotone), so only the extremes are kept.
    // The stored face centre is relative to the left cell; seen from the right cell it is
    // c - d with d = kappa w (rt_internal.cuh).
    double dmx[GB][2], dmn[GB][2];
#pragma unroll
    for (int g = 0; g < GB; g++) dmx[g][0] = dmx[g][1] = dmn[g][0] = dmn[g][1] = 0.0;
#pragma unroll 2
    for (int k = h0 + p; k < h1; k += 2) {
      const uint32_t e = v.hl[k];
      const int s = (int)(e & 0x7fffu);
      const double2 cl = ld2(sm.Cl + 2 * s);
      double rx = cl.x, ry = cl.y, rz = sm.Ch[2 * s];
      if (e & 0x8000u) {  // (a cell's right-side faces come last in its list: mostly uniform across a warp)
        const double2 wl = ld2(sm.Wl + 2 * s), wh = ld2(sm.Wh + 2 * s);
        rx = fma(-wh.y, wl.x, rx); ry = fma(-wh.y, wl.y, ry); rz = fma(-wh.y, wh.x, rz);
      }
#pragma unroll
      for (int g = 0; g < GB; g++)
#pragma unroll
        for (int f = 0; f < 2; f++) {
          const double d = gr[g][f][0] * rx + gr[g][f][1] * ry + gr[g][f][2] * rz;
          dmx[g][f] = dmax2(dmx[g][f], d); dmn[g][f] = dmin2(dmn[g][f], d);
        }
    }
#pragma unroll
    for (int g = 0; g < GB; g++) {
      double o[6];
#pragma unroll
      for (int f = 0; f < 2; f++) {
        const double dx = dmax2(dmx[g][f], shx(dmx[g][f], 1)), dn = dmin2(dmn[g][f], shx(dmn[g][f], 1));
        const double up = hi[g][f] - ui[g][f], dw = ui[g][f] - lo[g][f];
        double a = 1.0;
        // (reciprocals from the MUFU seed where the divisor is safely normal: a sixth of a division)
        if (dx > 0.0) a = dmin2(a, dx > 1e-280 ? up * fast_rcp(dx) : up / dx);
        if (dn < 0.0) a = dmin2(a, dn < -1e-280 ? dw * fast_rcp(-dn) : -dw / dn);
        o[3 * f] = a * gr[g][f][0]; o[3 * f + 1] = a * gr[g][f][1]; o[3 * f + 2] = a * gr[g][f][2];
      }
      // lane h of a pair owns the chunks 3h .. 3h + 2 of the (cell, group) row; the lanes p share the groups
      if (on && ((g0 + g) & 1) == p) {
        double *out = grad + 12 * ((v.c0 + x) * G + g0 + g) + 6 * h;
        st2(out, o[0], o[1]); st2(out + 2, o[2], o[3]); st2(out + 4, o[4], o[5]);
      }
    }
  }
}

// ---- mixed precision (rt_params.mixed, reading S28): the same lane mapping; the differences phi_j - phi_i are
// formed in double and rounded, everything after them is single precision in the length unit l0 (a power of
// two: the scaling is exact).  Stored: l0 * (limited gradient), 12 floats per (cell, group).
__device__ __forceinline__ float shxf(float v, int lane_mask) { return __shfl_xor_sync(0xffffffffu, v, lane_mask); }
__device__ __forceinline__ float flip_signf(float x, int sgn) { return __int_as_float(__float_as_int(x) ^ sgn); }

template <int G, int GB, bool BND>
__device__ __forceinline__ void grad_cells_mixed(const rt_geom &m, const tile_view &v, const grad_smem &sm, const int g0,
                                                 float *__restrict__ grad, const int tid, const int nt) {
  constexpr int US = 4 * G + 2;
  const int h = (tid >> 1) & 1, p = tid & 1;
  const double il0 = m.il0;
  for (int xb = 0; xb < v.ncell; xb += nt >> 2) {
    const int x = xb + (tid >> 2);
    const bool on = x < v.ncell && (!m.cact || (m.cact[v.c0 + x] & 5) == 1);
    const int xx = on ? x : 0;
    const int h0 = on ? (int)v.ho[xx] : 0, h1 = on ? (int)v.ho[xx + 1] : 0;
    const double *ui_p = sm.U + US * xx + 4 * g0 + 2 * h;
    double ui[GB][2];
    float b[GB][2][3], hi[GB][2], lo[GB][2];  // sums and the extreme differences (phi_i itself counts: hi >= 0 >= lo)
#pragma unroll
    for (int g = 0; g < GB; g++) {
      const double2 t = ld2(ui_p + 4 * g);
      ui[g][0] = t.x; ui[g][1] = t.y;
#pragma unroll
      for (int f = 0; f < 2; f++) { b[g][f][0] = b[g][f][1] = b[g][f][2] = 0.0f; hi[g][f] = lo[g][f] = 0.0f; }
    }
#pragma unroll 2
    for (int k = h0 + p; k < h1; k += 2) {
      const uint32_t e = v.hl[k];
      const int s = (int)(e & 0x7fffu);
      const uint32_t nb = e >> 16;
      const int sgn = (int)((e & 0x8000u) << 16);
      const double2 wl = ld2(sm.Wl + 2 * s);
      const double wzz = sm.Wh[2 * s];
      const float wx = flip_signf(__double2float_rn(wl.x * il0), sgn), wy = flip_signf(__double2float_rn(wl.y * il0), sgn),
                  wz = flip_signf(__double2float_rn(wzz * il0), sgn);  // w / l0: dimensionless
      double2 uj[GB];
      if (!BND || nb < 0xFF00u) {
        const double *q = sm.U + US * (int)nb + 4 * g0 + 2 * h;
#pragma unroll
        for (int g = 0; g < GB; g++) uj[g] = ld2(q + 4 * g);
      } else {
        const int code = (int)nb - 0x10000;
#pragma unroll
        for (int g = 0; g < GB; g++) {
          const double4 Ui = ld4(sm.U + US * xx + 4 * (g0 + g));
          const double4 gh = ghost_for_gradient(code, Ui, m.faceN, m.F, v.fbase + s, m.ghost, G, g0 + g);
          uj[g] = h ? make_double2(gh.z, gh.w) : make_double2(gh.x, gh.y);
        }
      }
#pragma unroll
      for (int g = 0; g < GB; g++) {
        const float d0 = __double2float_rn(uj[g].x - ui[g][0]), d1 = __double2float_rn(uj[g].y - ui[g][1]);
        b[g][0][0] = fmaf(wx, d0, b[g][0][0]); b[g][0][1] = fmaf(wy, d0, b[g][0][1]); b[g][0][2] = fmaf(wz, d0, b[g][0][2]);
        b[g][1][0] = fmaf(wx, d1, b[g][1][0]); b[g][1][1] = fmaf(wy, d1, b[g][1][1]); b[g][1][2] = fmaf(wz, d1, b[g][1][2]);
        hi[g][0] = fmaxf(hi[g][0], d0); hi[g][1] = fmaxf(hi[g][1], d1);
        lo[g][0] = fminf(lo[g][0], d0); lo[g][1] = fminf(lo[g][1], d1);
      }
    }
    // M^-1 in units of l0^-2
    const double *Mi = sm.M + 6 * xx;
    const double2 ma = ld2(Mi), mb = ld2(Mi + 2), mc = ld2(Mi + 4);
    const float m00 = __double2float_rn(ma.x * m.l0sq), m01 = __double2float_rn(ma.y * m.l0sq), m02 = __double2float_rn(mb.x * m.l0sq),
                m11 = __double2float_rn(mb.y * m.l0sq), m12 = __double2float_rn(mc.x * m.l0sq), m22 = __double2float_rn(mc.y * m.l0sq);
    float gr[GB][2][3];
#pragma unroll
    for (int g = 0; g < GB; g++)
#pragma unroll
      for (int f = 0; f < 2; f++) {
        const float b0 = b[g][f][0] + shxf(b[g][f][0], 1), b1 = b[g][f][1] + shxf(b[g][f][1], 1), b2 = b[g][f][2] + shxf(b[g][f][2], 1);
        hi[g][f] = fmaxf(hi[g][f], shxf(hi[g][f], 1));
        lo[g][f] = fminf(lo[g][f], shxf(lo[g][f], 1));
        gr[g][f][0] = m00 * b0 + m01 * b1 + m02 * b2;
        gr[g][f][1] = m01 * b0 + m11 * b1 + m12 * b2;
        gr[g][f][2] = m02 * b0 + m12 * b1 + m22 * b2;
      }
    float dmx[GB][2], dmn[GB][2];
#pragma unroll
    for (int g = 0; g < GB; g++) dmx[g][0] = dmx[g][1] = dmn[g][0] = dmn[g][1] = 0.0f;
#pragma unroll 2
    for (int k = h0 + p; k < h1; k += 2) {
      const uint32_t e = v.hl[k];
      const int s = (int)(e & 0x7fffu);
      const double2 cl = ld2(sm.Cl + 2 * s);
      double cx = cl.x, cy = cl.y, cz = sm.Ch[2 * s];
      if (e & 0x8000u) {  // seen from the right cell the face centre is c - kappa w
        const double2 wl = ld2(sm.Wl + 2 * s), wh = ld2(sm.Wh + 2 * s);
        cx = fma(-wh.y, wl.x, cx); cy = fma(-wh.y, wl.y, cy); cz = fma(-wh.y, wh.x, cz);
      }
      const float rx = __double2float_rn(cx * il0), ry = __double2float_rn(cy * il0), rz = __double2float_rn(cz * il0);
#pragma unroll
      for (int g = 0; g < GB; g++)
#pragma unroll
        for (int f = 0; f < 2; f++) {
          const float d = gr[g][f][0] * rx + gr[g][f][1] * ry + gr[g][f][2] * rz;
          dmx[g][f] = fmaxf(dmx[g][f], d); dmn[g][f] = fminf(dmn[g][f], d);
        }
    }
#pragma unroll
    for (int g = 0; g < GB; g++) {
      float o[6];
#pragma unroll
      for (int f = 0; f < 2; f++) {
        const float dx = fmaxf(dmx[g][f], shxf(dmx[g][f], 1)), dn = fminf(dmn[g][f], shxf(dmn[g][f], 1));
        float a = 1.0f;
        if (dx > 0.0f) a = fminf(a, __fdiv_rn(hi[g][f], dx));
        if (dn < 0.0f) a = fminf(a, __fdiv_rn(lo[g][f], dn));
        o[3 * f] = a * gr[g][f][0]; o[3 * f + 1] = a * gr[g][f][1]; o[3 * f + 2] = a * gr[g][f][2];
      }
      if (on && ((g0 + g) & 1) == p) {
        float2 *out = reinterpret_cast<float2 *>(grad + 12 * ((v.c0 + x) * G + g0 + g) + 6 * h);
        out[0] = make_float2(o[0], o[1]); out[1] = make_float2(o[2], o[3]); out[2] = make_float2(o[4], o[5]);
      }
    }
  }
}

template <int G, bool MIXED>
__global__ void __launch_bounds__(128, 4) k_grad(rt_geom m, const double *__restrict__ U, double *__restrict__ grad) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t bar, bar_blob;
  constexpr int US = 4 * G + 2;
  uint32_t *sB = reinterpret_cast<uint32_t *>(smem_raw);    // the tile's blob
  double *sWl = reinterpret_cast<double *>(sB + m.bstride);  // [smax][2]  (wx, wy)      the face records come as
  double *sWh = sWl + 2 * m.smax;                          // [smax][2]  (wz, kappa)   16-byte halves
  double *sCl = sWh + 2 * m.smax;                          // [smax][2]  (cx, cy)      (c = centre - s_L)
  double *sCh = sCl + 2 * m.smax;                          // [smax][2]  (cz, A)
  double *sU = sCh + 2 * m.smax;                           // [TC + hmax][4 G + 2]  tile cells, then halo cells
  double *sM = sU + US * (m.TC + m.hmax);                  // [TC][6]
  const int tid = threadIdx.x, nt = blockDim.x;
  const unsigned tile = (unsigned)m.tlist[m.tbase + blockIdx.x];
  if (m.tact && !(m.tact[tile] & 1)) return;  // no active cell in this tile: passive cells have no gradient
  if (tid == 0) { mbar_init(&bar, 1); mbar_init(&bar_blob, 1); }
  __syncthreads();
  // round 1: the tile's blob sits at a fixed stride: header (descriptor) + tables
  if (tid == 0) {
    mbar_expect(&bar_blob, 4u * m.bstride);
    bulk_g2s(sB, m.blob + (size_t)tile * m.bstride, 4u * m.bstride, &bar_blob);
  }
  mbar_wait(&bar_blob, 0);
  const tile_view v = view_tile(m, sB, tile);
  // round 2: what the descriptor locates (bulk copies: owned faces, M^-1) and what the tables locate
  // (gathers: the cells, the incoming faces), all in flight together
  if (tid == 0) {
    mbar_expect(&bar, 64u * v.nown + 48u * v.ncell);
    bulk_g2s(sWl, m.faceW + 2 * v.fbase, 16u * v.nown, &bar);
    bulk_g2s(sWh, m.faceW + 2 * m.F + 2 * v.fbase, 16u * v.nown, &bar);
    bulk_g2s(sCl, m.faceC + 2 * v.fbase, 16u * v.nown, &bar);
    bulk_g2s(sCh, m.faceC + 2 * m.F + 2 * v.fbase, 16u * v.nown, &bar);
    bulk_g2s(sM, m.Minv + 6 * v.c0, 48u * v.ncell, &bar);
  }
  // the tile's cells and the halo cells: 2 G chunks of 16 bytes each into padded rows
  {
    constexpr int CH = 2 * G;
    const int ne = v.ncell + v.nh;
    for (int idx = tid; idx < ne * CH; idx += nt) {
      const int ci = idx / CH, c = idx - ci * CH;
      const bool own = ci < v.ncell;
      const int64_t gid = own ? v.c0 + ci : (int64_t)v.halo[ci - v.ncell];
      const int row = own ? ci : m.TC + (ci - v.ncell);
      cp16(sU + US * row + 2 * c, U + (int64_t)(4 * G) * gid + 2 * c);
    }
  }
  for (int j = tid; j < v.ninc; j += nt) {
    const int64_t q = v.incf[j];
    cp16(sWl + 2 * (v.nown + j), m.faceW + 2 * q);
    cp16(sWh + 2 * (v.nown + j), m.faceW + 2 * m.F + 2 * q);
    cp16(sCl + 2 * (v.nown + j), m.faceC + 2 * q);
    cp16(sCh + 2 * (v.nown + j), m.faceC + 2 * m.F + 2 * q);
  }
  // (by one thread of the last warp once its own copies are on their way: the two dependent loads overlap the
  // wait for the staged data instead of delaying thread 0's copies)
  if (tid == nt - 32) {
    // a tile that starts a few gridfuls later: pull its contiguous runs into L2 now
    if ((int64_t)blockIdx.x + m.prefetch_tiles < (int64_t)gridDim.x) {
      const int64_t tp = m.tlist[m.tbase + blockIdx.x + m.prefetch_tiles];
      const rt_tile dp = m.tiles[tp];
      const int64_t cp = tp * m.TC;
      const unsigned nc = (unsigned)(cp + m.TC < m.C ? m.TC : m.C - cp);
      bulk_prefetch_l2(m.blob + (size_t)tp * m.bstride, 4u * m.bstride);
      bulk_prefetch_l2(m.faceW + 2 * dp.fbase, 16u * dp.nown);
      bulk_prefetch_l2(m.faceW + 2 * m.F + 2 * dp.fbase, 16u * dp.nown);
      bulk_prefetch_l2(m.faceC + 2 * dp.fbase, 16u * dp.nown);
      bulk_prefetch_l2(m.faceC + 2 * m.F + 2 * dp.fbase, 16u * dp.nown);
      bulk_prefetch_l2(U + 4 * G * cp, 32u * G * nc);
      bulk_prefetch_l2(m.Minv + 6 * cp, 48u * nc);
    }
  }
  mbar_wait(&bar, 0);
  cp_wait_all();
  __syncthreads();

  const grad_smem sm = {sWl, sWh, sCl, sCh, sU, sM};
  // groups in blocks of three (registers: 6 fields x (3 sums + min + max) per lane)
#pragma unroll
  for (int g0 = 0; g0 < G; g0 += 3) {
    constexpr int REM = G % 3;
    if (MIXED) {
      float *gf = reinterpret_cast<float *>(grad);
      if (g0 + 3 <= G) {
        if (v.bnd) grad_cells_mixed<G, 3, true>(m, v, sm, g0, gf, tid, nt);
        else grad_cells_mixed<G, 3, false>(m, v, sm, g0, gf, tid, nt);
      } else if (REM > 0) {
        if (v.bnd) grad_cells_mixed<G, REM ? REM : 1, true>(m, v, sm, g0, gf, tid, nt);
        else grad_cells_mixed<G, REM ? REM : 1, false>(m, v, sm, g0, gf, tid, nt);
      }
    } else if (g0 + 3 <= G) {
      if (v.bnd) grad_cells<G, 3, true>(m, v, sm, g0, grad, tid, nt);
      else grad_cells<G, 3, false>(m, v, sm, g0, grad, tid, nt);
    } else if (REM > 0) {
      if (v.bnd) grad_cells<G, REM ? REM : 1, true>(m, v, sm, g0, grad, tid, nt);
      else grad_cells<G, REM ? REM : 1, false>(m, v, sm, g0, grad, tid, nt);
    }
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
// rec: the cell's (N, Fx, Fy, Fz) followed by its 12 gradient components (field-major), in shared memory
// (use_grad false: a passive cell, whose gradient is not constructed: its face state is its cell value, S27)
template <bool SECOND>
__device__ __forceinline__ void extrapolate(const double *pu, const double *pg, double rx, double ry, double rz, double Uo[4],
                                            double &Ncentre, const bool use_grad = true) {
  const double4 u = ld4(pu);
  Ncentre = u.x;
  Uo[0] = u.x; Uo[1] = u.y; Uo[2] = u.z; Uo[3] = u.w;
  if (SECOND && use_grad) {
    const double4 a = ld4(pg), b = ld4(pg + 4), c = ld4(pg + 8);
    Uo[0] = fma(a.x, rx, fma(a.y, ry, fma(a.z, rz, u.x)));
    Uo[1] = fma(a.w, rx, fma(b.x, ry, fma(b.y, rz, u.y)));
    Uo[2] = fma(b.z, rx, fma(b.w, ry, fma(c.x, rz, u.z)));
    Uo[3] = fma(c.y, rx, fma(c.z, ry, fma(c.w, rz, u.w)));
  }
}

// the end of a4 for one (cell, group): a = sum_f s_if A_f Phi_f; source, Heun combine, floor, |F| <= c~ N
// (S3, S5, S11, S12).  Returns the photons the floor added (0 if none).
struct update_par { double ca, cb, dt, ct, n_floor; };
__device__ __forceinline__ double finish_cell(double a0, double a1, double a2, double a3, double V, double src,
                                              const double4 uc, const double4 u0, const update_par &p, double *out) {
  const double kk = p.dt * fast_rcp(V);  // dt / V
  a0 -= src;                              // isotropic source (S5): + dt Ndot / V on N
  double Un[4] = {p.ca * u0.x + p.cb * fma(-kk, a0, uc.x), p.ca * u0.y + p.cb * fma(-kk, a1, uc.y),
                  p.ca * u0.z + p.cb * fma(-kk, a2, uc.z), p.ca * u0.w + p.cb * fma(-kk, a3, uc.w)};
  double add = 0.0;
  if (Un[0] < p.n_floor) { add = V * (p.n_floor - Un[0]); Un[0] = p.n_floor; }
  const double f2 = Un[1] * Un[1] + Un[2] * Un[2] + Un[3] * Un[3], lim = p.ct * Un[0];
  if (f2 > lim * lim) {  // |F| <= c~ N (S12); 1/sqrt from the MUFU seed where f2 is safely normal
    const double sc = f2 > 1e-280 ? lim * fast_rsqrt(f2) : lim / sqrt(f2);
    Un[1] *= sc; Un[2] *= sc; Un[3] *= sc;
  }
  st4(out, Un[0], Un[1], Un[2], Un[3]);
  return add;
}

// ---- mixed precision (rt_params.mixed, reading S28): single-precision closure in per-face units
__device__ __forceinline__ float4 ldf4(const float *p) { return *reinterpret_cast<const float4 *>(p); }
// the power of two next above mx (clamped to the normal range) and its reciprocal: the unit of N at a face
__device__ __forceinline__ void unit_density(float mx, float &sc, float &is) {
  if (!(mx >= 1e-30f)) mx = 1e-30f;
  int eb = ((__float_as_int(mx) >> 23) & 0xff) + 1;  // mx = 1.x * 2^(eb - 128)
  eb = eb > 253 ? 253 : eb;
  sc = __int_as_float(eb << 23);
  is = __int_as_float((254 - eb) << 23);
}
// n D.nf for the normalised state (n, f = F / (c~ s)), lab frame (S1)
__device__ __forceinline__ void pressure_dot_n_f(float n, const float f[3], const float nf[3], float out[3]) {
  const float f2 = f[0] * f[0] + f[1] * f[1] + f[2] * f[2];
  const float den = fmaxf(n * n, 1e-30f);
  const float x2 = fminf(__fdiv_rn(f2, den), 1.0f);
  const float chi = __fdiv_rn(3.0f + 4.0f * x2, 5.0f + 2.0f * __fsqrt_rn(4.0f - 3.0f * x2));
  const float a = 0.5f * (1.0f - chi) * n;
  float bb = 0.0f;
  if (f2 > 0.0f) bb = __fdiv_rn(0.5f * (3.0f * chi - 1.0f) * n * (f[0] * nf[0] + f[1] * nf[1] + f[2] * nf[2]), f2);
  out[0] = fmaf(bb, f[0], a * nf[0]); out[1] = fmaf(bb, f[1], a * nf[1]); out[2] = fmaf(bb, f[2], a * nf[2]);
}
// the single-precision increments grad . r of (N, Fx, Fy, Fz) to a face centre; pg: 12 floats, field-major
__device__ __forceinline__ void increments_f(const float *pg, float rx, float ry, float rz, float inc[4]) {
  const float4 a = ldf4(pg), b = ldf4(pg + 4), c = ldf4(pg + 8);
  inc[0] = a.x * rx + a.y * ry + a.z * rz;
  inc[1] = a.w * rx + b.x * ry + b.y * rz;
  inc[2] = b.z * rx + b.w * ry + c.x * rz;
  inc[3] = c.y * rx + c.z * ry + c.w * rz;
}

template <int G, bool SECOND, bool MIXED>
__global__ void __launch_bounds__(256, 3) k_flux(rt_geom m, const double *__restrict__ Uin, const double *__restrict__ grad,
                                                 const double *U0, double *Uout, const int32_t *__restrict__ srcidx,
                                                 const double *__restrict__ srcrate, int nsrc, update_par up,
                                                 double *__restrict__ pacc, double *__restrict__ part_floor,
                                                 double *__restrict__ part_out, double *__restrict__ part_in) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ double red[32];
  __shared__ __align__(8) uint64_t bar, bar_blob;
  constexpr int NP = G > 3 ? G : 3;                        // planes of [omax][4]
  const int NE = (m.TC + m.fmax + 1) & ~1;                 // tile cells, then forward halo cells
  const int OM = m.omax;
  uint32_t *sB = reinterpret_cast<uint32_t *>(smem_raw);   // the tile's blob
  double *sF = reinterpret_cast<double *>(sB + m.bstride); // [2 NP][omax][2]: half-planes 0-5 hold the staged face records
                                                           // (cx, cy | cz, A), (nx, ny | nz, -), (wx, wy | wz, kappa) as
                                                           // 16-byte halves; the slot's thread then overwrites
                                                           // half-planes 2g, 2g + 1 with A * (Phi_N, Phi_F) of group g
  double *sU = sF + 4 * NP * OM;                           // [NE][G][4]
  constexpr int GW = MIXED ? 6 : 12;                       // doubles per (cell, group) of gradients (mixed: 12 floats)
  double *sG = sU + 4 * G * NE;                            // [NE][G][12]
  double *sV = sG + GW * G * NE;                           // [NE]  cell volumes
  int32_t *sSrc = reinterpret_cast<int32_t *>(sV + NE);    // [TC] source index or -1
  uint8_t *sAct = reinterpret_cast<uint8_t *>(sSrc + ((m.TC + 3) & ~3));  // [NE] active / touched flags (rt_set_active)
  const unsigned tile = (unsigned)m.tlist[m.tbase + blockIdx.x];
  const int tid = threadIdx.x, nt = blockDim.x;
  const double dt = up.dt, ct = up.ct;
  unsigned long long *tl = m.tl && tid == 0 ? m.tl + 8 * (size_t)tile : nullptr;  // rt_debug_tile_timeline
  if (tl) tl[0] = now_ns();
  if (m.tact && !(m.tact[tile] & 2)) {
    // no cell of this tile is active or shares a face with an active cell: none of its faces
    // carries a flux and none of its cells changes.  The right cells of its outgoing faces still read their
    // rows of xphi: zeros; the first Heun stage still has to carry the tile's cells into the stage buffer.
    const rt_tile d = m.tiles[tile];
    const int64_t c0 = (int64_t)tile * m.TC;
    const int ncell = (int)(c0 + m.TC < m.C ? m.TC : m.C - c0);
    double2 *xo = reinterpret_cast<double2 *>(m.xphi + (size_t)(4 * G) * d.xbase);
    for (int k = tid; k < 2 * G * d.nout; k += nt) xo[k] = make_double2(0.0, 0.0);
    if (Uout != Uin)
      for (int k = tid; k < 2 * G * ncell; k += nt)
        reinterpret_cast<double2 *>(Uout + 4 * G * c0)[k] = reinterpret_cast<const double2 *>(Uin + 4 * G * c0)[k];
    if (tid < G) {
      part_out[(size_t)tile * G + tid] = 0.0; part_in[(size_t)tile * G + tid] = 0.0; part_floor[(size_t)tile * G + tid] = 0.0;
    }
    return;
  }
  if (tid == 0) { mbar_init(&bar, 1); mbar_init(&bar_blob, 1); }
  __syncthreads();
  // round 1: the tile's blob sits at a fixed stride: header (descriptor) + tables
  if (tid == 0) {
    mbar_expect(&bar_blob, 4u * m.bstride);
    bulk_g2s(sB, m.blob + (size_t)tile * m.bstride, 4u * m.bstride, &bar_blob);
  }
  mbar_wait(&bar_blob, 0);
  const tile_view v = view_tile(m, sB, tile);
  if (tl) tl[1] = now_ns();
  // round 2: what the descriptor locates (bulk copies: owned faces, the tile's own cells) and what the
  // tables locate (gathers: forward halo cells), all in flight together
  if (tid == 0) {
    const unsigned nsb = (4u * v.ncell + 15u) & ~15u, nvb = (8u * v.ncell + 15u) & ~15u;  // srcidx and cellV are padded
    mbar_expect(&bar, 96u * v.nown + (SECOND ? 32u + 8u * GW : 32u) * G * v.ncell + nvb + nsb);
    bulk_g2s(sF, m.faceC + 2 * v.fbase, 16u * v.nown, &bar);
    bulk_g2s(sF + 2 * OM, m.faceC + 2 * m.F + 2 * v.fbase, 16u * v.nown, &bar);
    bulk_g2s(sF + 4 * OM, m.faceN + 2 * v.fbase, 16u * v.nown, &bar);
    bulk_g2s(sF + 6 * OM, m.faceN + 2 * m.F + 2 * v.fbase, 16u * v.nown, &bar);
    bulk_g2s(sF + 8 * OM, m.faceW + 2 * v.fbase, 16u * v.nown, &bar);
    bulk_g2s(sF + 10 * OM, m.faceW + 2 * m.F + 2 * v.fbase, 16u * v.nown, &bar);
    bulk_g2s(sU, Uin + 4 * G * v.c0, 32u * G * v.ncell, &bar);
    if (SECOND) bulk_g2s(sG, grad + GW * G * v.c0, 8u * GW * G * v.ncell, &bar);
    bulk_g2s(sV, m.cellV + v.c0, nvb, &bar);
    bulk_g2s(sSrc, srcidx + v.c0, nsb, &bar);
  }
  // round 2: what the blob locates: the forward halo cells (right cells of the outgoing faces)
  const int nf = v.nh - v.nb;
  // (gathers of 32 to 288 bytes: 16-byte asynchronous copies; a halo cell's gradients are split over G threads)
  for (int k = tid; k < nf * (G + 1); k += nt) {
    const int h = k / (G + 1), part = k - h * (G + 1);
    const int64_t id = v.halo[v.nb + h];
    if (part < G) {
      if (SECOND) cp_run<GW / 2>(sG + GW * (G * (m.TC + h) + part), grad + GW * (G * id + part));
    } else {
      cp_run<2 * G>(sU + 4 * G * (m.TC + h), Uin + (int64_t)(4 * G) * id);
      cp8(sV + m.TC + h, m.cellV + id);
    }
  }
  // (by one thread of the last warp once its own copies are on their way: the two dependent loads overlap the
  // wait for the staged data instead of delaying thread 0's copies)
  if (tid == nt - 32) {
    // a tile that starts a few gridfuls later: pull its contiguous runs into L2 now
    if ((int64_t)blockIdx.x + m.prefetch_tiles < (int64_t)gridDim.x) {
      const int64_t tp = m.tlist[m.tbase + blockIdx.x + m.prefetch_tiles];
      const rt_tile dp = m.tiles[tp];
      const int64_t cp = tp * m.TC;
      const unsigned nc = (unsigned)(cp + m.TC < m.C ? m.TC : m.C - cp);
      bulk_prefetch_l2(m.blob + (size_t)tp * m.bstride, 4u * m.bstride);
      for (int hf = 0; hf < 2; hf++) {
        bulk_prefetch_l2(m.faceC + 2 * m.F * hf + 2 * dp.fbase, 16u * dp.nown);
        bulk_prefetch_l2(m.faceN + 2 * m.F * hf + 2 * dp.fbase, 16u * dp.nown);
        bulk_prefetch_l2(m.faceW + 2 * m.F * hf + 2 * dp.fbase, 16u * dp.nown);
      }
      bulk_prefetch_l2(Uin + 4 * G * cp, 32u * G * nc);
      if (SECOND) bulk_prefetch_l2(grad + GW * G * cp, 8u * GW * G * nc);
      bulk_prefetch_l2(U0 + 4 * G * cp, 32u * G * nc);
    }
  }
  if (m.cact) {  // the flags of the tile's cells and of its forward halo cells
    for (int x = tid; x < v.ncell; x += nt) sAct[x] = m.cact[v.c0 + x];
    for (int h = tid; h < nf; h += nt) sAct[m.TC + h] = m.cact[v.halo[v.nb + h]];
  }
  mbar_wait(&bar, 0);
  cp_wait_all();
  __syncthreads();
  if (tl) tl[2] = now_ns();

  // ---- a3: one thread per owned face: its record is read once into registers (so the thread may
  // overwrite it in shared memory with the fluxes), then every group in turn
  int bnd = 0;
  const double hc2 = 0.5 * ct * ct, hc = 0.5 * ct;
  for (int s = tid; s < ((m.variant & 16) ? 0 : v.nown); s += nt) {  // (variant 16: timing experiment without a3)
    const double2 c01 = ld2(sF + 2 * s), c23 = ld2(sF + 2 * (OM + s)), n01 = ld2(sF + 2 * (2 * OM + s)), n23 = ld2(sF + 2 * (3 * OM + s)),
                  w01 = ld2(sF + 2 * (4 * OM + s)), w23 = ld2(sF + 2 * (5 * OM + s));
    const double4 fc = make_double4(c01.x, c01.y, c23.x, c23.y), fn = make_double4(n01.x, n01.y, n23.x, 0.0),
                  fw = make_double4(w01.x, w01.y, w23.x, w23.y);
    const uint32_t lr = v.slr[s];
    const int xl = (int)(lr & 0xffffu);
    int xr = (int)(lr >> 16);
    const bool rin = xr < 0xFF00;
    if (rin && xr >= m.TC) xr -= v.nb;  // forward halo cells follow the tile's cells in sU / sG / sS
    const int r = rin ? 0 : xr - 0x10000;  // boundary code (negative) where the face has no right cell
    const double n[3] = {fn.x, fn.y, fn.z};
    const double A = fc.w;
    const double rdtA = fast_rcp(dt * A);
    const double capL = sV[xl] * rdtA;
    // the face centre relative to the left cell is stored; relative to the right cell it is c - kappa w
    double capR = 0.0, rRx = 0.0, rRy = 0.0, rRz = 0.0;
    if (rin) {
      capR = sV[xr] * rdtA;
      rRx = fma(-fw.w, fw.x, fc.x); rRy = fma(-fw.w, fw.y, fc.y); rRz = fma(-fw.w, fw.z, fc.z);
    }
    const int xrr = rin ? xr : xl;
    if (!rin && r != RT_BC_REFLECT) bnd = 1;  // outflow or Dirichlet face: its flux enters a ledger
    // individual time steps: only a face with an active cell carries a flux
    const bool aL = !m.cact || (sAct[xl] & 1), aR = rin && (!m.cact || (sAct[xr] & 1));
    if (!(aL || aR)) {
#pragma unroll
      for (int g = 0; g < G; g++) { st2(sF + 2 * (2 * g * OM + s), 0.0, 0.0); st2(sF + 2 * ((2 * g + 1) * OM + s), 0.0, 0.0); }
      continue;
    }
    if (MIXED) {
      // single precision in the units l0 (lengths) and, per face and group, s (densities): reading S28
      const float *sGf = reinterpret_cast<const float *>(sG);
      const float nf[3] = {__double2float_rn(fn.x), __double2float_rn(fn.y), __double2float_rn(fn.z)};
      const float rLx = __double2float_rn(fc.x * m.il0), rLy = __double2float_rn(fc.y * m.il0), rLz = __double2float_rn(fc.z * m.il0);
      const float qRx = __double2float_rn(rRx * m.il0), qRy = __double2float_rn(rRy * m.il0), qRz = __double2float_rn(rRz * m.il0);
      const float ict = __fdiv_rn(1.0f, __double2float_rn(ct));
      const double rdt = fast_rcp(dt), Act = A * ct;
      const double photL = sV[xl] * rdt, photR = rin ? sV[xr] * rdt : 0.0;  // A |Phi_N| <= N V / dt (donor cap, S11)
#pragma unroll 1
      for (int g = 0; g < G; g++) {
        const double4 cl = ld4(sU + 4 * (xl * G + g));
        double4 cr = make_double4(0.0, 0.0, 0.0, 0.0);
        float iL[4] = {0.0f, 0.0f, 0.0f, 0.0f}, iR[4] = {0.0f, 0.0f, 0.0f, 0.0f}, UL[4], UR[4], J[4];
        if (SECOND && aL) increments_f(sGf + 12 * (xl * G + g), rLx, rLy, rLz, iL);
        UL[0] = __double2float_rn(cl.x) + iL[0]; UL[1] = __double2float_rn(cl.y) + iL[1];
        UL[2] = __double2float_rn(cl.z) + iL[2]; UL[3] = __double2float_rn(cl.w) + iL[3];
        if (rin) {
          cr = ld4(sU + 4 * (xrr * G + g));
          if (SECOND && aR) increments_f(sGf + 12 * (xrr * G + g), qRx, qRy, qRz, iR);
          UR[0] = __double2float_rn(cr.x) + iR[0]; UR[1] = __double2float_rn(cr.y) + iR[1];
          UR[2] = __double2float_rn(cr.z) + iR[2]; UR[3] = __double2float_rn(cr.w) + iR[3];
          // the jump: the cell values' part in double before rounding
          J[0] = __double2float_rn(cr.x - cl.x) + (iR[0] - iL[0]); J[1] = __double2float_rn(cr.y - cl.y) + (iR[1] - iL[1]);
          J[2] = __double2float_rn(cr.z - cl.z) + (iR[2] - iL[2]); J[3] = __double2float_rn(cr.w - cl.w) + (iR[3] - iL[3]);
        } else if (r == RT_BC_OUTFLOW) {
#pragma unroll
          for (int q = 0; q < 4; q++) { UR[q] = 0.0f; J[q] = -UL[q]; }
        } else if (r == RT_BC_REFLECT) {
          const float p = UL[1] * nf[0] + UL[2] * nf[1] + UL[3] * nf[2];
          UR[0] = UL[0]; J[0] = 0.0f;
#pragma unroll
          for (int a = 0; a < 3; a++) { J[1 + a] = -2.0f * p * nf[a]; UR[1 + a] = UL[1 + a] + J[1 + a]; }
        } else {
          const double4 gs = ld4(m.ghost + ((size_t)(RT_BC_DIRICHLET0 - r) * G + g) * 4);
          UR[0] = __double2float_rn(gs.x); UR[1] = __double2float_rn(gs.y); UR[2] = __double2float_rn(gs.z); UR[3] = __double2float_rn(gs.w);
          J[0] = __double2float_rn(gs.x - cl.x) - iL[0]; J[1] = __double2float_rn(gs.y - cl.y) - iL[1];
          J[2] = __double2float_rn(gs.z - cl.z) - iL[2]; J[3] = __double2float_rn(gs.w - cl.w) - iL[3];
        }
        float sc, is;
        unit_density(fmaxf(fabsf(UL[0]), fabsf(UR[0])), sc, is);
        const float nL = UL[0] * is, nR = UR[0] * is;
        const float fL[3] = {UL[1] * is * ict, UL[2] * is * ict, UL[3] * is * ict};
        const float fR[3] = {UR[1] * is * ict, UR[2] * is * ict, UR[3] * is * ict};
        float PL[3], PR[3];
        pressure_dot_n_f(nL, fL, nf, PL);
        pressure_dot_n_f(nR, fR, nf, PR);
        const float pn = 0.5f * ((fL[0] + fR[0]) * nf[0] + (fL[1] + fR[1]) * nf[1] + (fL[2] + fR[2]) * nf[2]) - 0.5f * (J[0] * is);
        const float p1 = 0.5f * (PL[0] + PR[0]) - 0.5f * (J[1] * is * ict), p2 = 0.5f * (PL[1] + PR[1]) - 0.5f * (J[2] * is * ict),
                    p3 = 0.5f * (PL[2] + PR[2]) - 0.5f * (J[3] * is * ict);
        // back to the caller's units and to double: A Phi_N = A c~ s phi_N, A Phi_F = A c~^2 s phi_F
        const double sN = Act * (double)sc, sFl = sN * ct;
        double aphi = (double)pn * sN;
        if (aphi > 0.0) aphi = dmin2(aphi, cl.x * photL);
        else if (rin) aphi = -dmin2(-aphi, cr.x * photR);
        st2(sF + 2 * (2 * g * OM + s), aphi, (double)p1 * sFl);
        st2(sF + 2 * ((2 * g + 1) * OM + s), (double)p2 * sFl, (double)p3 * sFl);
      }
    } else
#pragma unroll 1
    for (int g = 0; g < G; g++) {
      double UL[4], UR[4], NL, NR = 0.0;
      extrapolate<SECOND>(sU + 4 * (xl * G + g), sG + 12 * (xl * G + g), fc.x, fc.y, fc.z, UL, NL, aL);
      if (rin) extrapolate<SECOND>(sU + 4 * (xrr * G + g), sG + 12 * (xrr * G + g), rRx, rRy, rRz, UR, NR, aR);
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
      else if (rin) ph[0] = -dmin2(-ph[0], NR * capR);
      st2(sF + 2 * (2 * g * OM + s), A * ph[0], A * ph[1]);
      st2(sF + 2 * ((2 * g + 1) * OM + s), A * ph[2], A * ph[3]);
    }
  }
  __syncthreads();  // every owned slot holds its fluxes
  if (tl) tl[3] = now_ns();
  // the outgoing faces' fluxes go to xphi for the tiles of their right cells (k_finish)
  {
    double *xo = m.xphi + (size_t)(4 * G) * v.xbase;
    for (int k = tid; k < 2 * G * v.nout; k += nt) {
      const int j = k / (2 * G), c = k - j * (2 * G);
      *reinterpret_cast<double2 *>(xo + 2 * k) = ld2(sF + 2 * (c * OM + (int)v.outs[j]));  // chunk c = half c & 1 of group c >> 1
    }
  }
  // boundary ledgers: the number fluxes through the tile's outflow / Dirichlet faces, read back from
  // the slots; fixed-order block sums, one row per tile
  if (__syncthreads_or(bnd)) {
#pragma unroll
    for (int gg = 0; gg < G; gg++) {
      double b_out = 0.0, b_in = 0.0;
      for (int s = tid; s < v.nown; s += nt) {
        const int xr = (int)(v.slr[s] >> 16);
        if (xr < 0xFF00) continue;
        const int r = xr - 0x10000;
        const double aphi = sF[2 * (2 * gg * OM + s)];
        if (r == RT_BC_OUTFLOW) b_out += aphi;
        else if (r <= RT_BC_DIRICHLET0) b_in -= aphi;
      }
      const double so = block_sum(b_out, red), si = block_sum(b_in, red);
      if (tid == 0) { part_out[(size_t)tile * G + gg] = so; part_in[(size_t)tile * G + gg] = si; }
    }
  } else if (tid < G) {
    part_out[(size_t)tile * G + tid] = 0.0;
    part_in[(size_t)tile * G + tid] = 0.0;
  }

  // ---- a4: P lanes per (cell, group) gather the cell's faces (lane p takes entries p, p + P, ... of
  // the list, the partial sums are combined in a fixed order).  A cell all of whose faces are the
  // tile's is updated here; one with incoming faces leaves its partial sum in pacc for k_finish
  // (Uout may be U^n itself, which k_finish still needs)
  if (tl) tl[4] = now_ns();
  double fl[G];
#pragma unroll
  for (int gg = 0; gg < G; gg++) fl[gg] = 0.0;
  int floored = 0;
  const int P = nt >= 4 * m.TC * G ? 4 : (nt >= 2 * m.TC * G ? 2 : 1);
  const int nitem = v.ncell * G;
  for (int base = 0; base < nitem * P; base += nt) {  // (nt is a multiple of 32, P divides 32: whole warps iterate together)
    const int e = base + tid;
    const int item = e / P, p = e - item * P;
    const bool on = item < nitem;
    const int il = on ? item / G : 0, ig = on ? item - il * G : 0;
    const int h0 = on ? (int)v.ho[il] : 0, h1 = on ? (int)v.ho[il + 1] : 0;
    const double *pg = sF + 4 * ig * OM;  // half-planes 2 ig and 2 ig + 1
    // U^n of the cell (the stage buffer itself in stage 1): asked for now, needed after the sum
    const double4 u0 = on && p == 0 ? ld4(U0 + 4 * (v.c0 * G + item)) : make_double4(0, 0, 0, 0);
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    int incomplete = 0;
#pragma unroll 4
    for (int k = h0 + p; k < ((m.variant & 32) ? h0 : h1); k += P) {  // (variant 32: without the gather)
      const uint32_t w = v.hl[k];
      const int s = (int)(w & 0x7fffu);
      if (s >= v.nown) { incomplete = 1; continue; }  // incoming: its owner tile has the flux
      const double2 q01 = ld2(pg + 2 * s), q23 = ld2(pg + 2 * (OM + s));
      const double4 q = make_double4(q01.x, q01.y, q23.x, q23.y);
      const int sgn = (int)((w & 0x8000u) << 16);  // the flux leaves the left cell and enters the right one
      a0 += flip_sign(q.x, sgn); a1 += flip_sign(q.y, sgn); a2 += flip_sign(q.z, sgn); a3 += flip_sign(q.w, sgn);
    }
    for (int o = 1; o < P; o <<= 1) {
      a0 += __shfl_xor_sync(0xffffffffu, a0, o); a1 += __shfl_xor_sync(0xffffffffu, a1, o);
      a2 += __shfl_xor_sync(0xffffffffu, a2, o); a3 += __shfl_xor_sync(0xffffffffu, a3, o);
      incomplete |= __shfl_xor_sync(0xffffffffu, incomplete, o);
    }
    if (!on || p != 0) continue;
    const int ac = m.cact ? sAct[il] : 3;
    if (!(ac & 2)) {  // neither the cell nor a neighbour is active: it stays as it is, bit for bit
      if (!incomplete) { const double4 uc = ld4(sU + 4 * item); st4(Uout + 4 * (v.c0 * G + item), uc.x, uc.y, uc.z, uc.w); }
      continue;
    }
    if (incomplete) { st4(pacc + 4 * (v.c0 * G + item), a0, a1, a2, a3); continue; }
    const int32_t si = sSrc[il];
    const double src = si >= 0 && (ac & 5) == 1 ? srcrate[(size_t)ig * nsrc + si] : 0.0;  // (a passive cell injects nothing, nor does a ghost)
    const double add = finish_cell(a0, a1, a2, a3, sV[il], src, ld4(sU + 4 * item), u0, up,
                                   Uout + 4 * (v.c0 * G + item));
    if (add != 0.0) {
#pragma unroll
      for (int gg = 0; gg < G; gg++) if (gg == ig) fl[gg] += add;
      floored = 1;
    }
  }
  if (__syncthreads_or(floored)) {
#pragma unroll
    for (int gg = 0; gg < G; gg++) {
      const double t = block_sum(fl[gg], red);
      if (tid == 0) part_floor[(size_t)tile * G + gg] = t;
    }
  } else if (tid < G) part_floor[(size_t)tile * G + tid] = 0.0;
  if (m.tl) {  // (block-uniform)
    __syncthreads();
    if (tl) {
      unsigned sm;
      asm("mov.u32 %0, %smid;" : "=r"(sm));
      tl[5] = now_ns(); tl[6] = sm; tl[7] = blockIdx.x;
    }
  }
}

// a4 for the cells with incoming faces: pacc holds their partial sums (k_flux); subtract the
// incoming fluxes (the cell is their right cell) in list order and finish the update.
// One thread per (cell, group); part_floor: one row per block.
#define RT_FIN_BLOCK 128
template <int G>
__global__ void __launch_bounds__(RT_FIN_BLOCK) k_finish(int64_t n2, const int32_t *__restrict__ k2cell,
                                                         const int32_t *__restrict__ k2off, const int32_t *__restrict__ k2row,
                                                         const double *__restrict__ xphi, const double *__restrict__ pacc,
                                                         const double *__restrict__ cellV,
                                                         const double *__restrict__ Uin, const double *U0, double *Uout,
                                                         const int32_t *__restrict__ srcidx, const double *__restrict__ srcrate,
                                                         int nsrc, update_par up, double *__restrict__ part_floor,
                                                         const uint8_t *__restrict__ cact) {
  __shared__ double red[32];
  const int64_t item = (int64_t)blockIdx.x * RT_FIN_BLOCK + threadIdx.x;
  const int64_t k = item / G;
  const int g = (int)(item - k * G);
  double add = 0.0;
  const int ac = k < n2 && cact ? cact[k2cell[k]] : 3;
  if (k < n2 && !(ac & 2)) {  // neither the cell nor a neighbour is active: it stays as it is
    const int64_t i = k2cell[k];
    const double4 uc = ld4(Uin + 4 * (i * G + g));
    st4(Uout + 4 * (i * G + g), uc.x, uc.y, uc.z, uc.w);
  } else if (k < n2) {
    const int64_t i = k2cell[k];
    const int r0 = k2off[k], r1 = k2off[k + 1];
    double *out = Uout + 4 * (i * G + g);
    double4 a = ld4(pacc + 4 * (i * G + g));
    const double *xg = xphi + 4 * g;
#pragma unroll 4
    for (int r = r0; r < r1; r++) {
      const double4 p = ld4(xg + (size_t)(4 * G) * k2row[r]);
      a.x -= p.x; a.y -= p.y; a.z -= p.z; a.w -= p.w;
    }
    const int32_t si = srcidx[i];
    const double src = si >= 0 && (ac & 5) == 1 ? srcrate[(size_t)g * nsrc + si] : 0.0;
    add = finish_cell(a.x, a.y, a.z, a.w, cellV[i], src, ld4(Uin + 4 * (i * G + g)), ld4(U0 + 4 * (i * G + g)), up, out);
  }
  // fixed-order block sums per group
  const int any = __syncthreads_or(add != 0.0);
#pragma unroll
  for (int gg = 0; gg < G; gg++) {
    double t = 0.0;
    if (any) t = block_sum(g == gg ? add : 0.0, red);
    if (threadIdx.x == 0) part_floor[(size_t)blockIdx.x * G + gg] = t;
  }
}

// ------------------------------------------------------------------ ledgers
// acc[slot][g] += weight * sum_rows part[row][g].  Grid (G, jobs, RT_RED_BLOCKS): block z sums a
// fixed contiguous chunk of the rows (Neumaier per thread, fixed tree), the last block to finish
// adds the chunk sums in chunk order: the result does not depend on the scheduling.
__global__ void __launch_bounds__(1024) k_reduce(reduce_job j0, reduce_job j1, int G, rt_dev_ledger *led) {
  __shared__ double sm[1024];
  __shared__ bool last;
  reduce_job j = blockIdx.y == 0 ? j0 : j1;
  if (j.ncount) j.nrows = ((int64_t)*j.ncount + 31) / 32;
  if (j1.ncount) j1.nrows = ((int64_t)*j1.ncount + 31) / 32;
  const int g = blockIdx.x, y = blockIdx.y, z = blockIdx.z;
  // one job may be made of two partial-sum arrays: rows of the first, then rows of the second
  const bool two = gridDim.y == 1 && j1.part != j0.part;
  const int64_t n0 = j.nrows, ntot = n0 + (two ? j1.nrows : 0);
  const int64_t chunk = (ntot + RT_RED_BLOCKS - 1) / RT_RED_BLOCKS;
  const int64_t r0 = (int64_t)z * chunk, r1 = r0 + chunk < ntot ? r0 + chunk : ntot;
  double s = 0.0, c = 0.0;
  // rows r0 + tid, + 1024, ...: eight loads in flight, added in row order (a padding zero changes
  // neither the sum nor the compensation)
  for (int64_t r = r0 + threadIdx.x; r < r1; r += 8 * 1024) {
    double x[8];
#pragma unroll
    for (int u = 0; u < 8; u++) {
      const int64_t rr = r + 1024 * u;
      x[u] = rr < r1 ? (rr < n0 ? j.part[(size_t)rr * G + g] : j1.part[(size_t)(rr - n0) * G + g]) : 0.0;
    }
#pragma unroll
    for (int u = 0; u < 8; u++) {
      const double t = s + x[u];
      c += fabs(s) >= fabs(x[u]) ? (s - t) + x[u] : (x[u] - t) + s;
      s = t;
    }
  }
  sm[threadIdx.x] = s + c;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) sm[threadIdx.x] += sm[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    led->red_tmp[y][g][z] = sm[0];
    __threadfence();
    last = atomicAdd(&led->red_cnt[y][g], 1u) == RT_RED_BLOCKS - 1;
  }
  __syncthreads();
  if (!last || threadIdx.x != 0) return;
  __threadfence();
  led->red_cnt[y][g] = 0;
  double t = 0.0, tc = 0.0;
  for (int k = 0; k < RT_RED_BLOCKS; k++) {
    const double x = *(volatile double *)&led->red_tmp[y][g][k];
    const double u = t + x;
    tc += fabs(t) >= fabs(x) ? (t - u) + x : (x - u) + t;
    t = u;
  }
  const double total = t + tc;
  double *a = led->acc[j.slot][g];
  if (j.slot == 4) { a[0] = j.weight * total; a[1] = 0.0; }
  else {
    const double x = j.weight * total, u = a[0] + x;
    a[1] += fabs(a[0]) >= fabs(x) ? (a[0] - u) + x : (x - u) + a[0];
    a[0] = u;
  }
}

// stored photons per block: part[row][g] = sum_cells V N
template <int GG>
__global__ void __launch_bounds__(RT_BLOCK *GG) k_stored(int64_t C, const double *__restrict__ U,
                                                          const double *__restrict__ cellV, double *__restrict__ part,
                                                          const uint8_t *__restrict__ cact) {
  __shared__ double sm[GG][RT_BLOCK / 32];
  const int64_t i = (int64_t)blockIdx.x * RT_BLOCK + threadIdx.x;
  const int g = threadIdx.y;
  double v = i < C && !(cact && (cact[i] & 4)) ? cellV[i] * U[((size_t)i * GG + g) * 4] : 0.0;  // (a ghost's photons are its owner's)
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

// ------------------------------------------------------------------ active sets (individual time steps)
__global__ void k_active_in(int64_t C, const int32_t *__restrict__ perm, const uint8_t *__restrict__ active, uint8_t *__restrict__ ain) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p < C) ain[p] = active[perm[p]] & 3;  // bit 0 active, bit 1 ghost (rt_set_active)
}
// one block per tile, straight from the tile's tables in global memory: cact = active | touched << 1 | ghost << 2 per cell
// (touched: the cell or a cell across one of its faces is active), tact = OR over the tile's cells
__global__ void __launch_bounds__(128) k_touched(rt_geom m, const uint8_t *__restrict__ ain, uint8_t *__restrict__ cact, uint8_t *__restrict__ tact) {
  __shared__ int s_or;
  const int64_t t = blockIdx.x;
  const uint32_t *B = m.blob + (size_t)t * m.bstride;
  const rt_tile d = *reinterpret_cast<const rt_tile *>(B);
  const int64_t c0 = t * m.TC;
  const int ncell = (int)(c0 + m.TC < m.C ? m.TC : m.C - c0);
  const uint32_t *ho = B + RT_BLOB_HEAD, *hl = ho + m.TC + 1, *halo = hl + d.nhf + d.nown;
  if (threadIdx.x == 0) s_or = 0;
  __syncthreads();
  for (int x = threadIdx.x; x < ncell; x += blockDim.x) {
    const int a = ain[c0 + x];
    int f = a & 1;
    const int ghost = (a >> 1) & 1;  // a ghost is never updated here: its owner does that, rt_halo_unpack brings the result
    int touched = f;
    for (uint32_t k = ho[x]; k < ho[x + 1] && !touched; k++) {
      const uint32_t nb = hl[k] >> 16;
      if (nb >= 0xFF00u) continue;
      const int64_t id = nb < (uint32_t)m.TC ? c0 + nb : (int64_t)halo[nb - m.TC];
      touched |= ain[id] & 1;
    }
    f |= (ghost ? 0 : touched << 1) | (ghost << 2);
    cact[c0 + x] = (uint8_t)f;
    // per tile: bit 0 = a cell whose gradient is computed here, bit 1 = a cell one of whose faces carries a flux
    // (a ghost's too: the tile that owns the face evaluates it for the cell on the other side)
    const int ft = (ghost ? 0 : f & 1) | (touched << 1);
    if (ft) atomicOr(&s_or, ft);
  }
  __syncthreads();
  if (threadIdx.x == 0) tact[t] = (uint8_t)s_or;
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
#define K_GRAD(g) k_grad<g, false>
#define K_GRADM(g) k_grad<g, true>
#define K_FLUX2(g) k_flux<g, true, false>
#define K_FLUX1(g) k_flux<g, false, false>
#define K_FLUX2M(g) k_flux<g, true, true>
#define K_FLUX1M(g) k_flux<g, false, true>
#define K_FINISH(g) k_finish<g>
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
  // the opt-in is per kernel, not per context: several contexts with different tile capacities may live in one
  // process (the shards of shard.LocalGroup), so every kernel is allowed the most a block may have
  if (rt_smem_grad(c->TC, c->G, c->smax, c->hmax, c->bstride) > RT_SMEM_MAX - 1024 || rt_smem_flux(c->TC, c->G, c->omax, c->fmax, c->bstride) > RT_SMEM_MAX - 1024)
    return rt_fail(c, RT_EMESH, "a tile needs more shared memory than one block may have");
  const size_t sg = RT_SMEM_MAX - 1024, ss = RT_SMEM_MAX - 1024;  // (less the kernels' static shared memory)
  SET_SMEM_G(c->G, K_GRAD, sg, e);
  if (e == cudaSuccess) SET_SMEM_G(c->G, K_FLUX2, ss, e);
  if (e == cudaSuccess) SET_SMEM_G(c->G, K_FLUX1, ss, e);
  if (e == cudaSuccess) SET_SMEM_G(c->G, K_GRADM, sg, e);
  if (e == cudaSuccess) SET_SMEM_G(c->G, K_FLUX2M, ss, e);
  if (e == cudaSuccess) SET_SMEM_G(c->G, K_FLUX1M, ss, e);
  if (e != cudaSuccess) return rt_fail(c, RT_ECUDA, "cudaFuncSetAttribute(shared memory): %s", cudaGetErrorString(e));
  return RT_OK;
}

// threads per tile block (a whole number of warps, at most 256, the kernels' launch bound).
// k_grad has one thread per (cell, group); k_stage one lane per (slot, group), several passes.
// rt_tuning.flux_threads / grad_threads override the defaults for experiments.
static int round_threads(int n) { n = ((n + 31) / 32) * 32; return n > 256 ? 256 : (n < 32 ? 32 : n); }
static int tile_threads(const rt_ctx *c) { return round_threads(c->tun.flux_threads > 0 ? c->tun.flux_threads : 256); }
static int grad_threads(const rt_ctx *c) {  // four lanes per cell, at most k_grad's launch bound
  const int n = round_threads(c->tun.grad_threads > 0 ? c->tun.grad_threads : 4 * c->TC);
  return n > 128 ? 128 : n;
}

rt_geom rt_geom_of(const rt_ctx *c) {
  const rt_layout &l = c->lay;
  rt_geom m;
  m.C = c->C; m.F = c->F; m.G = c->G; m.TC = c->TC; m.smax = c->smax; m.omax = c->omax; m.hmax = c->hmax; m.fmax = c->fmax; m.bmax = c->bmax; m.bstride = c->bstride;
  m.cellV = rt_ptr<double>(c, l.cellV); m.Minv = rt_ptr<double>(c, l.Minv);
  m.faceC = rt_ptr<double>(c, l.faceC); m.faceN = rt_ptr<double>(c, l.faceN); m.faceW = rt_ptr<double>(c, l.faceW);
  m.tiles = rt_ptr<rt_tile>(c, l.tiles); m.blob = rt_ptr<uint32_t>(c, l.blob);
  m.xphi = rt_ptr<double>(c, l.xphi);
  m.variant = c->tun.variant;
  m.cact = c->has_active ? rt_ptr<uint8_t>(c, l.cact) : nullptr;
  m.tact = c->has_active ? rt_ptr<uint8_t>(c, l.tact) : nullptr;
  m.tl = c->dbg_tl;
  m.il0 = 1.0 / c->l0; m.l0sq = c->l0 * c->l0;
  m.prefetch_tiles = c->tun.prefetch_tiles > 0 ? c->tun.prefetch_tiles : (c->tun.prefetch_tiles < 0 ? (1 << 30) : 600);
  m.ghost = rt_ptr<double>(c, l.ghost);
  for (int a = 0; a < 3; a++) { m.box[a] = c->box[a]; m.per[a] = c->per[a]; }
  return m;
}

// the two tile classes of a kernel: class A (most tiles) with the smaller capacities, class B with the maxima
static void launch_grad(rt_ctx *c, rt_geom m, const double *U, double *grad) {
  m.tlist = rt_ptr<int32_t>(c, c->lay.tlistG);
  for (int cls = 0; cls < 2; cls++) {
    const int64_t n = cls == 0 ? c->nGA : c->T - c->nGA;
    if (n <= 0) continue;
    m.tbase = cls == 0 ? 0 : c->nGA;
    m.smax = cls == 0 ? c->smaxA : c->smax; m.hmax = cls == 0 ? c->hmaxA : c->hmax;
    const size_t sg = rt_smem_grad(c->TC, c->G, m.smax, m.hmax, c->bstride);
    if (c->par.mixed) {
      DISPATCH_G(c->G, K_GRADM, (unsigned)n, grad_threads(c), sg, c->stream, m, U, grad);
    } else {
      DISPATCH_G(c->G, K_GRAD, (unsigned)n, grad_threads(c), sg, c->stream, m, U, grad);
    }
    c->launches++;
  }
}

int rt_launch_gradients(rt_ctx *c, const double *U) {
  launch_grad(c, rt_geom_of(c), U, rt_ptr<double>(c, c->lay.grad));
  return RT_OK;
}

void rt_reduce2(rt_ctx *c, reduce_job a, reduce_job b, int njobs) {
  rt_prof_begin(c, RT_K_REDUCE);
  k_reduce<<<dim3(c->G, njobs, RT_RED_BLOCKS), 1024, 0, c->stream>>>(a, b, c->G, rt_ptr<rt_dev_ledger>(c, c->lay.led));
  rt_prof_end(c);
  c->launches++;
}

// one Heun stage: Uout = ca*U0 + cb*(Uin + dt R(Uin)); ledger weights wl (fluxes), wf (floor).
// parts: 1 = the gradient pass (a2), 2 = fluxes and update (a3 + a4), 3 = both; a sharded run exchanges the
// ghosts' gradients between the two (rt_step_phase)
static void stage(rt_ctx *c, const double *Uin, const double *U0, double *Uout, double ca, double cb, double dt,
                  double wl, double wf, int parts = 3) {
  const rt_layout &l = c->lay;
  const rt_geom m = rt_geom_of(c);
  const int G = c->G;
  double *grad = rt_ptr<double>(c, l.grad);
  double *part = rt_ptr<double>(c, l.part);
  const int64_t nchem = blocks_for(c->C, RT_CHEM_BLOCK);
  const int64_t nfin = (c->n2 * G + RT_FIN_BLOCK - 1) / RT_FIN_BLOCK;
  double *p_floor = part + (size_t)G * nchem * RT_CHEM_MAXPASS, *p_out = p_floor + (size_t)G * c->T, *p_in = p_out + (size_t)G * c->T;
  double *p_floor2 = p_in + (size_t)G * c->T;
  const int nt = tile_threads(c);
  const update_par up = {ca, cb, dt, c->par.ctilde, c->par.n_floor};
  double *pacc = rt_ptr<double>(c, l.pacc);
  const int32_t *srcidx = rt_ptr<int32_t>(c, l.srcidx);
  const double *srcrate = rt_ptr<double>(c, l.srcrate);
  if (c->par.order >= 2 && (parts & 1)) {
    rt_prof_begin(c, RT_K_GRAD);
    launch_grad(c, m, Uin, grad);
    rt_prof_end(c);
  }
  if (!(parts & 2)) return;
  rt_prof_begin(c, RT_K_FLUX);
  {
    rt_geom mf = m;
    mf.tlist = rt_ptr<int32_t>(c, l.tlistF);
    for (int cls = 0; cls < 2; cls++) {
      const int64_t n = cls == 0 ? c->nFA : c->T - c->nFA;
      if (n <= 0) continue;
      mf.tbase = cls == 0 ? 0 : c->nFA;
      mf.omax = cls == 0 ? c->omaxA : c->omax; mf.fmax = cls == 0 ? c->fmaxA : c->fmax;
      const size_t sf = rt_smem_flux(c->TC, G, mf.omax, mf.fmax, c->bstride, c->par.mixed != 0);
      if (c->par.mixed && c->par.order >= 2) {
        DISPATCH_G(G, K_FLUX2M, (unsigned)n, nt, sf, c->stream, mf, Uin, grad, U0, Uout, srcidx, srcrate, c->nsrc, up, pacc, p_floor, p_out, p_in);
      } else if (c->par.mixed) {
        DISPATCH_G(G, K_FLUX1M, (unsigned)n, nt, sf, c->stream, mf, Uin, grad, U0, Uout, srcidx, srcrate, c->nsrc, up, pacc, p_floor, p_out, p_in);
      } else if (c->par.order >= 2) {
        DISPATCH_G(G, K_FLUX2, (unsigned)n, nt, sf, c->stream, mf, Uin, grad, U0, Uout, srcidx, srcrate, c->nsrc, up, pacc, p_floor, p_out, p_in);
      } else {
        DISPATCH_G(G, K_FLUX1, (unsigned)n, nt, sf, c->stream, mf, Uin, grad, U0, Uout, srcidx, srcrate, c->nsrc, up, pacc, p_floor, p_out, p_in);
      }
      c->launches++;
    }
  }
  rt_prof_end(c);
  if (nfin > 0) {
    rt_prof_begin(c, RT_K_UPDATE);
    DISPATCH_G(G, K_FINISH, (unsigned)nfin, RT_FIN_BLOCK, 0, c->stream, c->n2, rt_ptr<int32_t>(c, l.k2cell),
               rt_ptr<int32_t>(c, l.k2off), rt_ptr<int32_t>(c, l.k2row), m.xphi, pacc, m.cellV, Uin, U0, Uout, srcidx, srcrate, c->nsrc, up,
               p_floor2, m.cact);
    rt_prof_end(c);
    c->launches++;
  }
  rt_reduce2(c, {p_out, c->T, wl * dt, 1, nullptr}, {p_in, c->T, wl * dt, 2, nullptr}, 2);
  rt_reduce2(c, {p_floor, c->T, wf, 3, nullptr}, {nfin > 0 ? p_floor2 : p_floor, nfin, wf, 3, nullptr}, 1);
}

// the phases of one subcycle, in order (rt_step_phase; rt_step runs them back to back):
// 0 chemistry, 1 gradients of U^n, 2 fluxes + update of stage 1, 3 gradients of U^1, 4 fluxes + update of stage 2
// (Heun off: 0, 1, 2).  parts = bit mask of the phases to run.
static void run_phases(rt_ctx *c, double dt, int parts) {
  rt_layout &l = c->lay;
  double *Ua = rt_ptr<double>(c, l.Ua), *Ub = rt_ptr<double>(c, l.Ub);
  if ((parts & 1) && c->par.chem_mode != RT_CHEM_NONE) {
    rt_chem_par P;
    P.ctilde = c->par.ctilde; P.y_he = c->par.y_he; P.T_fixed = c->par.T_fixed;
    P.alphaB_override = c->par.alphaB_override; P.f_accept = c->par.f_accept; P.f_target = c->par.f_target;
    P.x_floor_rel = c->par.x_floor_rel; P.max_substeps = c->par.max_substeps;
    for (int g = 0; g < RT_MAXG; g++)
      for (int j = 0; j < 3; j++) { P.sigma[g][j] = c->par.sigma[g][j]; P.eps[g][j] = c->par.eps_heat[g][j]; }
    rt_launch_chem(c, P, dt, Ua);
  }
  const int s1 = (parts >> 1) & 3, s2 = (parts >> 3) & 3;
  if (c->par.heun) {
    if (s1) stage(c, Ua, Ua, Ub, 0.0, 1.0, dt, 0.5, 0.5, s1);  // U1 = enforce(Un + dt R(Un))
    if (s2) stage(c, Ub, Ua, Ua, 0.5, 0.5, dt, 0.5, 1.0, s2);  // Un+1 = enforce(Un/2 + (U1 + dt R(U1))/2)
  } else {
    if (s1) stage(c, Ua, Ua, Ub, 0.0, 1.0, dt, 1.0, 1.0, s1);
    if (s1 & 2) { size_t t = l.Ua; l.Ua = l.Ub; l.Ub = t; }  // the new state lives in the other buffer
  }
}

int rt_launch_phase(rt_ctx *c, double dt, int phase) {
  run_phases(c, dt, 1 << phase);
  const int last = c->par.heun ? 4 : 2;
  if (phase == last) {
    for (int g = 0; g < c->G; g++) {  // injected photons: host-side compensated sum
      double *a = c->injected[g];
      const double x = dt * c->src_total[g], t = a[0] + x;
      a[1] += fabs(a[0]) >= fabs(x) ? (a[0] - t) + x : (x - t) + a[0];
      a[0] = t;
    }
    c->nsub_done++;
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return rt_fail(c, RT_ECUDA, "kernel launch: %s", cudaGetErrorString(e));
  return RT_OK;
}

int rt_launch_step(rt_ctx *c, double dt) {
  double tot[RT_MAXG];
  for (int g = 0; g < c->G; g++) tot[g] = dt * c->src_total[g];
  run_phases(c, dt, c->par.heun ? 31 : 7);
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

int rt_launch_active(rt_ctx *c, const uint8_t *active_dev) {
  const rt_layout &l = c->lay;
  uint8_t *ain = rt_ptr<uint8_t>(c, l.pacc);  // C bytes of scratch: pacc is free between steps
  k_active_in<<<blocks_for(c->C, 256), 256, 0, c->stream>>>(c->C, rt_ptr<int32_t>(c, l.perm), active_dev, ain);
  k_touched<<<(unsigned)c->T, 128, 0, c->stream>>>(rt_geom_of(c), ain, rt_ptr<uint8_t>(c, l.cact), rt_ptr<uint8_t>(c, l.tact));
  c->launches += 2;
  return RT_OK;
}

int rt_launch_stored(rt_ctx *c) {
  const rt_layout &l = c->lay;
  double *part = rt_ptr<double>(c, l.part);
  DISPATCH_G(c->G, K_STORED, (unsigned)l.nbc, dim3(RT_BLOCK, c->G), 0, c->stream, c->C, rt_ptr<double>(c, l.Ua),
             rt_ptr<double>(c, l.cellV), part, c->has_active ? rt_ptr<uint8_t>(c, l.cact) : nullptr);
  c->launches++;
  rt_reduce2(c, {part, l.nbc, 1.0, 4, nullptr}, {part, l.nbc, 1.0, 4, nullptr}, 1);
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

// ------------------------------------------------------------------ halo exchange of a sharded run (rt_halo_pack / rt_halo_unpack)
// rows of 16-byte chunks: buf[k][:] <-> field[iperm[cells[k]]][:]; one thread per (row, chunk)
template <bool PACK>
__global__ void __launch_bounds__(256) k_halo_rows(int64_t n, int chunks, const int32_t *__restrict__ cells, const int32_t *__restrict__ iperm,
                                                   double2 *field, double2 *buf) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n * chunks) return;
  const int64_t k = e / chunks;
  const int ch = (int)(e - k * chunks);
  const int64_t p = iperm[cells[k]];
  if (PACK) buf[e] = field[p * chunks + ch];
  else field[p * chunks + ch] = buf[e];
}

int rt_launch_halo(rt_ctx *c, bool pack, void *field, int row_bytes, int64_t n, const int32_t *cells_dev, void *buf_dev) {
  if (n <= 0) return RT_OK;
  const int chunks = row_bytes / 16;
  const unsigned nb = blocks_for(n * chunks, 256);
  const int32_t *iperm = rt_ptr<int32_t>(c, c->lay.iperm);
  if (pack) k_halo_rows<true><<<nb, 256, 0, c->stream>>>(n, chunks, cells_dev, iperm, (double2 *)field, (double2 *)buf_dev);
  else k_halo_rows<false><<<nb, 256, 0, c->stream>>>(n, chunks, cells_dev, iperm, (double2 *)field, (double2 *)buf_dev);
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return rt_fail(c, RT_ECUDA, "kernel launch: %s", cudaGetErrorString(e));
  return RT_OK;
}
