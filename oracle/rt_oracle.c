/* TEST INFRASTRUCTURE — NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded fp64 CPU oracle of one AREPO-RT radiative-transfer subcycle,
 * written from /root/reference/PAPER.md (arXiv 2404.17630) with the readings S1-S24 listed
 * in DESIGN.md section 3 where the paper is silent.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA path (paper_2404_17630_b200/csrc).
 *
 * The method is an explicit finite-volume iteration plus a sub-stepped ODE update, so the
 * oracle is the algorithm written out in the paper's order (Fig. 1):
 *   O1 thermochemistry over dt per cell       PAPER.md:125-127 (semi-implicit), 236-238 (sub-steps)
 *   O2 two-stage Heun over dt of  R(U)        north_star (paper names no integrator: reading S3)
 *   O3 gradients + slope limiter              PAPER.md:137-151, eqs (13)-(15)
 *   O4 face flux: extrapolate, rotate into the face frame, GLF/M1 Riemann flux, rotate back,
 *      donor cap                              PAPER.md:153-155, eqs (6)-(10)
 *   O5 apply fluxes + sources to the cells
 * No blocking, fusion or reordering: loops over cells, faces of a cell, groups.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P1 Stroemgren law, P2 budget identity,
 * P3 invariants, P4 beam speed, P5 2x2x2 brute force in numpy, P6 linear-exact gradients,
 * P8 stationarity, P9 rotation covariance, P10 closure values, P11 chemistry closed forms,
 * P12 travelling wave, P13 restart, P14 H II region, P15 one tiny sub-step = state + h RHS (helium solve,
 * heating shares, every cooling term), P16 helium closed forms, P17 photo-heating alone, P18 fixed
 * opacity halves exactly, P19 the donor cap active on a three-cell chain by hand, P20 active / passive
 * cells, P21 the mixed-precision mode against the fp64 path (1e-6 per step), exact scale covariance,
 * differences formed in double.  No function is "parity unpinned"; the one unpinnable choice is a reading (S23).
 * section 5.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define K_BOLTZ 1.380649e-16
#define T_MIN 10.0

enum { CHEM_NONE = 0, CHEM_FIXED_OPACITY = 1, CHEM_H_ISOTHERMAL = 2, CHEM_HHE_THERMAL = 3 };
enum { BC_OUTFLOW = -1, BC_REFLECT = -2, BC_DIRICHLET0 = -3 };
/* ledger rows per group */
enum { L_STORED = 0, L_INJECTED, L_ABSORBED, L_OUTFLOW, L_INFLOW_BC, L_FLOOR, L_NROW };

typedef struct {
  double s, c; /* Neumaier compensated sum */
} ksum;
static void kadd(ksum *k, double x) {
  double t = k->s + x;
  if (fabs(k->s) >= fabs(x)) k->c += (k->s - t) + x; else k->c += (x - t) + k->s;
  k->s = t;
}
static double kval(const ksum *k) { return k->s + k->c; }

typedef struct oracle_ctx {
  int64_t C, F;
  int G;
  double box[3];
  int periodic[3];
  const double *volume, *centroid, *area, *normal, *fcentroid; /* borrowed copies below */
  const int32_t *left, *right;
  double *own_d; int32_t *own_i;
  int nghost; double *ghost; /* [nghost][4G] */
  /* CSR of half-faces */
  int64_t *off; int32_t *hf_face; int8_t *hf_side; /* side +1: cell is left, -1: right */
  double *hf_w;     /* [nhf][3]  (A/|d|) n_hat, eq (15) second-term prefactor */
  double *hf_r;     /* [nhf][3]  face centroid minus cell centroid (min image)               */
  double *Minv;     /* [C][9]    inverse of sum_f A n_hat n_hat^T, eq (15) first term        */
  /* params */
  double ctilde, sigma[3 * 8], eps[3 * 8], T_fixed, alphaB_override, y_he, f_accept, f_target, x_floor_rel, n_floor;
  int chem_mode, order, heun; int64_t max_substeps;
  int mixed;         /* 1: single-precision primitives (reading S28) */
  float *gNf, *gFf;  /* mixed mode: limited gradients times the cell size, [G][3][C] and [G][3][3][C] */
  double *kappa;
  /* active set of the RT step (reading S27): NULL = every cell is active */
  uint8_t *active;
  uint8_t *touched; /* active, or sharing an interface with an active cell: the cells an RT step may change */
  /* sources */
  int nsrc; int32_t *src_cell; double *src_rate; /* [G][nsrc] */
  /* state: N[G][C], Fl[G][3][C] */
  double *N, *Fl, *xHII, *xHeII, *xHeIII, *eth, *nH;
  /* work */
  double *gN, *gF;   /* gN[G][3][C], gF[G][3(comp)][3(dir)][C] */
  double *phi;       /* face flux [F][G][4] */
  double *N0, *Fl0;
  ksum led[8][L_NROW];
  int64_t substeps_total, substeps_max, cells_hit_cap;
} oracle_ctx;

/* ------------------------------------------------------------------ small helpers */
static double minimg(double d, double L, int per) { return per ? d - L * rint(d / L) : d; }

static int inv3(const double m[9], double o[9]) {
  double c00 = m[4] * m[8] - m[5] * m[7], c01 = m[5] * m[6] - m[3] * m[8], c02 = m[3] * m[7] - m[4] * m[6];
  double det = m[0] * c00 + m[1] * c01 + m[2] * c02;
  if (det == 0.0) return -1;
  double id = 1.0 / det;
  o[0] = c00 * id; o[1] = (m[2] * m[7] - m[1] * m[8]) * id; o[2] = (m[1] * m[5] - m[2] * m[4]) * id;
  o[3] = c01 * id; o[4] = (m[0] * m[8] - m[2] * m[6]) * id; o[5] = (m[2] * m[3] - m[0] * m[5]) * id;
  o[6] = c02 * id; o[7] = (m[1] * m[6] - m[0] * m[7]) * id; o[8] = (m[0] * m[4] - m[1] * m[3]) * id;
  return 0;
}

/* ------------------------------------------------------------------ M1 closure (S1)
 * Eq (9): P = E D.  The paper defers the M1 formula to Kannan+19; reading S1 is the
 * Levermore form: f = |F|/(c N) clamped to [0,1], chi = (3+4f^2)/(5+2 sqrt(4-3f^2)),
 * D = (1-chi)/2 I + (3chi-1)/2 n n^T, n = F/|F|. */
double oracle_chi(double f) {
  if (f > 1.0) f = 1.0;
  if (f < 0.0) f = 0.0;
  return (3.0 + 4.0 * f * f) / (5.0 + 2.0 * sqrt(4.0 - 3.0 * f * f));
}

void oracle_eddington(double N, const double Fv[3], double ctilde, double D[9]) {
  double fn = sqrt(Fv[0] * Fv[0] + Fv[1] * Fv[1] + Fv[2] * Fv[2]);
  double den = ctilde * N;
  if (den < 1e-300) den = 1e-300;
  double f = fn / den;
  double chi = oracle_chi(f);
  double a = 0.5 * (1.0 - chi), b = 0.5 * (3.0 * chi - 1.0);
  for (int i = 0; i < 9; i++) D[i] = 0.0;
  D[0] = D[4] = D[8] = a;
  if (fn > 0.0) {
    double n[3] = {Fv[0] / fn, Fv[1] / fn, Fv[2] / fn};
    for (int i = 0; i < 3; i++)
      for (int j = 0; j < 3; j++) D[3 * i + j] += b * n[i] * n[j];
  }
}

/* ------------------------------------------------------------------ O4: Riemann flux at one face
 * rotate the face states so the normal is the x-axis, solve, rotate back.
 * Riemann solver = global Lax-Friedrichs with signal speed ctilde (reading S2) on the flux
 * function of eq (10): F(U) = (F_r, c^2 P_r).
 * UL, UR = (N, Fx, Fy, Fz); n = unit normal L->R; out = (Phi_N, Phi_Fx, Phi_Fy, Phi_Fz) in the lab frame. */
void oracle_riemann(const double UL[4], const double UR[4], const double n[3], double ctilde, double out[4]) {
  /* orthonormal frame (n, t1, t2): t1 = n x e_k / |.| with e_k the axis of the smallest |n_k| */
  int k = 0;
  if (fabs(n[1]) < fabs(n[k])) k = 1;
  if (fabs(n[2]) < fabs(n[k])) k = 2;
  double e[3] = {0, 0, 0};
  e[k] = 1.0;
  double t1[3] = {n[1] * e[2] - n[2] * e[1], n[2] * e[0] - n[0] * e[2], n[0] * e[1] - n[1] * e[0]};
  double l1 = sqrt(t1[0] * t1[0] + t1[1] * t1[1] + t1[2] * t1[2]);
  t1[0] /= l1; t1[1] /= l1; t1[2] /= l1;
  double t2[3] = {n[1] * t1[2] - n[2] * t1[1], n[2] * t1[0] - n[0] * t1[2], n[0] * t1[1] - n[1] * t1[0]};
  double FL[3], FR[3];
  FL[0] = UL[1] * n[0] + UL[2] * n[1] + UL[3] * n[2];
  FL[1] = UL[1] * t1[0] + UL[2] * t1[1] + UL[3] * t1[2];
  FL[2] = UL[1] * t2[0] + UL[2] * t2[1] + UL[3] * t2[2];
  FR[0] = UR[1] * n[0] + UR[2] * n[1] + UR[3] * n[2];
  FR[1] = UR[1] * t1[0] + UR[2] * t1[1] + UR[3] * t1[2];
  FR[2] = UR[1] * t2[0] + UR[2] * t2[1] + UR[3] * t2[2];
  double DL[9], DR[9];
  oracle_eddington(UL[0], FL, ctilde, DL);
  oracle_eddington(UR[0], FR, ctilde, DR);
  double ph[4];
  ph[0] = 0.5 * (FL[0] + FR[0]) - 0.5 * ctilde * (UR[0] - UL[0]);
  for (int a = 0; a < 3; a++) {
    double PLx = UL[0] * DL[3 * a + 0], PRx = UR[0] * DR[3 * a + 0]; /* P e_x */
    ph[1 + a] = 0.5 * ctilde * ctilde * (PLx + PRx) - 0.5 * ctilde * (FR[a] - FL[a]);
  }
  out[0] = ph[0];
  for (int a = 0; a < 3; a++) out[1 + a] = ph[1] * n[a] + ph[2] * t1[a] + ph[3] * t2[a];
}

/* ------------------------------------------------------------------ rate coefficients (S21, DESIGN.md appendix A)
 * r[0..2]  alpha_B  HII, HeII, HeIII   [cm^3/s]
 * r[3..5]  beta     HI, HeI, HeII      [cm^3/s]
 * r[6..8]  recombination cooling HII, HeII, HeIII [erg cm^3/s]
 * r[9..11] collisional-ionisation cooling HI, HeI, HeII
 * r[12..13] collisional-excitation cooling HI, HeII
 * r[14]    bremsstrahlung coefficient 1.42e-27 g_ff sqrt(T) */
static double alphaB_H_fit(double lam) { return 2.753e-14 * pow(lam, 1.5) / pow(1.0 + pow(lam / 2.74, 0.407), 2.242); }
static double rcool_H_fit(double T, double lam) {
  return 3.435e-30 * T * pow(lam, 1.970) / pow(1.0 + pow(lam / 2.250, 0.376), 3.720);
}
void oracle_rates(double T, double r[15]) {
  const double THI = 157807.0, THeI = 285335.0, THeII = 631515.0;
  double lHI = 2.0 * THI / T, lHeI = 2.0 * THeI / T, lHeII = 2.0 * THeII / T;
  double sq = sqrt(T), q = 1.0 / (1.0 + sqrt(T / 1.0e5));
  r[0] = alphaB_H_fit(lHI);
  r[1] = 1.26e-14 * pow(lHeI, 0.75);
  r[2] = 2.0 * alphaB_H_fit(lHeII);
  r[3] = 5.85e-11 * sq * exp(-157809.1 / T) * q;
  r[4] = 2.38e-11 * sq * exp(-285335.4 / T) * q;
  r[5] = 5.68e-12 * sq * exp(-631515.0 / T) * q;
  r[6] = rcool_H_fit(T, lHI);
  r[7] = K_BOLTZ * T * r[1];
  r[8] = 8.0 * rcool_H_fit(T, lHeII);
  r[9] = 1.27e-21 * sq * exp(-157809.1 / T) * q;
  r[10] = 9.38e-22 * sq * exp(-285335.4 / T) * q;
  r[11] = 4.95e-22 * sq * exp(-631515.0 / T) * q;
  r[12] = 7.50e-19 * exp(-118348.0 / T) * q;
  r[13] = 5.54e-17 * pow(T, -0.397) * exp(-473638.0 / T) * q;
  double lt = log10(T);
  double gff = 1.1 + 0.34 * exp(-(5.5 - lt) * (5.5 - lt) / 3.0);
  r[14] = 1.42e-27 * gff * sq;
}

/* ------------------------------------------------------------------ O1: chemistry of one cell over dt
 * Semi-implicit update (everything implicit except the thermal energy) with the
 * adaptive sub-stepping of PAPER.md:238.  The scheme's formulas are reading S17 (C1-C8).
 * par: ctilde, y_he, T_fixed, alphaB_override, f_accept, f_target, x_floor_rel
 * st (in/out): N[G], F[3G] (g-major: Fx,Fy,Fz per group), xHII, xHeII, xHeIII, eth; nH fixed.
 * trace (optional): [ntrace_max][3] rows (h, f, accepted). Returns attempts; *hit_cap set if capped. */
typedef struct {
  double N[8], F[24], xHII, xHeII, xHeIII, e;
} chem_state;

static double chem_try(const oracle_ctx *c, const chem_state *s, double nH, double h, chem_state *o) {
  const int G = c->G;
  const double y = c->y_he, nHe = y * nH;
  const int thermal = (c->chem_mode == CHEM_HHE_THERMAL);
  /* C1 */
  double xe = s->xHII + y * (s->xHeII + 2.0 * s->xHeIII);
  double ne = nH * xe;
  double ntot = nH * (1.0 + y + xe);
  double T = thermal ? (2.0 / 3.0) * s->e / (K_BOLTZ * ntot) : c->T_fixed;
  /* C2 */
  double r[15];
  oracle_rates(T, r);
  if (c->alphaB_override > 0.0) r[0] = c->alphaB_override;
  /* C3: photons, implicit in N with absorbers frozen at the start of the sub-step */
  double nj[3] = {nH * (1.0 - s->xHII), nHe * (1.0 - s->xHeII - s->xHeIII), nHe * s->xHeII};
  double P[3] = {0, 0, 0}, heat = 0.0;
  for (int g = 0; g < G; g++) {
    double k = 0.0;
    for (int j = 0; j < 3; j++) k += c->sigma[3 * g + j] * nj[j];
    double D = c->ctilde * k;
    double Nn = s->N[g] / (1.0 + h * D);
    o->N[g] = Nn;
    for (int a = 0; a < 3; a++) o->F[3 * g + a] = s->F[3 * g + a] / (1.0 + h * D);
    double dN = s->N[g] - Nn;
    if (k > 0.0)
      for (int j = 0; j < 3; j++) {
        double share = dN * (c->sigma[3 * g + j] * nj[j]) / k;
        P[j] += share;
        heat += share * c->eps[3 * g + j];
      }
  }
  /* C4: hydrogen, backward Euler with n_e frozen */
  double nHII = nH * s->xHII;
  double nHIIn = (nHII + P[0] + h * r[3] * ne * nH) / (1.0 + h * ne * (r[3] + r[0]));
  if (nHIIn < 0.0) nHIIn = 0.0;
  if (nHIIn > nH) nHIIn = nH;
  o->xHII = nHIIn / nH;
  /* C5: helium, backward Euler, 2x2 solve for a = n_HeI', cc = n_HeIII' */
  double nHeIn = 0.0, nHeIIn = 0.0, nHeIIIn = 0.0;
  if (nHe > 0.0) {
    double a11 = 1.0 + h * ne * (r[4] + r[1]), a12 = h * ne * r[1];
    double a21 = h * ne * r[5], a22 = 1.0 + h * ne * (r[2] + r[5]);
    double b1 = nj[1] - P[1] + h * ne * r[1] * nHe;
    double b2 = nHe * s->xHeIII + P[2] + h * ne * r[5] * nHe;
    double det = a11 * a22 - a12 * a21;
    double a = (b1 * a22 - a12 * b2) / det, cc = (a11 * b2 - a21 * b1) / det;
    if (a < 0.0) a = 0.0;
    if (a > nHe) a = nHe;
    if (cc < 0.0) cc = 0.0;
    if (cc > nHe - a) cc = nHe - a;
    nHeIn = a; nHeIIIn = cc; nHeIIn = nHe - a - cc;
    o->xHeII = nHeIIn / nHe; o->xHeIII = nHeIIIn / nHe;
  } else { o->xHeII = s->xHeII; o->xHeIII = s->xHeIII; }
  /* C6: thermal energy, explicit; rates at the old T, new abundances (S23) */
  double f = 0.0;
  if (thermal) {
    double xen = o->xHII + y * (o->xHeII + 2.0 * o->xHeIII);
    double nen = nH * xen;
    double nHIn = nH - nHIIn;
    double lam = nen * (r[6] * nHIIn + r[7] * nHeIIn + r[8] * nHeIIIn + r[9] * nHIn + r[10] * nHeIn + r[11] * nHeIIn +
                        r[12] * nHIn + r[13] * nHeIIn + r[14] * (nHIIn + nHeIIn + 4.0 * nHeIIIn));
    double en = s->e + heat - h * lam;
    double efloor = 1.5 * nH * (1.0 + y + xen) * K_BOLTZ * T_MIN;
    if (en < efloor) en = efloor;
    o->e = en;
    f = fabs(en - s->e) / s->e;
  } else o->e = s->e;
  /* C7: largest relative change of the five abundances (S18, S20) */
  double xo[5] = {1.0 - s->xHII, s->xHII, 1.0 - s->xHeII - s->xHeIII, s->xHeII, s->xHeIII};
  double xn[5] = {1.0 - o->xHII, o->xHII, 1.0 - o->xHeII - o->xHeIII, o->xHeII, o->xHeIII};
  int nk = nHe > 0.0 ? 5 : 2;
  for (int k = 0; k < nk; k++) {
    double den = xo[k] > c->x_floor_rel ? xo[k] : c->x_floor_rel;
    double fk = fabs(xn[k] - xo[k]) / den;
    if (fk > f) f = fk;
  }
  return f;
}

static int64_t chem_cell(const oracle_ctx *c, chem_state *s, double nH, double dt, int *hit_cap, double *trace,
                         int64_t ntrace_max, int64_t *ntrace) {
  /* C8: PAPER.md:238 — start with h = dt; reject if f > 0.1 and shrink by f_s/f; on accept
   * multiply by f_s/f but at most double. h is not carried between subcycles (S19). */
  double t = 0.0, h = dt;
  int64_t attempts = 0;
  int last = 1; /* h == dt - t */
  *hit_cap = 0;
  while (1) {
    if (attempts >= c->max_substeps) { *hit_cap = 1; break; }
    chem_state o;
    double f = chem_try(c, s, nH, h, &o);
    attempts++;
    int acc = f <= c->f_accept; /* accepted only if the change stays below 10 %; a NaN is not */
    if (trace && *ntrace < ntrace_max) {
      trace[3 * *ntrace] = h; trace[3 * *ntrace + 1] = f; trace[3 * *ntrace + 2] = acc; (*ntrace)++;
    }
    if (!acc) { h = h * c->f_target / f; last = 0; continue; }
    *s = o;
    if (last) break;
    t += h;
    double fm = f > 1e-300 ? f : 1e-300;
    double grow = c->f_target / fm;
    if (grow > 2.0) grow = 2.0;
    h = h * grow;
    if (h >= dt - t) { h = dt - t; last = 1; }
  }
  return attempts;
}

/* ------------------------------------------------------------------ construction */
static void *dup(const void *p, size_t n) { void *q = malloc(n ? n : 1); if (p && n) memcpy(q, p, n); return q; }

oracle_ctx *oracle_create(int64_t C, int64_t F, int G, const double *box, const int32_t *periodic, const double *volume,
                          const double *centroid, const double *area, const double *normal, const double *fcentroid,
                          const int32_t *left, const int32_t *right, int nghost, const double *ghost) {
  oracle_ctx *c = (oracle_ctx *)calloc(1, sizeof(oracle_ctx));
  c->C = C; c->F = F; c->G = G;
  for (int a = 0; a < 3; a++) { c->box[a] = box[a]; c->periodic[a] = periodic[a]; }
  c->volume = (double *)dup(volume, C * sizeof(double));
  c->centroid = (double *)dup(centroid, 3 * C * sizeof(double));
  c->area = (double *)dup(area, F * sizeof(double));
  c->normal = (double *)dup(normal, 3 * F * sizeof(double));
  c->fcentroid = (double *)dup(fcentroid, 3 * F * sizeof(double));
  c->left = (int32_t *)dup(left, F * sizeof(int32_t));
  c->right = (int32_t *)dup(right, F * sizeof(int32_t));
  c->nghost = nghost;
  c->ghost = (double *)dup(ghost, (size_t)nghost * 4 * G * sizeof(double));
  /* CSR cell -> half-faces (offset + count + interface index list) */
  c->off = (int64_t *)calloc(C + 1, sizeof(int64_t));
  for (int64_t f = 0; f < F; f++) { c->off[left[f] + 1]++; if (right[f] >= 0) c->off[right[f] + 1]++; }
  for (int64_t i = 0; i < C; i++) c->off[i + 1] += c->off[i];
  int64_t nhf = c->off[C];
  c->hf_face = (int32_t *)malloc(nhf * sizeof(int32_t) + 4);
  c->hf_side = (int8_t *)malloc(nhf + 1);
  int64_t *fill = (int64_t *)dup(c->off, C * sizeof(int64_t));
  for (int64_t f = 0; f < F; f++) {
    int64_t k = fill[left[f]]++; c->hf_face[k] = (int32_t)f; c->hf_side[k] = 1;
    if (right[f] >= 0) { k = fill[right[f]]++; c->hf_face[k] = (int32_t)f; c->hf_side[k] = -1; }
  }
  free(fill);
  /* O3 geometry, once per mesh (the matrix depends only on the mesh) */
  c->hf_w = (double *)malloc(nhf * 3 * sizeof(double) + 8);
  c->hf_r = (double *)malloc(nhf * 3 * sizeof(double) + 8);
  c->Minv = (double *)malloc(C * 9 * sizeof(double));
  for (int64_t i = 0; i < C; i++) {
    double M[9] = {0};
    for (int64_t k = c->off[i]; k < c->off[i + 1]; k++) {
      int64_t f = c->hf_face[k];
      int sd = c->hf_side[k];
      int64_t j = sd > 0 ? right[f] : left[f];
      double ri[3], d[3];
      for (int a = 0; a < 3; a++) ri[a] = minimg(fcentroid[a * F + f] - centroid[a * C + i], box[a], periodic[a]);
      if (j >= 0) {
        /* s_j - s_i measured through the face: (c_f - s_i) - (c_f - s_j), each min-imaged */
        for (int a = 0; a < 3; a++)
          d[a] = ri[a] - minimg(fcentroid[a * F + f] - centroid[a * C + j], box[a], periodic[a]);
      } else {
        /* boundary face: mirror point s_i + 2((c_f - s_i).n) n  (S13) */
        double nn[3] = {sd * normal[f], sd * normal[F + f], sd * normal[2 * F + f]};
        double p = ri[0] * nn[0] + ri[1] * nn[1] + ri[2] * nn[2];
        for (int a = 0; a < 3; a++) d[a] = 2.0 * p * nn[a];
      }
      double dl = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
      double nh[3] = {d[0] / dl, d[1] / dl, d[2] / dl};
      for (int a = 0; a < 3; a++) {
        c->hf_r[3 * k + a] = ri[a];
        c->hf_w[3 * k + a] = area[f] / dl * nh[a];
        for (int b = 0; b < 3; b++) M[3 * a + b] += area[f] * nh[a] * nh[b];
      }
    }
    if (inv3(M, c->Minv + 9 * i) != 0) memset(c->Minv + 9 * i, 0, 9 * sizeof(double));
  }
  /* defaults */
  c->ctilde = 1.0; c->f_accept = 0.1; c->f_target = 0.05; c->x_floor_rel = 1e-3; c->max_substeps = 1000000;
  c->order = 2; c->heun = 1; c->T_fixed = 1e4;
  c->N = (double *)calloc((size_t)G * C, sizeof(double));
  c->Fl = (double *)calloc((size_t)G * 3 * C, sizeof(double));
  c->N0 = (double *)calloc((size_t)G * C, sizeof(double));
  c->Fl0 = (double *)calloc((size_t)G * 3 * C, sizeof(double));
  c->xHII = (double *)calloc(C, sizeof(double)); c->xHeII = (double *)calloc(C, sizeof(double));
  c->xHeIII = (double *)calloc(C, sizeof(double)); c->eth = (double *)calloc(C, sizeof(double));
  c->nH = (double *)calloc(C, sizeof(double));
  c->gN = (double *)calloc((size_t)G * 3 * C, sizeof(double));
  c->gF = (double *)calloc((size_t)G * 9 * C, sizeof(double));
  c->phi = (double *)calloc((size_t)F * G * 4, sizeof(double));
  c->kappa = (double *)calloc(C, sizeof(double));
  return c;
}

void oracle_destroy(oracle_ctx *c) {
  if (!c) return;
  free((void *)c->volume); free((void *)c->centroid); free((void *)c->area); free((void *)c->normal);
  free((void *)c->fcentroid); free((void *)c->left); free((void *)c->right); free(c->ghost); free(c->off);
  free(c->hf_face); free(c->hf_side); free(c->hf_w); free(c->hf_r); free(c->Minv); free(c->kappa);
  free(c->gNf); free(c->gFf); free(c->active); free(c->touched); free(c->src_cell); free(c->src_rate); free(c->N); free(c->Fl); free(c->N0); free(c->Fl0); free(c->xHII);
  free(c->xHeII); free(c->xHeIII); free(c->eth); free(c->nH); free(c->gN); free(c->gF); free(c->phi);
  free(c);
}

void oracle_set_params(oracle_ctx *c, double ctilde, const double *sigma, const double *eps, int chem_mode,
                       const double *kappa, double T_fixed, double alphaB_override, double y_he, double f_accept,
                       double f_target, double x_floor_rel, double n_floor, int64_t max_substeps, int order, int heun) {
  c->ctilde = ctilde;
  for (int k = 0; k < 3 * c->G; k++) { c->sigma[k] = sigma ? sigma[k] : 0.0; c->eps[k] = eps ? eps[k] : 0.0; }
  c->chem_mode = chem_mode;
  if (kappa) memcpy(c->kappa, kappa, c->C * sizeof(double));
  c->T_fixed = T_fixed; c->alphaB_override = alphaB_override; c->y_he = y_he; c->f_accept = f_accept;
  c->f_target = f_target; c->x_floor_rel = x_floor_rel; c->n_floor = n_floor; c->max_substeps = max_substeps;
  c->order = order; c->heun = heun;
}

/* Individual time steps ("fluxes for interfaces with at least one active neighbour. For passive
 * particles, only their conserved quantities are updated, taking into account the fluxes from the interfaces
 * they share with active cells"; cells and interfaces in active / passive categories that
 * stay fixed during the subcycles of one RT step).  Reading S27: a passive cell does no chemistry, injects
 * no source photons, has no gradient (its mesh is not constructed: its face state is its cell value), and
 * faces between two passive cells carry no flux.  active: (C) bytes, or NULL for "all active". */
void oracle_set_active(oracle_ctx *c, const uint8_t *active) {
  free(c->active); free(c->touched);
  c->active = active ? (uint8_t *)dup(active, (size_t)c->C) : NULL;
  c->touched = NULL;
  if (!active) return;
  c->touched = (uint8_t *)dup(active, (size_t)c->C);
  for (int64_t f = 0; f < c->F; f++) {
    int64_t L = c->left[f], R = c->right[f];
    if (R < 0) continue;
    if (active[L]) c->touched[R] = 1;
    if (active[R]) c->touched[L] = 1;
  }
}
static int is_active(const oracle_ctx *c, int64_t i) { return !c->active || c->active[i]; }
/* a cell none of whose interfaces has an active cell is left alone altogether: "passive" */
static int is_touched(const oracle_ctx *c, int64_t i) { return !c->touched || c->touched[i]; }

/* Mixed precision ("primitive variables could be converted to single precision, conserved
 * quantities and flux summations should remain in double precision", "special care ... to avoid numerical
 * overflows ... a suitable unit system").  Reading S28: the state U, the face-flux sums, the update, the cap and
 * the ledgers stay fp64; the gradient estimate, the slope limiter, the states reconstructed at the face centres,
 * the M1 closure and the Riemann flux are evaluated in fp32, in units that keep every number O(1):
 * lengths in units of the cell size l_i ~ V_i^(1/3) (the stored gradient is l_i grad phi, a float), face
 * states in units of s ~ max(|N_L|, |N_R|) for N and c~ s for F; l_i and s are rounded to powers of two, so that
 * the choice of unit changes no rounding at all (only c~ is not a power of two).  Differences phi_j - phi_i are formed in
 * fp64 and then rounded, so a small contrast on a large background survives. */
void oracle_set_precision(oracle_ctx *c, int mixed) {
  c->mixed = mixed;
  if (mixed && !c->gNf) {
    c->gNf = (float *)calloc((size_t)c->G * 3 * c->C, sizeof(float));
    c->gFf = (float *)calloc((size_t)c->G * 9 * c->C, sizeof(float));
  }
}

void oracle_set_sources(oracle_ctx *c, int nsrc, const int32_t *cell, const double *rate) {
  free(c->src_cell); free(c->src_rate);
  c->nsrc = nsrc;
  c->src_cell = (int32_t *)dup(cell, (size_t)nsrc * sizeof(int32_t));
  c->src_rate = (double *)dup(rate, (size_t)nsrc * c->G * sizeof(double));
}

static void ledger_reset(oracle_ctx *c) {
  memset(c->led, 0, sizeof(c->led));
  c->substeps_total = c->substeps_max = c->cells_hit_cap = 0;
  for (int g = 0; g < c->G; g++)
    for (int64_t i = 0; i < c->C; i++) kadd(&c->led[g][L_STORED], c->volume[i] * c->N[(size_t)g * c->C + i]);
}

void oracle_set_state(oracle_ctx *c, const double *N, const double *Fl, const double *xHII, const double *xHeII,
                      const double *xHeIII, const double *eth, const double *nH) {
  size_t C = c->C, G = c->G;
  memcpy(c->N, N, G * C * 8); memcpy(c->Fl, Fl, G * 3 * C * 8);
  memcpy(c->xHII, xHII, C * 8); memcpy(c->xHeII, xHeII, C * 8); memcpy(c->xHeIII, xHeIII, C * 8);
  memcpy(c->eth, eth, C * 8); memcpy(c->nH, nH, C * 8);
  ledger_reset(c);
}

void oracle_get_state(const oracle_ctx *c, double *N, double *Fl, double *xHII, double *xHeII, double *xHeIII,
                      double *eth) {
  size_t C = c->C, G = c->G;
  memcpy(N, c->N, G * C * 8); memcpy(Fl, c->Fl, G * 3 * C * 8);
  memcpy(xHII, c->xHII, C * 8); memcpy(xHeII, c->xHeII, C * 8); memcpy(xHeIII, c->xHeIII, C * 8);
  memcpy(eth, c->eth, C * 8);
}

/* ledger[G][6] = stored, injected, absorbed, outflow, inflow_bc, floor_added; counters[3] */
void oracle_get_ledger(oracle_ctx *c, double *ledger, int64_t *counters) {
  for (int g = 0; g < c->G; g++) {
    ksum st = {0, 0};
    for (int64_t i = 0; i < c->C; i++) kadd(&st, c->volume[i] * c->N[(size_t)g * c->C + i]);
    c->led[g][L_STORED] = st;
    for (int r = 0; r < L_NROW; r++) ledger[g * L_NROW + r] = kval(&c->led[g][r]);
  }
  counters[0] = c->substeps_total; counters[1] = c->substeps_max; counters[2] = c->cells_hit_cap;
}

/* ------------------------------------------------------------------ O1 over all cells */
static void chemistry(oracle_ctx *c, double dt) {
  const int64_t C = c->C;
  const int G = c->G;
  if (c->chem_mode == CHEM_NONE) return;
  for (int64_t i = 0; i < C; i++) {
    if (!is_active(c, i)) continue; /* S27 */
    if (c->chem_mode == CHEM_FIXED_OPACITY) {
      /* one implicit step N' = N/(1 + dt c kappa): eq (6)-(7) right-hand sides */
      double den = 1.0 + dt * c->ctilde * c->kappa[i];
      for (int g = 0; g < G; g++) {
        double Nb = c->N[(size_t)g * C + i];
        c->N[(size_t)g * C + i] = Nb / den;
        for (int a = 0; a < 3; a++) c->Fl[((size_t)g * 3 + a) * C + i] /= den;
        kadd(&c->led[g][L_ABSORBED], c->volume[i] * (Nb - c->N[(size_t)g * C + i]));
      }
      continue;
    }
    chem_state s;
    for (int g = 0; g < G; g++) {
      s.N[g] = c->N[(size_t)g * C + i];
      for (int a = 0; a < 3; a++) s.F[3 * g + a] = c->Fl[((size_t)g * 3 + a) * C + i];
    }
    s.xHII = c->xHII[i]; s.xHeII = c->xHeII[i]; s.xHeIII = c->xHeIII[i]; s.e = c->eth[i];
    double Nb[8];
    for (int g = 0; g < G; g++) Nb[g] = s.N[g];
    int cap;
    int64_t nt = 0;
    int64_t att = chem_cell(c, &s, c->nH[i], dt, &cap, 0, 0, &nt);
    c->substeps_total += att;
    if (att > c->substeps_max) c->substeps_max = att;
    c->cells_hit_cap += cap;
    for (int g = 0; g < G; g++) {
      c->N[(size_t)g * C + i] = s.N[g];
      for (int a = 0; a < 3; a++) c->Fl[((size_t)g * 3 + a) * C + i] = s.F[3 * g + a];
      kadd(&c->led[g][L_ABSORBED], c->volume[i] * (Nb[g] - s.N[g])); /* C9 */
    }
    c->xHII[i] = s.xHII; c->xHeII[i] = s.xHeII; c->xHeIII[i] = s.xHeIII; c->eth[i] = s.e;
  }
}

/* value of field q (0: N, 1..3: F) of group g in cell i */
static double fld(const oracle_ctx *c, int g, int q, int64_t i) {
  return q == 0 ? c->N[(size_t)g * c->C + i] : c->Fl[((size_t)g * 3 + (q - 1)) * c->C + i];
}

/* neighbour (or ghost) state seen by cell i across half-face k, all four fields (S13) */
static void nbr_state(const oracle_ctx *c, int g, int64_t i, int64_t k, double U[4]) {
  int64_t f = c->hf_face[k];
  int sd = c->hf_side[k];
  int64_t j = sd > 0 ? c->right[f] : c->left[f];
  if (j >= 0) { for (int q = 0; q < 4; q++) U[q] = fld(c, g, q, j); return; }
  for (int q = 0; q < 4; q++) U[q] = fld(c, g, q, i);
  if (j == BC_OUTFLOW) return; /* copy ghost */
  if (j == BC_REFLECT) {
    double n[3] = {c->normal[f], c->normal[c->F + f], c->normal[2 * c->F + f]};
    double p = U[1] * n[0] + U[2] * n[1] + U[3] * n[2];
    for (int a = 0; a < 3; a++) U[1 + a] -= 2.0 * p * n[a];
    return;
  }
  int kg = BC_DIRICHLET0 - (int)j;
  for (int q = 0; q < 4; q++) U[q] = c->ghost[(size_t)kg * 4 * c->G + 4 * g + q];
}

/* ------------------------------------------------------------------ O3: gradients + limiter */
static void gradients(oracle_ctx *c) {
  const int64_t C = c->C;
  const int G = c->G;
  for (int64_t i = 0; i < C; i++)
    for (int g = 0; g < G; g++)
      for (int q = 0; q < 4; q++) {
        double *out[3];
        for (int a = 0; a < 3; a++)
          out[a] = q == 0 ? &c->gN[((size_t)g * 3 + a) * C + i] : &c->gF[(((size_t)g * 3 + (q - 1)) * 3 + a) * C + i];
        if (c->order < 2 || !is_active(c, i)) { *out[0] = *out[1] = *out[2] = 0.0; continue; } /* passive: S27 */
        double pi = fld(c, g, q, i);
        double b[3] = {0, 0, 0}, pmax = pi, pmin = pi;
        /* first neighbour loop: second term of eq (15) and min/max */
        for (int64_t k = c->off[i]; k < c->off[i + 1]; k++) {
          double U[4];
          nbr_state(c, g, i, k, U);
          double pj = U[q];
          for (int a = 0; a < 3; a++) b[a] += c->hf_w[3 * k + a] * (pj - pi);
          if (pj > pmax) pmax = pj;
          if (pj < pmin) pmin = pj;
        }
        const double *Mi = c->Minv + 9 * i;
        double gr[3];
        for (int a = 0; a < 3; a++) gr[a] = Mi[3 * a] * b[0] + Mi[3 * a + 1] * b[1] + Mi[3 * a + 2] * b[2];
        /* second neighbour loop: limit so the face-centre values create no new extremum (S8-S10) */
        double alpha = 1.0;
        for (int64_t k = c->off[i]; k < c->off[i + 1]; k++) {
          double d = gr[0] * c->hf_r[3 * k] + gr[1] * c->hf_r[3 * k + 1] + gr[2] * c->hf_r[3 * k + 2];
          double psi = 1.0;
          if (d > 0.0) psi = (pmax - pi) / d;
          else if (d < 0.0) psi = (pmin - pi) / d;
          if (psi < alpha) alpha = psi;
        }
        for (int a = 0; a < 3; a++) *out[a] = alpha * gr[a];
      }
}

void oracle_gradients(oracle_ctx *c, double *gN, double *gF) {
  gradients(c);
  memcpy(gN, c->gN, (size_t)c->G * 3 * c->C * 8);
  memcpy(gF, c->gF, (size_t)c->G * 9 * c->C * 8);
}

/* ------------------------------------------------------------------ O4 over all faces */
static void extrapolate(const oracle_ctx *c, int g, int64_t i, int64_t f, double U[4]) {
  const int64_t C = c->C, F = c->F;
  double r[3];
  for (int a = 0; a < 3; a++) r[a] = minimg(c->fcentroid[a * F + f] - c->centroid[a * C + i], c->box[a], c->periodic[a]);
  U[0] = c->N[(size_t)g * C + i];
  for (int a = 0; a < 3; a++) U[0] += c->gN[((size_t)g * 3 + a) * C + i] * r[a];
  for (int q = 0; q < 3; q++) {
    U[1 + q] = c->Fl[((size_t)g * 3 + q) * C + i];
    for (int a = 0; a < 3; a++) U[1 + q] += c->gF[(((size_t)g * 3 + q) * 3 + a) * C + i] * r[a];
  }
}

static void fluxes(oracle_ctx *c, double dt) {
  const int64_t F = c->F;
  const int G = c->G;
  for (int64_t f = 0; f < F; f++) {
    int64_t L = c->left[f], R = c->right[f];
    double n[3] = {c->normal[f], c->normal[F + f], c->normal[2 * F + f]};
    /* only interfaces with at least one active cell carry a flux */
    if (!(is_active(c, L) || (R >= 0 && is_active(c, R)))) {
      for (int k = 0; k < 4 * G; k++) c->phi[(size_t)f * G * 4 + k] = 0.0;
      continue;
    }
    for (int g = 0; g < G; g++) {
      double UL[4], UR[4];
      extrapolate(c, g, L, f, UL);
      if (R >= 0) extrapolate(c, g, R, f, UR);
      else if (R == BC_OUTFLOW) { UR[0] = UR[1] = UR[2] = UR[3] = 0.0; } /* vacuum ghost (S13) */
      else if (R == BC_REFLECT) {
        double p = UL[1] * n[0] + UL[2] * n[1] + UL[3] * n[2];
        UR[0] = UL[0];
        for (int a = 0; a < 3; a++) UR[1 + a] = UL[1 + a] - 2.0 * p * n[a];
      } else {
        int kg = BC_DIRICHLET0 - (int)R;
        for (int q = 0; q < 4; q++) UR[q] = c->ghost[(size_t)kg * 4 * G + 4 * g + q];
      }
      double ph[4];
      oracle_riemann(UL, UR, n, c->ctilde, ph);
      /* "a further limiter is applied to prevent negative photon densities" PAPER.md:155 (S11):
       * the donor cell cannot lose more photons than it holds through this face in dt, so the
       * magnitude of the number flux is clamped; the momentum flux Phi_F is left alone (scaling
       * it by the same factor is discontinuous where Phi_N changes sign next to an empty cell:
       * tests/test_oracle_conditioning.py) */
      int64_t d = ph[0] > 0.0 ? L : (ph[0] < 0.0 ? R : -1);
      if (d >= 0) {
        double lim = c->N[(size_t)g * c->C + d] * c->volume[d] / (dt * c->area[f]);
        if (fabs(ph[0]) > lim) ph[0] = ph[0] > 0.0 ? lim : -lim;
      }
      for (int q = 0; q < 4; q++) c->phi[((size_t)f * G + g) * 4 + q] = ph[q];
    }
  }
}

/* ------------------------------------------------------------------ O3 + O4 in mixed precision (S28) */
/* the units are powers of two: changing units then changes no rounding, it only keeps the exponents in range */
static double unit_length(double V) { int e; frexp(cbrt(V), &e); return ldexp(1.0, e); }            /* l <= 2 V^(1/3) */
static float unit_density(float m) {                                                                 /* s <= 2 m */
  int e;
  if (!(m >= 1e-30f)) m = 1e-30f;
  frexpf(m, &e);
  if (e > 126) e = 126;
  return ldexpf(1.0f, e);
}
static void gradients_mixed(oracle_ctx *c) {
  const int64_t C = c->C;
  const int G = c->G;
  for (int64_t i = 0; i < C; i++) {
    const double l = unit_length(c->volume[i]);
    float Mi[9];
    for (int a = 0; a < 9; a++) Mi[a] = (float)(c->Minv[9 * i + a] * l * l);
    for (int g = 0; g < G; g++)
      for (int q = 0; q < 4; q++) {
        float *out[3];
        for (int a = 0; a < 3; a++)
          out[a] = q == 0 ? &c->gNf[((size_t)g * 3 + a) * C + i] : &c->gFf[(((size_t)g * 3 + (q - 1)) * 3 + a) * C + i];
        if (c->order < 2 || !is_active(c, i)) { *out[0] = *out[1] = *out[2] = 0.0f; continue; }
        const double pi = fld(c, g, q, i);
        /* b = sum w (phi_j - phi_i) and the extreme differences (S8: phi_i itself counts, so hi >= 0 >= lo) */
        float b[3] = {0, 0, 0}, hid = 0.0f, lod = 0.0f;
        for (int64_t k = c->off[i]; k < c->off[i + 1]; k++) {
          double U[4];
          nbr_state(c, g, i, k, U);
          const float d = (float)(U[q] - pi);
          for (int a = 0; a < 3; a++) {
            const float w = (float)(c->hf_w[3 * k + a] / l);
            b[a] = b[a] + w * d;
          }
          if (d > hid) hid = d;
          if (d < lod) lod = d;
        }
        float gr[3];
        for (int a = 0; a < 3; a++) gr[a] = Mi[3 * a] * b[0] + Mi[3 * a + 1] * b[1] + Mi[3 * a + 2] * b[2];
        float alpha = 1.0f;
        for (int64_t k = c->off[i]; k < c->off[i + 1]; k++) {
          const float rx = (float)(c->hf_r[3 * k] / l), ry = (float)(c->hf_r[3 * k + 1] / l), rz = (float)(c->hf_r[3 * k + 2] / l);
          const float d = gr[0] * rx + gr[1] * ry + gr[2] * rz;
          float psi = 1.0f;
          if (d > 0.0f) psi = hid / d;
          else if (d < 0.0f) psi = lod / d;
          if (psi < alpha) alpha = psi;
        }
        for (int a = 0; a < 3; a++) *out[a] = alpha * gr[a];
      }
  }
}

/* cell value (double) and single-precision increment to the centre of face f, fields (N, Fx, Fy, Fz) of
 * group g in cell i: the face state is (float)cell + inc */
static void extrapolate_mixed(const oracle_ctx *c, int g, int64_t i, int64_t f, double cell[4], float inc[4]) {
  const int64_t C = c->C, F = c->F;
  const double l = unit_length(c->volume[i]);
  float r[3];
  for (int a = 0; a < 3; a++)
    r[a] = (float)(minimg(c->fcentroid[a * F + f] - c->centroid[a * C + i], c->box[a], c->periodic[a]) / l);
  cell[0] = c->N[(size_t)g * C + i];
  inc[0] = c->gNf[((size_t)g * 3) * C + i] * r[0] + c->gNf[((size_t)g * 3 + 1) * C + i] * r[1] + c->gNf[((size_t)g * 3 + 2) * C + i] * r[2];
  for (int q = 0; q < 3; q++) {
    cell[1 + q] = c->Fl[((size_t)g * 3 + q) * C + i];
    const float *gq = c->gFf + ((size_t)g * 3 + q) * 3 * C + i;
    inc[1 + q] = gq[0] * r[0] + gq[C] * r[1] + gq[2 * C] * r[2];
  }
}

/* n D.nf of the M1 closure (S1) for the normalised state (n, f), lab frame, single precision */
static void pressure_mixed(float n, const float f[3], const float nf[3], float out[3]) {
  const float f2 = f[0] * f[0] + f[1] * f[1] + f[2] * f[2];
  float den = n * n;
  if (den < 1e-30f) den = 1e-30f;
  float x2 = f2 / den; /* (|F| / (c~ N))^2 */
  if (x2 > 1.0f) x2 = 1.0f;
  const float chi = (3.0f + 4.0f * x2) / (5.0f + 2.0f * sqrtf(4.0f - 3.0f * x2));
  const float a = 0.5f * (1.0f - chi) * n;
  for (int k = 0; k < 3; k++) out[k] = a * nf[k];
  if (f2 > 0.0f) {
    const float bb = 0.5f * (3.0f * chi - 1.0f) * n * (f[0] * nf[0] + f[1] * nf[1] + f[2] * nf[2]) / f2;
    for (int k = 0; k < 3; k++) out[k] = out[k] + bb * f[k];
  }
}

static void fluxes_mixed(oracle_ctx *c, double dt) {
  const int64_t F = c->F;
  const int G = c->G;
  const float ctf = (float)c->ctilde;
  for (int64_t f = 0; f < F; f++) {
    const int64_t L = c->left[f], R = c->right[f];
    const float nf[3] = {(float)c->normal[f], (float)c->normal[F + f], (float)c->normal[2 * F + f]};
    if (!(is_active(c, L) || (R >= 0 && is_active(c, R)))) {
      for (int k = 0; k < 4 * G; k++) c->phi[(size_t)f * G * 4 + k] = 0.0;
      continue;
    }
    for (int g = 0; g < G; g++) {
      /* face states UL, UR for the mean and the closure; the jump J = UR - UL takes the cell-value part
       * in double before rounding, like the differences of the gradient estimate */
      double cL[4], cR[4];
      float iL[4], iR[4], UL[4], UR[4], J[4];
      extrapolate_mixed(c, g, L, f, cL, iL);
      for (int q = 0; q < 4; q++) UL[q] = (float)cL[q] + iL[q];
      if (R >= 0) {
        extrapolate_mixed(c, g, R, f, cR, iR);
        for (int q = 0; q < 4; q++) { UR[q] = (float)cR[q] + iR[q]; J[q] = (float)(cR[q] - cL[q]) + (iR[q] - iL[q]); }
      } else if (R == BC_OUTFLOW) {
        for (int q = 0; q < 4; q++) { UR[q] = 0.0f; J[q] = -UL[q]; }
      } else if (R == BC_REFLECT) {
        const float p = UL[1] * nf[0] + UL[2] * nf[1] + UL[3] * nf[2];
        UR[0] = UL[0]; J[0] = 0.0f;
        for (int a = 0; a < 3; a++) { J[1 + a] = -2.0f * p * nf[a]; UR[1 + a] = UL[1 + a] + J[1 + a]; }
      } else {
        const int kg = BC_DIRICHLET0 - (int)R;
        for (int q = 0; q < 4; q++) {
          cR[q] = c->ghost[(size_t)kg * 4 * G + 4 * g + q];
          UR[q] = (float)cR[q];
          J[q] = (float)(cR[q] - cL[q]) - iL[q];
        }
      }
      /* units: s for N, c~ s for F, so that every number below is O(1) */
      const float sc = unit_density(fabsf(UL[0]) > fabsf(UR[0]) ? fabsf(UL[0]) : fabsf(UR[0]));
      const float is = 1.0f / sc, ict = 1.0f / ctf;
      const float nL = UL[0] * is, nR = UR[0] * is;
      const float fL[3] = {UL[1] * is * ict, UL[2] * is * ict, UL[3] * is * ict}, fR[3] = {UR[1] * is * ict, UR[2] * is * ict, UR[3] * is * ict};
      float PL[3], PR[3];
      pressure_mixed(nL, fL, nf, PL);
      pressure_mixed(nR, fR, nf, PR);
      const float pn = 0.5f * ((fL[0] + fR[0]) * nf[0] + (fL[1] + fR[1]) * nf[1] + (fL[2] + fR[2]) * nf[2]) - 0.5f * (J[0] * is);
      double ph[4];
      ph[0] = (double)pn * c->ctilde * (double)sc;
      for (int a = 0; a < 3; a++)
        ph[1 + a] = (double)(0.5f * (PL[a] + PR[a]) - 0.5f * (J[1 + a] * is * ict)) * c->ctilde * c->ctilde * (double)sc;
      /* donor cap (S11): in double, on the cell's own N */
      const int64_t d = ph[0] > 0.0 ? L : (ph[0] < 0.0 ? R : -1);
      if (d >= 0) {
        const double lim = c->N[(size_t)g * c->C + d] * c->volume[d] / (dt * c->area[f]);
        if (fabs(ph[0]) > lim) ph[0] = ph[0] > 0.0 ? lim : -lim;
      }
      for (int q = 0; q < 4; q++) c->phi[((size_t)f * G + g) * 4 + q] = ph[q];
    }
  }
}

/* ------------------------------------------------------------------ O5 + O2: apply, enforce, Heun */
static void enforce(oracle_ctx *c, int g, int64_t i, double wfloor) {
  const int64_t C = c->C;
  double *N = &c->N[(size_t)g * C + i];
  if (*N < c->n_floor) { kadd(&c->led[g][L_FLOOR], wfloor * c->volume[i] * (c->n_floor - *N)); *N = c->n_floor; }
  double *fx = &c->Fl[((size_t)g * 3 + 0) * C + i], *fy = &c->Fl[((size_t)g * 3 + 1) * C + i],
         *fz = &c->Fl[((size_t)g * 3 + 2) * C + i];
  double fn = sqrt(*fx * *fx + *fy * *fy + *fz * *fz), lim = c->ctilde * *N;
  if (fn > lim) { double s = lim / fn; *fx *= s; *fy *= s; *fz *= s; } /* |F| <= c N (S12) */
}

/* U <- a*U0 + b*(U + dt R(U)), ledger increments weighted by wl */
static void stage(oracle_ctx *c, double dt, double a, double b, double wl, double wfloor) {
  const int64_t C = c->C, F = c->F;
  const int G = c->G;
  if (c->mixed) { gradients_mixed(c); fluxes_mixed(c, dt); }
  else {
    if (c->order >= 2) gradients(c);
    else { memset(c->gN, 0, (size_t)G * 3 * C * 8); memset(c->gF, 0, (size_t)G * 9 * C * 8); }
    fluxes(c, dt);
  }
  /* boundary ledgers */
  for (int64_t f = 0; f < F; f++) {
    int64_t R = c->right[f];
    if (R >= 0 || R == BC_REFLECT) continue;
    for (int g = 0; g < G; g++) {
      double x = wl * dt * c->area[f] * c->phi[((size_t)f * G + g) * 4];
      if (R == BC_OUTFLOW) kadd(&c->led[g][L_OUTFLOW], x); else kadd(&c->led[g][L_INFLOW_BC], -x);
    }
  }
  /* sources enter the transport right-hand side, isotropically (S5) */
  double *srcN = (double *)calloc((size_t)G * C, sizeof(double));
  for (int s = 0; s < c->nsrc; s++)
    for (int g = 0; g < G; g++) {
      if (!is_active(c, c->src_cell[s])) continue; /* a passive cell injects nothing during this RT step (S27) */
      srcN[(size_t)g * C + c->src_cell[s]] += c->src_rate[(size_t)g * c->nsrc + s];
      kadd(&c->led[g][L_INJECTED], wl * dt * c->src_rate[(size_t)g * c->nsrc + s]);
    }
  for (int64_t i = 0; i < C; i++)
    for (int g = 0; g < G; g++) {
      if (!is_touched(c, i)) continue;
      double sum[4] = {0, 0, 0, 0};
      for (int64_t k = c->off[i]; k < c->off[i + 1]; k++) {
        int64_t f = c->hf_face[k];
        for (int q = 0; q < 4; q++) sum[q] += c->hf_side[k] * c->area[f] * c->phi[((size_t)f * G + g) * 4 + q];
      }
      double Rr[4];
      for (int q = 0; q < 4; q++) Rr[q] = -sum[q] / c->volume[i];
      Rr[0] += srcN[(size_t)g * C + i] / c->volume[i];
      double *N = &c->N[(size_t)g * C + i];
      *N = a * c->N0[(size_t)g * C + i] + b * (*N + dt * Rr[0]);
      for (int q = 0; q < 3; q++) {
        double *Fq = &c->Fl[((size_t)g * 3 + q) * C + i];
        *Fq = a * c->Fl0[((size_t)g * 3 + q) * C + i] + b * (*Fq + dt * Rr[1 + q]);
      }
    }
  free(srcN);
  for (int64_t i = 0; i < C; i++)
    for (int g = 0; g < G; g++)
      if (is_touched(c, i)) enforce(c, g, i, wfloor);
}

static void transport(oracle_ctx *c, double dt) {
  const size_t C = c->C, G = c->G;
  memcpy(c->N0, c->N, G * C * 8);
  memcpy(c->Fl0, c->Fl, G * 3 * C * 8);
  if (c->heun) {
    stage(c, dt, 0.0, 1.0, 0.5, 0.5); /* U1 = enforce(Un + dt R(Un)) */
    stage(c, dt, 0.5, 0.5, 0.5, 1.0); /* Un+1 = enforce(Un/2 + (U1 + dt R(U1))/2) */
  } else stage(c, dt, 0.0, 1.0, 1.0, 1.0);
}

void oracle_step(oracle_ctx *c, double dt, int nsub) {
  for (int s = 0; s < nsub; s++) {
    chemistry(c, dt); /* Fig. 1 order (S4): chemistry(dt), then transport(dt) */
    transport(c, dt);
  }
}

/* single pieces, for the pins */
void oracle_transport_only(oracle_ctx *c, double dt) { transport(c, dt); }
void oracle_chemistry_only(oracle_ctx *c, double dt) { chemistry(c, dt); }

/* chemistry of one cell with a trace of (h, f, accepted); state arrays as in chem_state.
 * x[4] = xHII, xHeII, xHeIII, eth (in/out). Returns attempts. */
int64_t oracle_chem_cell(oracle_ctx *c, double *N, double *Fv, double *x, double nH, double dt, double *trace,
                         int64_t ntrace_max, int64_t *ntrace, int *hit_cap) {
  chem_state s;
  for (int g = 0; g < c->G; g++) { s.N[g] = N[g]; for (int a = 0; a < 3; a++) s.F[3 * g + a] = Fv[3 * g + a]; }
  s.xHII = x[0]; s.xHeII = x[1]; s.xHeIII = x[2]; s.e = x[3];
  *ntrace = 0;
  int64_t att = chem_cell(c, &s, nH, dt, hit_cap, trace, ntrace_max, ntrace);
  for (int g = 0; g < c->G; g++) { N[g] = s.N[g]; for (int a = 0; a < 3; a++) Fv[3 * g + a] = s.F[3 * g + a]; }
  x[0] = s.xHII; x[1] = s.xHeII; x[2] = s.xHeIII; x[3] = s.e;
  return att;
}

/* geometry accessors for the pins: hf_w/hf_r in CSR order, Minv */
int64_t oracle_nhalf(const oracle_ctx *c) { return c->off[c->C]; }
void oracle_get_geometry(const oracle_ctx *c, int64_t *off, int32_t *hf_face, double *hf_w, double *hf_r, double *Minv) {
  memcpy(off, c->off, (c->C + 1) * sizeof(int64_t));
  memcpy(hf_face, c->hf_face, c->off[c->C] * sizeof(int32_t));
  memcpy(hf_w, c->hf_w, c->off[c->C] * 3 * 8);
  memcpy(hf_r, c->hf_r, c->off[c->C] * 3 * 8);
  memcpy(Minv, c->Minv, c->C * 9 * 8);
}
