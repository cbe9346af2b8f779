"""The five synthetic workloads of BASELINE.json (`configs[0..4]`), recipe in SURVEY.md §8(d)
and DESIGN.md §4, plus config 5, the expanding H II region of PAPER.md:175-180, 290.  Input generators only: they produce the arrays handed to BOTH the oracle
and the CUDA path (`rt_mesh`, `rt_state`, `rt_sources`, `rt_params`, dt).  CGS units.

Configs 3/4 stand in for the paper's cosmological boxes (Table 1), whose
initial conditions are not available; config 0 has the geometry of a Stroemgren-sphere test.
Every config takes `n` so that tests can run the same recipe on a smaller lattice.
"""
from dataclasses import dataclass, field

import numpy as np

from . import mesh as M
from . import rng

C_LIGHT = 2.99792458e10
KPC = 3.0856775814913673e21
MYR = 3.15576e13
K_B = 1.380649e-16
EV = 1.602176634e-12

CHEM_NONE, CHEM_FIXED_OPACITY, CHEM_H_ISOTHERMAL, CHEM_HHE_THERMAL = 0, 1, 2, 3

# Grey cross-sections [cm^2] and heating energies [erg] per group (rows) and absorber
# (HI, HeI, HeII) for a 1e5 K black body, groups 13.6-24.6 / 24.6-54.4 / 54.4-inf eV
# (a stated simplification that defines the synthetic workload).
SIGMA3 = np.array([[2.8018e-18, 0.0, 0.0],
                   [4.7461e-19, 4.1567e-18, 0.0],
                   [6.3140e-20, 1.1071e-18, 1.0102e-18]])
EPS3 = np.array([[3.726, 0.0, 0.0],
                 [17.393, 7.546, 0.0],
                 [48.449, 38.414, 7.649]]) * EV
SHARE3 = np.array([0.44743, 0.49402, 0.05855])
Y_HE = 0.24 / (4.0 * 0.76)

SEED_MESH, SEED_RHO, SEED_SRC = 2404176300, 2404176310, 2404176320


@dataclass
class Params:
    ngroup: int = 1
    ctilde: float = 1.0
    sigma: np.ndarray = None        # (G,3)
    eps_heat: np.ndarray = None     # (G,3) erg
    chem_mode: int = CHEM_NONE
    T_fixed: float = 1.0e4
    alphaB_override: float = 0.0    # >0: replaces alpha_B,HII
    y_he: float = 0.0
    f_accept: float = 0.1
    f_target: float = 0.05
    x_floor_rel: float = 1.0e-3
    n_floor: float = 0.0
    max_substeps: int = 1000000
    order: int = 2
    heun: int = 1
    mixed: int = 0                  # 1: single-precision primitives, double-precision sums
    kappa: np.ndarray = None        # (C,) FIXED_OPACITY only [1/length]
    ghost_state: np.ndarray = None  # (K, 4G) Dirichlet ghost states (N, Fx, Fy, Fz per group)

    def __post_init__(self):
        if self.sigma is None:
            self.sigma = np.zeros((self.ngroup, 3))
        if self.eps_heat is None:
            self.eps_heat = np.zeros((self.ngroup, 3))


@dataclass
class State:
    N: np.ndarray       # (G, C)
    F: np.ndarray       # (G, 3, C)
    xHII: np.ndarray    # (C,)
    xHeII: np.ndarray
    xHeIII: np.ndarray
    eth: np.ndarray     # erg cm^-3
    nH: np.ndarray      # cm^-3

    def copy(self):
        return State(*(getattr(self, k).copy() for k in ("N", "F", "xHII", "xHeII", "xHeIII", "eth", "nH")))


@dataclass
class Sources:
    cell: np.ndarray    # (nsrc,) int32
    rate: np.ndarray    # (G, nsrc) photons/s


@dataclass
class Workload:
    name: str
    mesh: M.Mesh
    params: Params
    state: State
    sources: Sources
    dt: float
    meta: dict = field(default_factory=dict)


def eth_from_T(T, nH, xHII, xHeII, xHeIII, y):
    xe = xHII + y * (xHeII + 2.0 * xHeIII)
    return 1.5 * nH * (1.0 + y + xe) * K_B * T


def cfl_dt(mesh, ctilde, eta=0.3):
    """eq (11) PAPER.md:117 with v_c = 0, eta = 0.3; effective width 6V/sum(A) (S14)."""
    sa = np.bincount(mesh.left, weights=mesh.area, minlength=mesh.ncell)
    ok = mesh.right >= 0
    sa += np.bincount(mesh.right[ok], weights=mesh.area[ok], minlength=mesh.ncell)
    return float(eta * np.min(6.0 * mesh.volume / sa) / ctilde)


def _uniform_state(G, C, N0, nH, T, x, y):
    xHII = np.full(C, x[0]); xHeII = np.full(C, x[1]); xHeIII = np.full(C, x[2])
    nHa = np.full(C, nH) if np.isscalar(nH) else np.asarray(nH, dtype=np.float64)
    return State(np.full((G, C), N0), np.zeros((G, 3, C)), xHII, xHeII, xHeIII,
                 eth_from_T(T, nHa, xHII, xHeII, xHeIII, y), nHa)


def config0(n=32):
    """Isothermal single-source ionisation (octant of a Stroemgren sphere)."""
    box = 6.6 * KPC
    mesh = M.cartesian(n, box, periodic=False,
                       bc=(M.BC_REFLECT, M.BC_OUTFLOW, M.BC_REFLECT, M.BC_OUTFLOW, M.BC_REFLECT, M.BC_OUTFLOW))
    ct = 0.01 * C_LIGHT
    p = Params(ngroup=1, ctilde=ct, sigma=np.array([[6.3e-18, 0.0, 0.0]]), eps_heat=np.zeros((1, 3)),
               chem_mode=CHEM_H_ISOTHERMAL, T_fixed=1.0e4, alphaB_override=2.59e-13, y_he=0.0)
    st = _uniform_state(1, mesh.ncell, 0.0, 1.0e-3, 1.0e4, (1.2e-3, 0.0, 0.0), 0.0)
    src = Sources(np.array([0], dtype=np.int32), np.array([[5.0e48 / 8.0]]))
    return Workload("config0_stromgren_%d" % n, mesh, p, st, src, cfl_dt(mesh, ct),
                    {"ndot_full": 5.0e48, "t_end": 500 * MYR})


def config1(n=128):
    """Free-streaming beam and shadow behind an opaque clump."""
    mesh = M.cartesian(n, 1.0, periodic=False)
    h = 1.0 / n
    # Dirichlet ghost 0 on x=0 faces whose centre is within 0.2 of (0, 1/2, 1/2)
    fc = mesh.fcentroid
    on_x0 = (mesh.right < 0) & (mesh.normal[0] < -0.5)
    disc = on_x0 & ((fc[1] - 0.5) ** 2 + (fc[2] - 0.5) ** 2 <= 0.2 ** 2)
    mesh.right[disc] = M.BC_DIRICHLET0
    c = mesh.centroid
    r2 = (c[0] - 0.5) ** 2 + (c[1] - 0.5) ** 2 + (c[2] - 0.5) ** 2
    kappa = np.where(r2 < 0.1 ** 2, 1.0e3 / 0.2, 0.0)
    p = Params(ngroup=1, ctilde=1.0, chem_mode=CHEM_FIXED_OPACITY, kappa=kappa, n_floor=1.0e-10,
               ghost_state=np.array([[1.0, 1.0, 0.0, 0.0]]))
    st = _uniform_state(1, mesh.ncell, 1.0e-10, 1.0, 1.0, (0.0, 0.0, 0.0), 0.0)
    src = Sources(np.zeros(0, dtype=np.int32), np.zeros((1, 0)))
    return Workload("config1_beam_%d" % n, mesh, p, st, src, 0.3 * h / 1.0, {})


def _hhe_params(ct):
    return Params(ngroup=3, ctilde=ct, sigma=SIGMA3.copy(), eps_heat=EPS3.copy(), chem_mode=CHEM_HHE_THERMAL,
                  y_he=Y_HE)


def config2(n=64):
    """Multi-frequency H+He ionisation with thermal evolution on a clipped Voronoi mesh."""
    box = 6.6 * KPC * n / 64.0 if n < 64 else 6.6 * KPC
    mesh = M.voronoi(n, box, 0.3, SEED_MESH + 2, periodic=False, bc_code=M.BC_OUTFLOW)
    ct = 0.01 * C_LIGHT
    p = _hhe_params(ct)
    st = _uniform_state(3, mesh.ncell, 0.0, 1.0e-3, 100.0, (1.0e-6, 1.0e-6, 0.0), Y_HE)
    ic = n // 2
    cell = (ic * n + ic) * n + ic  # lattice cell holding the box centre
    src = Sources(np.array([cell], dtype=np.int32), (5.0e48 * SHARE3)[:, None].copy())
    return Workload("config2_hhe_%d" % n, mesh, p, st, src, cfl_dt(mesh, ct), {})


def gaussian_field(n, seed):
    """Unit-variance Gaussian random field with P(k) ~ k^-2 on the n^3 lattice."""
    w = rng.normal(seed, 0, np.arange(n ** 3, dtype=np.uint64)).reshape(n, n, n)
    k = np.fft.fftfreq(n) * n
    k2 = k[:, None, None] ** 2 + k[None, :, None] ** 2 + k[None, None, :] ** 2
    amp = np.zeros_like(k2)
    amp[k2 > 0] = 1.0 / np.sqrt(k2[k2 > 0])
    g = np.fft.ifftn(np.fft.fftn(w) * amp).real
    return (g / g.std()).ravel()


def reion_fields(n, seed_rho, seed_src, nsrc, sigma_ln=1.5, nH_mean=2.0e-4):
    g = gaussian_field(n, seed_rho)
    nH = nH_mean * np.exp(sigma_ln * g - 0.5 * sigma_ln ** 2)
    order = np.argsort(-nH, kind="stable")[:nsrc]
    cells = np.sort(order).astype(np.int32)
    lg = 50.0 + 3.0 * rng.u01(seed_src, 0, cells.astype(np.uint64))
    rate = SHARE3[:, None] * (10.0 ** lg)[None, :]
    return nH, Sources(cells, np.ascontiguousarray(rate))


def config34(n, cfg):
    """Reionisation-like periodic volume (cfg 3: n=256, cfg 4: n=384); host build."""
    spacing = 10.0 * KPC
    mesh = M.voronoi(n, n * spacing, 0.3, SEED_MESH + cfg, periodic=True)
    ct = 0.2 * C_LIGHT
    p = _hhe_params(ct)
    full = 256 if cfg == 3 else 384
    nsrc_full = 10000 if cfg == 3 else 34000
    nsrc = max(1, int(round(nsrc_full * (n / full) ** 3)))
    nH, src = reion_fields(n, SEED_RHO + cfg, SEED_SRC + cfg, nsrc)
    st = _uniform_state(3, mesh.ncell, 0.0, nH, 1.0e4, (1.0e-6, 1.0e-6, 0.0), Y_HE)
    return Workload("config%d_reion_%d" % (cfg, n), mesh, p, st, src, cfl_dt(mesh, ct), {"spacing": spacing})


def grey_blackbody(Tbb, edges_eV=(13.6, 24.6, 54.4, np.inf)):
    """Photon-number-weighted grey cross-sections [cm^2], mean excess energies [erg] and photon
    shares per group for a black body of temperature Tbb ("flux-weighted
    cross-sections and photoheating rates for each bin"), power-law sigma_j(nu) of SURVEY.md
    Appendix A, Gauss-Legendre panels.  Reproduces SIGMA3 / EPS3 / SHARE3 at 1e5 K
    (tests/test_oracle_physics.py); an input generator: it fixes the workload's constants."""
    kT = K_B * Tbb / EV
    thr = np.array([13.6, 24.6, 54.4])
    s0 = np.array([6.3e-18, 7.4e-18, 1.575e-18])
    slope = np.array([3.0, 2.0, 3.0])
    x, wq = np.polynomial.legendre.leggauss(64)
    G = len(edges_eV) - 1
    sig, eps, share = np.zeros((G, 3)), np.zeros((G, 3)), np.zeros(G)
    for g in range(G):
        lo = edges_eV[g]
        hi = min(edges_eV[g + 1], lo + 80.0 * kT)
        pts = np.geomspace(lo, hi, 33)
        a, b = pts[:-1, None], pts[1:, None]
        E = (0.5 * (b - a) * x + 0.5 * (b + a)).ravel()
        W = (0.5 * (b - a) * wq).ravel()
        with np.errstate(over="ignore"):
            nph = W * E ** 2 / np.expm1(E / kT)
        share[g] = nph.sum()
        for j in range(3):
            if lo < thr[j] - 1e-9:
                continue
            sj = s0[j] * (E / thr[j]) ** (-slope[j])
            sig[g, j] = (nph * sj).sum() / share[g]
            eps[g, j] = (nph * sj * (E - thr[j])).sum() / (nph * sj).sum() * EV
    return sig, eps, share / share.sum()


def hii_region(n=44):
    """Expanding H II region (eq 16, and its three-bin H+He variant PAPER.md:290):
    box (1.6 kpc)^3, n_H = n0 for r < r0 else n0 (r0/r)^2 with n0 = 3.2 cm^-3, r0 = 91.5 pc,
    T = 100 K, c~ = 1e-3 c, photons injected homogeneously (rate per volume constant) in a sphere
    of radius 0.05 kpc at the centre at 1e50 / 5e48 / 3e48 s^-1 per bin, grey constants from a
    5e4 K black body.  Mesh: the paper's 2 x N^3 staggered grid = the Voronoi cells of two
    interleaved cubic lattices (14-faced cells), generators offset by 5 % of the spacing (seeded) so that the
    clipped boundary cells are not degenerate; 2 x 44^3 = 170 368 cells at full size.  Not given by the paper
    (DESIGN.md 4): He mass fraction 0.24; dt from the CFL rule."""
    box = 1.6 * KPC
    mesh = M.voronoi(n, box, 0.05, SEED_MESH + 5, periodic=False, bc_code=M.BC_OUTFLOW, stagger=True)
    ct = 1.0e-3 * C_LIGHT
    sig, eps, _ = grey_blackbody(5.0e4)
    p = Params(ngroup=3, ctilde=ct, sigma=sig, eps_heat=eps, chem_mode=CHEM_HHE_THERMAL, y_he=Y_HE)
    c = mesh.centroid
    r = np.sqrt((c[0] - 0.5 * box) ** 2 + (c[1] - 0.5 * box) ** 2 + (c[2] - 0.5 * box) ** 2)
    r0 = 91.5e-3 * KPC
    nH = np.where(r < r0, 3.2, 3.2 * (r0 / np.maximum(r, r0)) ** 2)
    st = _uniform_state(3, mesh.ncell, 0.0, nH, 100.0, (1.0e-6, 1.0e-6, 0.0), Y_HE)
    inside = np.flatnonzero(r < 0.05 * KPC)
    if inside.size == 0:
        inside = np.array([int(np.argmin(r))])
    cells = inside.astype(np.int32)
    wv = mesh.volume[cells] / mesh.volume[cells].sum()
    rate = np.array([1.0e50, 5.0e48, 3.0e48])[:, None] * wv[None, :]
    return Workload("config5_hii_region_%d" % n, mesh, p, st, Sources(cells, np.ascontiguousarray(rate)),
                    cfl_dt(mesh, ct), {"r0": r0, "n0": 3.2})


def travelling_wave(n, jitter=0.1, order=2, seed=SEED_MESH + 9):
    """PAPER.md:280-284 (eq 17): E = 1 + 1e-6 sin(2 pi (x+y+z)), |F| = c E along (1,1,1), c = 1,
    periodic unit box, zero opacity, 'irregular mesh' = lattice generators offset by 10 %."""
    if jitter > 0:
        mesh = M.voronoi(n, 1.0, jitter, seed, periodic=True)
    else:
        mesh = M.cartesian(n, 1.0, periodic=True)
    c = mesh.centroid
    E = 1.0 + 1.0e-6 * np.sin(2.0 * np.pi * (c[0] + c[1] + c[2]))
    Fv = np.stack([E, E, E]) / np.sqrt(3.0)
    C = mesh.ncell
    st = State(E[None, :].copy(), Fv[None, :, :].copy(), np.zeros(C), np.zeros(C), np.zeros(C), np.ones(C), np.ones(C))
    p = Params(ngroup=1, ctilde=1.0, chem_mode=CHEM_NONE, order=order)
    src = Sources(np.zeros(0, dtype=np.int32), np.zeros((1, 0)))
    return Workload("travelling_wave_%d" % n, mesh, p, st, src, cfl_dt(mesh, 1.0), {})


def get(cfg, n=None):
    if cfg == 0:
        return config0(n or 32)
    if cfg == 1:
        return config1(n or 128)
    if cfg == 2:
        return config2(n or 64)
    if cfg in (3, 4):
        return config34(n or (256 if cfg == 3 else 384), cfg)
    if cfg == 5:
        return hii_region(n or 44)
    if cfg == 6:
        return travelling_wave(n or 128)
    raise ValueError(cfg)


def active_at(level, k, lmax):
    """Individual power-of-two time steps: a cell on level l of a hierarchy with finest level
    lmax takes a step every 2^(lmax - l) fine steps, so it is active at fine step k iff k is a multiple of
    that.  level: (C,) ints in [0, lmax].  Returns the (C,) boolean active mask of fine step k."""
    level = np.asarray(level)
    return (k % (1 << (lmax - level))) == 0


def levels_by_density(nH, lmax):
    """A synthetic level assignment for tests: denser cells (smaller cells and shorter time steps in a real
    run) sit on finer levels; quantiles of nH split the cells evenly over the lmax + 1 levels."""
    q = np.quantile(nH, np.linspace(0, 1, lmax + 2)[1:-1]) if lmax > 0 else np.zeros(0)
    return np.searchsorted(q, nH).astype(np.int8)
