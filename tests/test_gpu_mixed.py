"""rt_params.mixed = 1 on the GPU (reading S28) against the oracle's
mixed-precision mode and against the fp64 oracle, through the C ABI.  Run with -m gpu.

Both sides of the first comparison do the same single-precision arithmetic in the same units, but not in the
same order (the kernels contract a*b+c into one rounding and sum a cell's faces over two lanes), so they agree
to a few single-precision roundings of the face flux, not bit for bit: the tolerance is TOL_MIXED = 1e-6 in the
domain-of-dependence metric of tests/parity.py (24 bits = 6e-8 relative per operation, a handful of operations,
fluxes of up to 16 faces).  What is exact in the mode is tested exactly: the photon budget (sums in double),
covariance under power-of-two changes of unit, cells that no flux reaches.
"""
import numpy as np
import pytest

from paper_2404_17630_b200.inputs import configs as cfg
from paper_2404_17630_b200.inputs import mesh as M
import parity as P

pytestmark = pytest.mark.gpu
TOL_MIXED = 1e-6


def _solver(w, mixed, state=None, tuning=None):
    from paper_2404_17630_b200 import rt
    w.params.mixed = mixed
    s = rt.Solver(w.mesh, w.params, tuning=tuning)
    s.init(state if state is not None else w.state, w.sources)
    w.params.mixed = 0
    return s


def _oracle(oracle_mod, w, mixed, state):
    w.params.mixed = mixed
    o = oracle_mod.Oracle(w.mesh, w.params)
    w.params.mixed = 0
    o.set_sources(w.sources); o.set_state(state)
    return o


# several tiles and a ragged last tile everywhere: tiles of 8 cells on the small meshes
@pytest.mark.parametrize("c,n,k,tile", [(0, 12, 30, 0), (1, 24, 30, 0), (2, 10, 20, 8), (3, 10, 15, 0), (4, 9, 15, 8), (5, 8, 20, 0),
                                        (6, 12, 5, 0), (2, 24, 20, 0)])
def test_mixed_step_from_developed_state(oracle_mod, c, n, k, tile):
    """The mixed GPU path runs k subcycles and downloads; both oracles advance that state by one subcycle."""
    w = cfg.get(c, n)
    s = _solver(w, 1, tuning={"tile_cells": tile} if tile else None)
    s.step(w.dt, k)
    dev, l0 = s.download()
    dev["nH"] = w.state.nH
    s.step(w.dt, 1)
    got, lg = s.download()
    st = P.as_state(dev)
    errs = {}
    for mixed in (1, 0):
        o = _oracle(oracle_mod, w, mixed, st)
        o.step(w.dt, 1)
        errs[mixed] = P.step_errors(w.mesh, w.params.ctilde, dev, o.get_state(), got)
    print("config %d at %d^3 after %d subcycles: vs mixed oracle" % (c, n, k), errs[1], "vs fp64 oracle", errs[0])
    for mixed in (1, 0):
        e = errs[mixed]
        assert e["N"] <= TOL_MIXED and e["F"] <= TOL_MIXED, (mixed, e)
        assert max(e["xHII"], e["xHeII"], e["xHeIII"]) <= 1e-9 and e["eth"] <= 1e-8, (mixed, e)   # chemistry stays fp64
    assert max(errs[0]["N"], errs[0]["F"]) > 1e-12          # (it is not the fp64 path that ran)
    stored0 = (w.state.N * w.mesh.volume).sum(1)
    assert P.budget_residual(lg, stored0).max() <= P.TOL_LEDGER
    assert got["N"].min() >= 0.0
    Fm = np.sqrt((got["F"] ** 2).sum(1))
    assert np.all(Fm <= w.params.ctilde * got["N"] * (1 + 1e-12))


@pytest.mark.parametrize("order,heun", [(1, 1), (2, 0), (1, 0)])
def test_mixed_other_integrator_settings(oracle_mod, order, heun):
    w = cfg.get(3, 10)
    w.params.order, w.params.heun = order, heun
    s = _solver(w, 1)
    s.step(w.dt, 10)
    dev, _ = s.download()
    dev["nH"] = w.state.nH
    s.step(w.dt, 1)
    got, lg = s.download()
    o = _oracle(oracle_mod, w, 1, P.as_state(dev))
    o.step(w.dt, 1)
    e = P.step_errors(w.mesh, w.params.ctilde, dev, o.get_state(), got)
    assert e["N"] <= TOL_MIXED and e["F"] <= TOL_MIXED, e
    assert P.budget_residual(lg, (w.state.N * w.mesh.volume).sum(1)).max() <= P.TOL_LEDGER


@pytest.mark.parametrize("k", [-40, 40])
def test_mixed_is_covariant_under_power_of_two_units(k):
    """U -> 2^k U gives 2^k times the result bit for bit (per-face units), although c~^2 N 2^40 would overflow
    single precision without them; so does a power-of-two change of the length unit."""
    w = cfg.travelling_wave(10, jitter=0.2)
    w.params.ctilde = 1.0e10
    w.state.F *= 1.0e10
    w.dt = cfg.cfl_dt(w.mesh, 1.0e10)
    s = _solver(w, 1)
    s.step(w.dt, 3)
    ref, _ = s.download()
    lam = 2.0 ** k
    st = w.state.copy()
    st.N *= lam; st.F *= lam
    s = _solver(w, 1, state=st)
    s.step(w.dt, 3)
    got, _ = s.download()
    assert np.array_equal(got["N"], lam * ref["N"]) and np.array_equal(got["F"], lam * ref["F"])


def test_mixed_keeps_a_contrast_below_single_precision():
    """Differences are formed in double before rounding: a 1e-10 contrast on an O(1) background diffuses as in
    the fp64 path (to 1e-5 of the change), where a flux of rounded states would lose it entirely."""
    mesh = M.cartesian(16, 1.0, periodic=True)
    C = mesh.ncell
    c = mesh.centroid
    N = 1.0 + 1e-10 * np.sin(2 * np.pi * c[0]) * np.cos(2 * np.pi * c[1])
    p = cfg.Params(ngroup=1, ctilde=1.0, chem_mode=cfg.CHEM_NONE, heun=0)
    st = cfg.State(N[None, :].copy(), np.zeros((1, 3, C)), np.zeros(C), np.zeros(C), np.zeros(C), np.ones(C), np.ones(C))
    w = cfg.Workload("contrast", mesh, p, st, cfg.Sources(np.zeros(0, np.int32), np.zeros((1, 0))), cfg.cfl_dt(mesh, 1.0), {})
    out = []
    for mixed in (0, 1):
        s = _solver(w, mixed)
        s.step(w.dt, 1)
        out.append(s.download()[0]["N"][0] - N)
    d64, d32 = out
    assert np.abs(d64).max() > 1e-12
    # (to 1e-5 of the change, or to two units in the last place of N = 1 where that is coarser)
    assert np.abs(d32 - d64).max() <= 1e-5 * np.abs(d64).max() + 2 * np.finfo(np.float64).eps
    assert np.abs(d32 - d64).max() <= 1e-3 * np.abs(d64).max()


@pytest.mark.parametrize("c,n", [(0, 16), (2, 12)])
def test_mixed_100_subcycles_against_the_fp64_path(c, n):
    """The long run, fp64 GPU path as the reference.  The photon budget still closes to 1e-12 and the ionised
    mass agrees to 1e-6, but single cells do NOT meet north_star's 1e-6 on the fractions: in the cells of an
    ionisation front N is orders of magnitude below its neighbours', so a flux error of 1e-7 of the
    neighbourhood is 1e-3 of the cell's own photons (measured: 2e-5 on config 0, 1e-7 on config 2 after 100
    subcycles).  That is the price of the mode (S28); the bound asserted here is 1e-4."""
    w = cfg.get(c, n)
    res = []
    for mixed in (0, 1):
        s = _solver(w, mixed)
        s.step(w.dt, 100)
        res.append(s.download())
    (a, la), (b, lb) = res
    dx = max(np.abs(a[f] - b[f]).max() for f in ("xHII", "xHeII", "xHeIII"))
    print("config %d at %d^3, 100 subcycles, mixed against fp64: max |dx| = %.2e" % (c, n, dx))
    assert dx <= 1e-4
    V, nH = w.mesh.volume, w.state.nH
    ia, ib = (a["xHII"] * nH * V).sum(), (b["xHII"] * nH * V).sum()
    assert abs(ia - ib) <= 1e-6 * ia
    assert P.budget_residual(lb, (w.state.N * w.mesh.volume).sum(1)).max() <= P.TOL_LEDGER
    assert P.ledger_errors(la, lb) <= 1e-5


def test_mixed_with_active_sets(oracle_mod):
    """Individual time steps (S27) in mixed precision: passive cells out of reach stay bit-identical."""
    w = cfg.get(2, 10)
    s = _solver(w, 1)
    s.step(w.dt, 8)
    dev, _ = s.download()
    dev["nH"] = w.state.nH
    active = w.mesh.centroid[0] < 0.5 * w.mesh.box[0]
    s.set_active(active)
    s.step(w.dt, 1)
    got, lg = s.download()
    o = _oracle(oracle_mod, w, 1, P.as_state(dev))
    o.set_active(active)
    o.step(w.dt, 1)
    ref = o.get_state()
    e = P.step_errors(w.mesh, w.params.ctilde, dev, ref, got)
    assert e["N"] <= TOL_MIXED and e["F"] <= TOL_MIXED, e
    same = np.all(ref["N"] == dev["N"], axis=0) & np.all(ref["F"] == dev["F"], axis=(0, 1))   # cells the oracle left alone
    assert same.sum() > 100
    assert np.array_equal(got["N"][:, same], dev["N"][:, same]) and np.array_equal(got["F"][:, :, same], dev["F"][:, :, same])
    assert P.budget_residual(lg, (w.state.N * w.mesh.volume).sum(1)).max() <= P.TOL_LEDGER
