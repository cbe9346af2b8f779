"""Pins of the oracle's mixed-precision mode (reading S28 of DESIGN.md).
CPU only.  The fp64 oracle, pinned by P1-P20, is the reference the mixed mode is held against: the mode is
an approximation of it with a stated error (single-precision rounding of the face flux), not a new method.

  P21a  one subcycle from a developed state: within 1e-6 of the fp64 oracle in the domain-of-dependence
        metric on every configuration; the photon budget still closes to 1e-12 (sums stay in double)
  P21b  a uniform field at rest on a periodic mesh: N bit-identical after one stage, the flux picks up
        single-precision noise only (the floor of the mode)
  P21c  differences are formed in double before rounding: a 1e-10 contrast on an O(1) background (below
        single-precision resolution) diffuses as in the fp64 oracle
  P21d  the per-face units make the flux scale-free: multiplying the state by 2^k multiplies the result
        by 2^k bit for bit, far outside the single-precision range of the unscaled flux c~^2 N
  P21e  100 subcycles: global quantities within 1e-5 of the fp64 run, budget closed, N >= 0, |F| <= c~ N
  P21f  the noise floor, stated: on the paper's travelling wave (amplitude 1e-6 on a background of 1, PAPER.md:
        280-284) one period in mixed precision differs from the fp64 run by 1e-7..5e-7 of the BACKGROUND (single-
        precision rounding of the mean flux and of the pressure), i.e. a quarter of the wave's amplitude: the mode
        is for contrasts well above 1e-6, and the test says so rather than hiding it
"""
import numpy as np
import pytest

import parity as P
from paper_2404_17630_b200.inputs import configs as cfg
from paper_2404_17630_b200.inputs import mesh as M


def _oracle(oracle_mod, w, mixed, state=None):
    w.params.mixed = mixed
    o = oracle_mod.Oracle(w.mesh, w.params)
    w.params.mixed = 0
    o.set_sources(w.sources)
    o.set_state(state if state is not None else w.state)
    return o


@pytest.mark.parametrize("c,n,k", [(0, 10, 10), (2, 8, 6), (3, 8, 4), (4, 12, 12), (5, 6, 8), (6, 12, 5)])
def test_p21a_one_step_against_fp64(oracle_mod, c, n, k):
    w = cfg.get(c, n)
    a = _oracle(oracle_mod, w, 0)
    a.step(w.dt, k)
    prev = a.get_state()
    st = P.as_state(prev)
    a.step(w.dt, 1)
    ref = a.get_state()
    b = _oracle(oracle_mod, w, 1, st)
    b.step(w.dt, 1)
    got, led = b.get_state(), b.ledger()
    e = P.step_errors(w.mesh, w.params.ctilde, prev, ref, got)
    assert 1e-12 < max(e["N"], e["F"]) < 1e-6, e            # single-precision rounding, and not the fp64 path
    for q in ("xHII", "xHeII", "xHeIII", "eth"):
        assert e[q] < 1e-6, (q, e)
    assert P.budget_residual(led, (st.N * w.mesh.volume).sum(1)).max() < 1e-12
    assert got["N"].min() >= 0.0


def test_p21b_uniform_field_at_rest_is_stationary(oracle_mod):
    mesh = M.voronoi(6, 1.0, 0.3, 77, periodic=True)
    C = mesh.ncell
    p = cfg.Params(ngroup=1, ctilde=3.0, chem_mode=cfg.CHEM_NONE)
    st = cfg.State(np.full((1, C), 0.7), np.zeros((1, 3, C)), np.zeros(C), np.zeros(C), np.zeros(C), np.ones(C), np.ones(C))
    w = cfg.Workload("uniform", mesh, p, st, cfg.Sources(np.zeros(0, np.int32), np.zeros((1, 0))), cfg.cfl_dt(mesh, 3.0), {})
    w.params.heun = 0
    o = _oracle(oracle_mod, w, 1)
    o.step(w.dt, 1)
    got = o.get_state()
    assert np.array_equal(got["N"], st.N)                     # no jump, no mean flux: Phi_N = 0 exactly
    # the pressure N/3 is the same on both sides of every face; its surface integral vanishes to
    # single-precision rounding only, which is the noise floor of the mode (S28)
    assert np.abs(got["F"]).max() < 1e-6 * 3.0 * 0.7
    w.params.heun = 1
    o = _oracle(oracle_mod, w, 1)
    o.step(w.dt, 3)
    got = o.get_state()
    assert np.abs(got["N"] - 0.7).max() < 1e-6 * 0.7 and np.abs(got["F"]).max() < 3e-6 * 3.0 * 0.7


def test_p21c_small_contrast_survives(oracle_mod):
    mesh = M.cartesian(8, 1.0, periodic=True)
    C = mesh.ncell
    c = mesh.centroid
    N = 1.0 + 1e-10 * np.sin(2 * np.pi * c[0]) * np.cos(2 * np.pi * c[1])
    p = cfg.Params(ngroup=1, ctilde=1.0, chem_mode=cfg.CHEM_NONE, heun=0)
    st = cfg.State(N[None, :].copy(), np.zeros((1, 3, C)), np.zeros(C), np.zeros(C), np.zeros(C), np.ones(C), np.ones(C))
    w = cfg.Workload("contrast", mesh, p, st, cfg.Sources(np.zeros(0, np.int32), np.zeros((1, 0))), cfg.cfl_dt(mesh, 1.0), {})
    out = []
    for mixed in (0, 1):
        o = _oracle(oracle_mod, w, mixed)
        o.step(w.dt, 1)
        out.append(o.get_state()["N"][0] - N)
    d64, d32 = out
    assert np.abs(d64).max() > 1e-12                          # the contrast diffuses
    assert np.abs(d32 - d64).max() < 1e-5 * np.abs(d64).max()


@pytest.mark.parametrize("k", [-40, 40, 90])
def test_p21d_scale_free(oracle_mod, k):
    w = cfg.travelling_wave(6, jitter=0.2)
    w.params.ctilde = 1.0e10                                  # c~^2 N 2^90 = 1e47: outside single precision unscaled
    w.state.F *= 1.0e10
    w.dt = cfg.cfl_dt(w.mesh, 1.0e10)
    a = _oracle(oracle_mod, w, 1)
    a.step(w.dt, 2)
    ref = a.get_state()
    lam = 2.0 ** k
    st = w.state.copy()
    st.N *= lam
    st.F *= lam
    b = _oracle(oracle_mod, w, 1, st)
    b.step(w.dt, 2)
    got = b.get_state()
    if k <= 40:
        assert np.array_equal(got["N"], lam * ref["N"]) and np.array_equal(got["F"], lam * ref["F"])
    else:
        # the cell values themselves leave the single-precision range: the stated limit of the mode is
        # |F| < 3e38 in the caller's units ("a suitable unit system"); nothing may turn
        # into NaN silently below it, and 2^90 * 1e10 = 1e37 is still inside
        assert np.all(np.isfinite(got["N"])) and np.all(np.isfinite(got["F"]))
        assert np.allclose(got["N"], lam * ref["N"], rtol=1e-6)


def test_p21e_hundred_subcycles(oracle_mod):
    w = cfg.get(0, 10)
    stored0 = (w.state.N * w.mesh.volume).sum(1)
    res = []
    for mixed in (0, 1):
        o = _oracle(oracle_mod, w, mixed)
        o.step(w.dt, 100)
        res.append((o.get_state(), o.ledger()))
    (s64, l64), (s32, l32) = res
    V = w.mesh.volume
    ion64, ion32 = (s64["xHII"] * s64["nH"] * V).sum(), (s32["xHII"] * s32["nH"] * V).sum()
    assert abs(ion32 - ion64) < 1e-5 * ion64
    assert np.abs(l32["stored"] - l64["stored"]).max() < 1e-5 * np.abs(l64["stored"]).max()
    assert np.abs(l32["absorbed"] - l64["absorbed"]).max() < 1e-5 * np.abs(l64["absorbed"]).max()
    assert P.budget_residual(l32, stored0).max() < 1e-12
    assert s32["N"].min() >= 0.0
    Fm = np.sqrt((s32["F"] ** 2).sum(1))
    assert np.all(Fm <= w.params.ctilde * s32["N"] * (1 + 1e-12))


def test_p21f_noise_floor_on_the_travelling_wave(oracle_mod):
    out = []
    for mixed in (0, 1):
        w = cfg.travelling_wave(16, jitter=0.0)
        o = _oracle(oracle_mod, w, mixed)
        T = 1.0 / np.sqrt(3.0)
        ns = int(np.ceil(T / w.dt))
        o.step(T / ns, ns)
        out.append(o.get_state()["N"][0])
    l1 = np.sum(w.mesh.volume * np.abs(out[1] - out[0]))      # relative to the background N = 1
    assert 1e-8 < l1 < 5e-7, l1                                # measured 2.3e-7: rounding noise, not a bias in the scheme
    assert abs(np.sum(w.mesh.volume * (out[1] - out[0]))) < 1e-15   # and it moves no photons: the sums are double
