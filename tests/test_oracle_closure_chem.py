"""Pins P10 (closure / Riemann flux) and P11 (chemistry closed forms) of the oracle; CPU only."""
import os

import numpy as np
import pytest

from paper_2404_17630_b200.inputs import configs as cfg
from paper_2404_17630_b200.inputs import mesh as M

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_chi_values_and_monotone(oracle_mod):
    assert oracle_mod.chi(0.0) == pytest.approx(1.0 / 3.0, abs=1e-15)
    assert oracle_mod.chi(1.0) == pytest.approx(1.0, abs=1e-15)
    assert oracle_mod.chi(2.0) == oracle_mod.chi(1.0)          # clamped (S1)
    f = np.linspace(0, 1, 201)
    c = np.array([oracle_mod.chi(x) for x in f])
    assert np.all(np.diff(c) > 0)
    # Levermore closure value at f = 1/2: (3+1)/(5+2 sqrt(13/4)) = 4/(5+sqrt(13))
    assert oracle_mod.chi(0.5) == pytest.approx(4.0 / (5.0 + np.sqrt(13.0)), abs=1e-15)


def test_eddington_trace_and_limits(oracle_mod):
    rs = np.random.RandomState(1)
    for _ in range(20):
        F = rs.randn(3)
        N = np.linalg.norm(F) / rs.uniform(0.05, 1.5)
        D = oracle_mod.eddington(N, F, 1.0)
        assert np.trace(D) == pytest.approx(1.0, abs=1e-14)
        assert np.allclose(D, D.T, atol=1e-16)
    D = oracle_mod.eddington(2.0, np.zeros(3), 1.0)            # isotropic: D = I/3
    assert np.allclose(D, np.eye(3) / 3, atol=1e-15)
    n = np.array([1.0, 2.0, -2.0]) / 3.0
    D = oracle_mod.eddington(2.0, 2.0 * 0.7 * n, 0.7)          # free streaming: D = n n^T
    assert np.allclose(D, np.outer(n, n), atol=1e-15)


def test_riemann_free_streaming_between_equal_states(oracle_mod):
    # f = 1 along the normal: Phi_N = c N, Phi_F = c^2 N n
    ct = 0.3
    n = np.array([2.0, -1.0, 2.0]) / 3.0
    N = 1.7
    U = np.concatenate([[N], ct * N * n])
    ph = oracle_mod.riemann(U, U, n, ct)
    assert ph[0] == pytest.approx(ct * N, rel=1e-15)
    assert np.allclose(ph[1:], ct * ct * N * n, rtol=1e-14, atol=0)


def test_riemann_matches_lab_frame_form_and_rotates(oracle_mod):
    from dense_reference import _glf
    rs = np.random.RandomState(7)
    for _ in range(50):
        n = rs.randn(3); n /= np.linalg.norm(n)
        ct = rs.uniform(0.1, 3.0)
        UL = np.concatenate([[rs.uniform(0.1, 2)], rs.randn(3) * 0.3])
        UR = np.concatenate([[rs.uniform(0.1, 2)], rs.randn(3) * 0.3])
        a = oracle_mod.riemann(UL, UR, n, ct)
        b = _glf(UL, UR, n, ct)
        assert np.allclose(a, b, rtol=0, atol=1e-14 * (1 + ct * ct))
        # covariance under a random rotation Q (P9 at the face level)
        Q, _ = np.linalg.qr(rs.randn(3, 3))
        ULr = np.concatenate([[UL[0]], Q @ UL[1:]]); URr = np.concatenate([[UR[0]], Q @ UR[1:]])
        c = oracle_mod.riemann(ULr, URr, Q @ n, ct)
        assert c[0] == pytest.approx(a[0], abs=1e-14 * (1 + ct))
        assert np.allclose(c[1:], Q @ a[1:], atol=1e-14 * (1 + ct * ct))
    # antisymmetry: swapping sides and flipping the normal flips the whole flux vector
    a = oracle_mod.riemann(UL, UR, n, ct); b = oracle_mod.riemann(UR, UL, -n, ct)
    assert b[0] == pytest.approx(-a[0], abs=1e-15) and np.allclose(b[1:], -a[1:], atol=1e-14)


def test_rates_against_appendixA_table(oracle_mod):
    rows = [l.split() for l in open(os.path.join(GOLD, "rates_appendixA.txt")) if l.strip() and l[0] != "#"]
    r4, r5 = oracle_mod.rates(1.0e4), oracle_mod.rates(1.0e5)
    for idx, name, v4, v5 in rows:
        k = int(idx)
        # brems slot holds the coefficient 1.42e-27 g_ff sqrt(T); same number
        assert r4[k] == pytest.approx(float(v4), rel=2e-4), name
        assert r5[k] == pytest.approx(float(v5), rel=2e-4), name


def _one_cell(oracle_mod, params):
    mesh = M.cartesian(1, 1.0, periodic=False)
    return oracle_mod.Oracle(mesh, params)


def test_recombination_only_closed_form(oracle_mod):
    # dx/dt = -alpha n x^2  ->  x(t) = x0 / (1 + alpha n x0 t)   (pure H, no photons, beta ~ 0 at 3e3 K)
    aB, nH, x0 = 2.59e-13, 1.0e-2, 0.9
    p = cfg.Params(ngroup=1, ctilde=1.0, sigma=np.array([[6.3e-18, 0, 0]]), chem_mode=cfg.CHEM_H_ISOTHERMAL,
                   T_fixed=3.0e3, alphaB_override=aB)
    o = _one_cell(oracle_mod, p)
    t_end = 3.0 / (aB * nH)
    r = o.chem_cell([0.0], [[0, 0, 0]], x0, 0, 0, 1.0, nH, t_end)
    exact = x0 / (1 + aB * nH * x0 * t_end)
    assert r["xHII"] == pytest.approx(exact, rel=0.02)
    tr = r["trace"]
    acc = tr[tr[:, 2] == 1]
    assert acc[:, 0].sum() == pytest.approx(t_end, rel=1e-14)   # accepted h sum to dt
    assert np.all(acc[:, 1] <= 0.1) and np.all(tr[tr[:, 2] == 0][:, 1] > 0.1)
    assert len(acc) > 10                                        # it did sub-step
    # step growth at most a factor 2 between accepted steps, except the clipped last one
    hs = acc[:, 0]
    assert np.all(hs[1:-1] <= 2.0 * hs[:-2] * (1 + 1e-14))


def test_photoionisation_equilibrium(oracle_mod):
    # photon field held fixed (reset every call), optically thin: Gamma (1-x) = alpha n x^2, Gamma = c sigma N
    aB, nH, sig, ct = 2.59e-13, 1.0e-3, 6.3e-18, 3.0e8
    p = cfg.Params(ngroup=1, ctilde=ct, sigma=np.array([[sig, 0, 0]]), chem_mode=cfg.CHEM_H_ISOTHERMAL,
                   T_fixed=3.0e3, alphaB_override=aB)
    o = _one_cell(oracle_mod, p)
    N0 = 1.0e-3
    Gam = ct * sig * N0
    dt = 0.002 / (ct * sig * nH)                                 # h D << 1
    x = 0.01
    for _ in range(4000):
        x = o.chem_cell([N0], [[0, 0, 0]], x, 0, 0, 1.0, nH, dt)["xHII"]
    a, b, c = aB * nH, Gam, -Gam
    xeq = (-b + np.sqrt(b * b - 4 * a * c)) / (2 * a)
    assert x == pytest.approx(xeq, rel=0.02)


def test_fixed_absorber_exponential_decay(oracle_mod):
    # huge absorber reservoir: x barely moves, N(t) -> N0 exp(-c sigma n t) at first order
    nH, sig, ct = 1.0, 6.3e-18, 3.0e8
    p = cfg.Params(ngroup=1, ctilde=ct, sigma=np.array([[sig, 0, 0]]), chem_mode=cfg.CHEM_H_ISOTHERMAL,
                   T_fixed=3.0e3, alphaB_override=1e-30)
    o = _one_cell(oracle_mod, p)
    D = ct * sig * nH
    N, F = np.array([1e-8]), np.array([[1e-9 * ct, 0, 0]])
    for _ in range(50):
        r = o.chem_cell(N, F, 0.0 if _ == 0 else r["xHII"], 0, 0, 1.0, nH, 0.02 / D)
        N, F = r["N"], r["F"]
    assert N[0] == pytest.approx(1e-8 * np.exp(-1.0), rel=0.02)
    assert F[0, 0] / N[0] == pytest.approx(0.1 * ct, rel=1e-12)   # N and F absorbed alike (S16)


def test_hhe_fractions_stay_closed_and_energy_positive(oracle_mod):
    p = cfg._hhe_params(0.01 * cfg.C_LIGHT)
    o = _one_cell(oracle_mod, p)
    nH = 1e-3
    e0 = cfg.eth_from_T(100.0, nH, 1e-6, 1e-6, 0.0, cfg.Y_HE)
    r = o.chem_cell([3e-4, 3e-4, 5e-5], np.zeros((3, 3)), 1e-6, 1e-6, 0.0, e0, nH, 1.0e13)
    assert 0 <= r["xHII"] <= 1 and 0 <= r["xHeII"] and 0 <= r["xHeIII"] and r["xHeII"] + r["xHeIII"] <= 1 + 1e-15
    assert r["eth"] > e0 and r["xHII"] > 1e-3                   # photo-heated and ionised
    acc = r["trace"][r["trace"][:, 2] == 1]
    assert acc[:, 0].sum() == pytest.approx(1.0e13, rel=1e-13)
    assert np.all(acc[:, 1] <= 0.1)
    assert np.all(r["N"] >= 0) and np.all(r["N"] <= [3e-4, 3e-4, 5e-5])
