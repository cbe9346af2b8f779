"""Pins P1-P4 of the oracle: Stroemgren law, photon budget, invariants, beam speed; CPU only."""
import os

import numpy as np
import pytest

from paper_2404_17630_b200.inputs import configs as cfg

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _run(oracle_mod, w, nsub):
    o = oracle_mod.Oracle(w.mesh, w.params)
    o.set_sources(w.sources); o.set_state(w.state)
    o.step(w.dt, nsub)
    return o


def budget_residual(led, stored0):
    lhs = led["stored"] + led["absorbed"] + led["outflow"]
    rhs = stored0 + led["injected"] + led["inflow_bc"] + led["floor_added"]
    return np.abs(lhs - rhs) / np.maximum(np.abs(rhs), 1e-300)


def test_p1_stromgren_front_law(oracle_mod):
    """Config 0 recipe on a 16^3 mesh (same box): ionised volume follows r(t) = R_S (1-e^{-t/t_rec})^{1/3}."""
    gold = {}
    for l in open(os.path.join(GOLD, "stromgren.txt")):
        if l.strip() and l[0] != "#":
            k, v = l.split(); gold[k] = float(v)
    aB, nH, Nd = 2.59e-13, 1e-3, 5e48
    RS = (3 * Nd / (4 * np.pi * aB * nH ** 2)) ** (1 / 3)
    assert RS / cfg.KPC == pytest.approx(gold["R_S_kpc"], rel=1e-4)
    assert 1 / (aB * nH) / cfg.MYR == pytest.approx(gold["t_rec_Myr"], rel=1e-4)
    w = cfg.get(0, 16)
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(w.state)
    stored0 = (w.state.N * w.mesh.volume).sum(1)
    done = 0
    r = np.sqrt((w.mesh.centroid ** 2).sum(0))
    for T in (10, 30, 100):
        k = int(round(T * cfg.MYR / w.dt))
        o.step(w.dt, k - done); done = k
        s = o.get_state()
        rV = (3 * 8 * (s["xHII"] * w.mesh.volume).sum() / (4 * np.pi)) ** (1 / 3) / cfg.KPC
        assert rV == pytest.approx(gold[str(T)], rel=0.05), T      # north_star: within 5 %
        # x_HII = 0.5 radius from the shell-averaged profile: within one cell of the law
        h = w.mesh.meta["h"]
        shell = np.floor(r / h).astype(int)
        prof = np.bincount(shell, weights=s["xHII"]) / np.maximum(np.bincount(shell), 1)
        j = int(np.argmax(prof < 0.5))
        r05 = (j - 0.5 + (prof[j - 1] - 0.5) / (prof[j - 1] - prof[j])) * h / cfg.KPC
        assert abs(r05 - gold[str(T)]) < h / cfg.KPC
        assert s["N"].min() >= 0
        fn = np.sqrt((s["F"][0] ** 2).sum(0))
        assert np.all(fn <= w.params.ctilde * s["N"][0] * (1 + 1e-14))
    led = o.ledger()
    assert budget_residual(led, stored0).max() < 1e-12
    assert led["cells_hit_cap"] == 0


@pytest.mark.parametrize("c,n,nsub", [(1, 16, 30), (2, 8, 12), (3, 8, 6)])
def test_p2_p3_budget_and_invariants(oracle_mod, c, n, nsub):
    w = cfg.get(c, n)
    stored0 = (w.state.N * w.mesh.volume).sum(1)
    o = _run(oracle_mod, w, nsub)
    led = o.ledger()
    assert budget_residual(led, stored0).max() < 1e-12
    s = o.get_state()
    assert s["N"].min() >= w.params.n_floor
    for g in range(w.params.ngroup):
        fn = np.sqrt((s["F"][g] ** 2).sum(0))
        assert np.all(fn <= w.params.ctilde * s["N"][g] * (1 + 1e-14))
    if c >= 2:
        assert led["injected"].min() > 0 and led["absorbed"].min() > 0
        assert np.all(s["xHII"] >= 0) and np.all(s["xHII"] <= 1)
        assert np.all(s["xHeII"] + s["xHeIII"] <= 1 + 1e-14) and s["eth"].min() > 0
        assert s["xHII"].max() > (0.5 if c == 2 else 0.1)            # the source cells ionise
    if c == 1:
        assert led["inflow_bc"][0] > 0


def test_p4_beam_speed_and_shadow(oracle_mod):
    """Config 1 recipe at 32^3: front at x = c t, |F| = c N in the beam, shadow behind the clump."""
    n = 32
    w = cfg.get(1, n)
    h = 1.0 / n
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(w.state)
    cx, cy, cz = w.mesh.centroid
    axis_off = (np.abs(cy - 0.15 - 0.5) < 0.6 * h) & (np.abs(cz - 0.5) < 0.6 * h)   # a ray that misses the clump
    k1 = int(round(0.3 / w.dt))
    o.step(w.dt, k1)
    s = o.get_state()
    line = np.argsort(cx[axis_off]); x = cx[axis_off][line]; N = s["N"][0][axis_off][line]
    j = int(np.argmax(N < 0.5))
    xf = x[j - 1] + (N[j - 1] - 0.5) / (N[j - 1] - N[j]) * h
    assert abs(xf - k1 * w.dt) < 2 * h                                # front within 2 cells of c t
    inside = axis_off & (cx < 0.15)
    f = np.sqrt((s["F"][0] ** 2).sum(0)) / s["N"][0]
    assert np.all(f[inside] > 0.99) and np.all(f <= 1 + 1e-14)
    k2 = int(round(0.95 / w.dt))
    o.step(w.dt, k2 - k1)
    s = o.get_state()
    behind = (cx > 0.7) & (cx < 0.9) & ((cy - 0.5) ** 2 + (cz - 0.5) ** 2 < 0.04 ** 2)
    beam = (cx > 0.7) & (cx < 0.9) & (np.sqrt((cy - 0.5) ** 2 + (cz - 0.5) ** 2) > 0.13) & \
           (np.sqrt((cy - 0.5) ** 2 + (cz - 0.5) ** 2) < 0.17)
    ratio = s["N"][0][behind].mean() / s["N"][0][beam].mean()
    assert ratio < 0.5                                                # shadow (value unpinned by the paper)
    stored0 = (w.state.N * w.mesh.volume).sum(1)
    assert budget_residual(o.ledger(), stored0).max() < 1e-12
