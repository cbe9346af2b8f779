"""Pins of the oracle's active / passive machinery for individual time steps (PAPER.md:78,
258, 264-270; reading S27 of DESIGN.md).  CPU only.

  P20a  an all-active mask gives today's result bit for bit
  P20b  a passive region: cells without an active neighbour are bit-identical after the step; passive cells
        beside active ones keep their chemistry state and change only through the shared faces
  P20c  the photon budget closes to 1e-12 with mixed active sets and passive sources
  P20d  hand sums on the three-cell chain: the face between two passive cells carries nothing, the face
        between an active and a passive cell moves the same photons out of one and into the other
  P20e  a two-level power-of-two schedule keeps the budget closed and every invariant
"""
import numpy as np
import pytest

from paper_2404_17630_b200.inputs import configs as cfg
from paper_2404_17630_b200.inputs import mesh as M
from test_oracle_pins_he_energy_cap import _chain3


def _run(oracle_mod, w, active, nsub=2):
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(w.state)
    o.set_active(active)
    o.step(w.dt, nsub)
    return o.get_state(), o.ledger()


def _neighbour_has(mesh, mask):
    out = np.zeros(mesh.ncell, bool)
    ok = mesh.right >= 0
    l, r = mesh.left[ok], mesh.right[ok]
    np.logical_or.at(out, l, mask[r]); np.logical_or.at(out, r, mask[l])
    return out


def _budget(led, stored0):
    lhs = led["stored"] + led["absorbed"] + led["outflow"]
    rhs = stored0 + led["injected"] + led["inflow_bc"] + led["floor_added"]
    return np.max(np.abs(lhs - rhs) / np.abs(rhs))


def test_p20a_all_active_is_todays_result(oracle_mod):
    w = cfg.get(2, 6)
    a, la = _run(oracle_mod, w, None, 3)
    b, lb = _run(oracle_mod, w, np.ones(w.mesh.ncell, bool), 3)
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    for k in ("stored", "injected", "absorbed", "outflow"):
        assert np.array_equal(la[k], lb[k])


def test_p20b_passive_region(oracle_mod):
    w = cfg.get(2, 8)
    # develop the state first so that there is radiation everywhere near the source
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(w.state); o.step(w.dt, 6)
    s0 = o.get_state()
    w.state = cfg.State(s0["N"], s0["F"], s0["xHII"], s0["xHeII"], s0["xHeIII"], s0["eth"], s0["nH"])
    c = w.mesh.centroid
    active = c[0] < 0.5 * w.mesh.box[0]                       # the left half of the box takes the step
    got, _ = _run(oracle_mod, w, active, 1)
    touched = active | _neighbour_has(w.mesh, active)
    far = ~touched
    assert far.sum() > 50 and (touched & ~active).sum() > 20
    for k in ("N", "F", "xHII", "xHeII", "xHeIII", "eth"):
        assert np.array_equal(got[k][..., far], s0[k][..., far]), k          # bit-identical
    rim = touched & ~active                                    # passive cells with an active neighbour
    for k in ("xHII", "xHeII", "xHeIII", "eth"):
        assert np.array_equal(got[k][rim], s0[k][rim]), k      # no chemistry in passive cells
    assert np.any(got["N"][:, rim] != s0["N"][:, rim])         # but their photons moved through the shared faces
    assert np.any(got["xHII"][active] != s0["xHII"][active])


def test_p20c_budget_with_mixed_sets_and_passive_sources(oracle_mod):
    w = cfg.get(3, 8)
    stored0 = (w.state.N * w.mesh.volume).sum(1)
    rs = np.random.RandomState(3)
    active = rs.rand(w.mesh.ncell) < 0.4
    active[w.sources.cell[::2]] = True
    active[w.sources.cell[1::2]] = False                       # half of the sources sit in passive cells
    got, led = _run(oracle_mod, w, active, 4)
    assert _budget(led, stored0) < 1e-12
    want = 4 * w.dt * w.sources.rate[:, ::2].sum(1)            # only the active sources inject
    assert np.allclose(led["injected"], want, rtol=1e-13)
    assert got["N"].min() >= 0
    for g in range(3):
        assert np.all(np.sqrt((got["F"][g] ** 2).sum(0)) <= w.params.ctilde * got["N"][g] * (1 + 1e-14))


def test_p20d_three_cell_hand_sums(oracle_mod):
    # c = 1, dt = 1/4, V = A = 1, first order, forward Euler; N = (1, 2, 4), Fx = (1/4, 1/2, 1):
    #   face A = (0|1): Phi_N = (1/4 + 1/2)/2 - (2 - 1)/2 = -1/8;  face B = (1|2): Phi_N = (1/2 + 1)/2 - (4 - 2)/2 = -1/4
    # (negative: the donor is the right cell, far from empty: the cap is idle; reflective walls: Phi_N = 0)
    mesh = _chain3()
    p = cfg.Params(ngroup=1, ctilde=1.0, chem_mode=cfg.CHEM_NONE, order=1, heun=0, n_floor=0.0)
    N = np.array([[1.0, 2.0, 4.0]])
    F = np.zeros((1, 3, 3)); F[0, 0] = [0.25, 0.5, 1.0]
    w = cfg.Workload("chain3", mesh, p, cfg.State(N, F, np.zeros(3), np.zeros(3), np.zeros(3), np.ones(3), np.ones(3)),
                     cfg.Sources(np.zeros(0, np.int32), np.zeros((1, 0))), 0.25)
    dt, pa, pb = 0.25, -0.125, -0.25
    cases = {(1, 1, 1): [1 - dt * pa, 2 - dt * (pb - pa), 4 + dt * pb],
             (0, 1, 0): [1 - dt * pa, 2 - dt * (pb - pa), 4 + dt * pb],   # both faces touch the active cell
             (1, 0, 0): [1 - dt * pa, 2 + dt * pa, 4.0],                  # face B lies between two passive cells
             (0, 0, 1): [1.0, 2 - dt * pb, 4 + dt * pb],
             (0, 0, 0): [1.0, 2.0, 4.0]}
    for mask, want in cases.items():
        got, led = _run(oracle_mod, w, np.array(mask, dtype=bool), 1)
        assert np.array_equal(got["N"][0], np.array(want)), mask            # powers of two: exact
        assert got["N"][0].sum() == 7.0
    # the momentum flux of a wall is applied to an active cell only: cell 0's Fx with and without its walls
    a, _ = _run(oracle_mod, w, np.array([1, 1, 1], bool), 1)
    b, _ = _run(oracle_mod, w, np.array([0, 1, 0], bool), 1)
    assert a["F"][0, 0, 0] != b["F"][0, 0, 0] and a["F"][0, 0, 1] == b["F"][0, 0, 1]


def test_p20e_power_of_two_schedule(oracle_mod):
    w = cfg.get(3, 8)
    lmax = 2
    level = cfg.levels_by_density(w.state.nH, lmax)
    assert set(np.unique(level)) == {0, 1, 2}
    assert cfg.active_at(level, 0, lmax).all() and (cfg.active_at(level, 1, lmax) == (level == 2)).all()
    assert (cfg.active_at(level, 2, lmax) == (level >= 1)).all()
    stored0 = (w.state.N * w.mesh.volume).sum(1)
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(w.state)
    for k in range(2 * (1 << lmax)):                            # two full cycles of the hierarchy
        o.set_active(cfg.active_at(level, k, lmax))
        o.step(w.dt, 1)
    led, st = o.ledger(), o.get_state()
    assert _budget(led, stored0) < 1e-12
    assert st["N"].min() >= 0 and st["xHII"].max() <= 1.0
    # the coarsest cells did chemistry twice, the finest eight times: more sub-steps than one step of all cells ...
    assert led["substeps_total"] > w.mesh.ncell * 2
    # ... and fewer than eight steps of all cells would take at the very least
    assert led["substeps_total"] < 8 * led["substeps_max"] * w.mesh.ncell
