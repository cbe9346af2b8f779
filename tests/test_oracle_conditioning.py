"""Conditioning of the oracle in the parity metric: its own response to 1-ulp input noise on a
developed config-0 state (optical depth ~10 per cell, N falling by e^-10 per cell ahead of the
front, empty cells next to streaming ones).  This is the test that rejected SURVEY.md's first
reading of the donor cap (scale all four flux components by theta: response 4e-2) in favour of
clamping |Phi_N| only (reading S11 in DESIGN.md: response ~1e-15).  CPU only."""
import copy

import numpy as np

from paper_2404_17630_b200.inputs import configs as cfg
import parity as P


def test_oracle_is_well_conditioned_in_the_parity_metric(oracle_mod):
    w = cfg.get(0, 12)
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(w.state)
    o.step(w.dt, 40)
    dev = o.get_state()
    p = copy.deepcopy(w.params)
    p.chem_mode = cfg.CHEM_NONE

    def run(st):
        a = oracle_mod.Oracle(w.mesh, p); a.set_sources(w.sources); a.set_state(P.as_state(st))
        a.step(w.dt, 1)
        return a.get_state()

    r0 = run(dev)
    rs = np.random.RandomState(0)
    d2 = {k: v.copy() for k, v in dev.items()}
    d2["N"] = d2["N"] * (1 + 1.1e-16 * rs.randn(*d2["N"].shape))
    d2["F"] = d2["F"] * (1 + 1.1e-16 * rs.randn(*d2["F"].shape))
    r1 = run(d2)
    e = P.step_errors(w.mesh, p.ctilde, dev, r0, r1)
    assert max(e["N"], e["F"]) < 1e-13


def test_beam_edge_needs_the_whole_domain_of_dependence(oracle_mod):
    """Config 1 (beam, N = 1 next to the floor 1e-10 within two cells): 1-ulp noise on the beam
    cells (absolute 1e-16) reaches cells two and three rings away whose own stencil holds only
    1e-10, so in the one-ring metric the oracle's own response exceeds the 1e-10 bar; on the scale
    of the subcycle's domain of dependence (4 rings: 2 Heun stages x (gradient + flux),
    tests/test_patch_oracle.py) it is ~1e-15.  This is why the full-size beam parity case uses
    rings = DEPENDENCE_RINGS."""
    w = cfg.get(1, 32)
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(w.state)
    o.step(w.dt, 30)
    dev = o.get_state()

    def run(st):
        a = oracle_mod.Oracle(w.mesh, w.params); a.set_sources(w.sources); a.set_state(P.as_state(st))
        a.step(w.dt, 1)
        return a.get_state()

    r0 = run(dev)
    rs = np.random.RandomState(0)
    d2 = {k: v.copy() for k, v in dev.items()}
    d2["N"] = d2["N"] * (1 + 1.1e-16 * rs.randn(*d2["N"].shape))
    d2["F"] = d2["F"] * (1 + 1.1e-16 * rs.randn(*d2["F"].shape))
    r1 = run(d2)
    e1 = P.step_errors(w.mesh, w.params.ctilde, dev, r0, r1, rings=1)
    e4 = P.step_errors(w.mesh, w.params.ctilde, dev, r0, r1, rings=P.DEPENDENCE_RINGS)
    assert max(e1["N"], e1["F"]) > 1e-10
    assert max(e4["N"], e4["F"]) < 1e-13


def test_substepping_is_chaotic_in_the_hii_region_source_cell(oracle_mod):
    """Config 5 (H II region): in the strongly irradiated, almost fully ionised source cell the
    controller of PAPER.md:238 takes several hundred sub-steps per subcycle and its accept/reject
    sequence amplifies 1e-13 relative input noise to the integration error (the number of trials
    changes, x moves by 1e-5..1e-4): the oracle itself fixes that cell's result only to that level.
    All but a handful of the 4096 cells respond below 1e-11.  parity.chaotic_cells finds such cells; the full-size
    config-5 GPU case compares them at the integration-error level and everything outside their
    domain of dependence at the usual tolerances."""
    w = cfg.get(5, 16)
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(w.state)
    o.step(w.dt, 40)
    dev = o.get_state()
    bad = P.chaotic_cells(oracle_mod, w, dev)
    assert 1 <= bad.sum() <= 10 and np.any(bad[w.sources.cell])      # of 4096 cells

    def chem(st):
        a = oracle_mod.Oracle(w.mesh, w.params); a.set_sources(w.sources); a.set_state(P.as_state(st))
        a.chemistry_only(w.dt)
        return a.get_state(), a.ledger()

    r0, l0 = chem(dev)
    spread, trials = 0.0, set()
    for seed in range(4):
        rs = np.random.RandomState(100 + seed)
        d2 = {k: v.copy() for k, v in dev.items()}
        d2["xHII"] = d2["xHII"] * (1 + 1e-13 * rs.randn(*d2["xHII"].shape))
        r1, l1 = chem(d2)
        spread = max(spread, float(np.max(np.abs(r1["xHII"] - r0["xHII"])[bad])))
        trials.add(int(l1["substeps_total"]))
        assert np.max(np.abs(r1["xHII"] - r0["xHII"])[~bad]) < 1e-10
    assert 1e-8 < spread < 5e-3 and len(trials | {int(l0["substeps_total"])}) > 1
