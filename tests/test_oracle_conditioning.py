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
