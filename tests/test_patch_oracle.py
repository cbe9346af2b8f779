"""The patch extraction behind the full-size sampled-cell parity test (tests/parity.py:patch_around),
checked on the CPU: the oracle run on a 5-ring patch reproduces, for the seeds and their ring-1
neighbours, the oracle run on the whole mesh (periodic Voronoi and bounded Cartesian)."""
import numpy as np
import pytest

from paper_2404_17630_b200.inputs import configs as cfg
import parity as P


@pytest.mark.parametrize("c,n,k", [(3, 12, 6), (0, 14, 25), (5, 12, 10)])
def test_patch_reproduces_whole_mesh(oracle_mod, c, n, k):
    w = cfg.get(c, n)
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(w.state)
    o.step(w.dt, k)
    prev = o.get_state()
    o.step(w.dt, 1)
    ref = o.get_state()
    seeds = np.unique(np.concatenate([w.sources.cell[:2], [3, w.mesh.ncell // 2 + 5]])).astype(np.int64)
    pm, cells, ring = P.patch_around(w.mesh, seeds)
    assert pm.ncell < w.mesh.ncell and ring.max() == P.PATCH_RINGS and np.all(ring[np.isin(cells, seeds)] == 0)
    assert pm.left.min() >= 0 and pm.right.max() < pm.ncell and pm.left.max() < pm.ncell
    po = oracle_mod.Oracle(pm, w.params)
    po.set_sources(P.restrict_sources(w.sources, cells))
    po.set_state(P.restrict_state(prev, cells, w.state.nH))
    po.step(w.dt, 1)
    got = po.get_state()
    which = np.flatnonzero(ring <= 1)
    sub = lambda s: {"N": s["N"][:, cells], "F": s["F"][:, :, cells], "xHII": s["xHII"][cells], "xHeII": s["xHeII"][cells],
                     "xHeIII": s["xHeIII"][cells], "eth": s["eth"][cells]}
    e = P.cell_errors(pm, w.params.ctilde, sub(prev), sub(ref), got, which)
    assert max(e.values()) <= 1e-13, e
    # and the patch is not trivially the answer: its outermost ring differs (open faces)
    if c != 0:
        outer = np.flatnonzero(ring == P.PATCH_RINGS)
        assert outer.size > 0


def test_domain_of_dependence_is_four_rings(oracle_mod):
    """One subcycle (two Heun stages x (gradient + flux)) reaches exactly four rings of face
    neighbours: a 4-ring patch is exact for its seeds but not for their neighbours, a 3-ring patch is
    not exact for the seeds.  parity.DEPENDENCE_RINGS and PATCH_RINGS rest on this."""
    w = cfg.get(3, 12)
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(w.state)
    o.step(w.dt, 6)
    prev = o.get_state()
    o.step(w.dt, 1)
    ref = o.get_state()
    seeds = w.sources.cell[:2].astype(np.int64)
    keys = ("N", "F", "xHII", "xHeII", "xHeIII", "eth")
    err = {}
    for rings in (3, 4):
        pm, cells, ring = P.patch_around(w.mesh, seeds, rings=rings)
        po = oracle_mod.Oracle(pm, w.params)
        po.set_sources(P.restrict_sources(w.sources, cells))
        po.set_state(P.restrict_state(prev, cells, w.state.nH))
        po.step(w.dt, 1)
        got = po.get_state()
        sub = lambda s: {k: s[k][..., cells] for k in keys}
        for r in (0, 1):
            e = P.cell_errors(pm, w.params.ctilde, sub(prev), sub(ref), got, np.flatnonzero(ring <= r))
            err[rings, r] = max(e["N"], e["F"])
    assert P.DEPENDENCE_RINGS == 4 and P.PATCH_RINGS == P.DEPENDENCE_RINGS + 1
    assert err[4, 0] == 0.0 and err[4, 1] > 1e-12 and err[3, 0] > 1e-12, err
