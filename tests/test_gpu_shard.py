"""The sharded path on ONE GPU (include/rt.h "sharded runs"; paper_2404_17630_b200/shard.py): the mesh
cut into 2 or 3 contiguous Peano-Hilbert ranges, every shard a librt context of its own with ghost cells, advanced
in lock-step by shard.LocalGroup with the exchanges as plain device copies (no rank's kernels wait on another's).
Compared with the oracle on the whole mesh, and with the unsharded GPU path.  Run with -m gpu.

The sharded result is not bit-identical to the unsharded one: a cell's faces are summed in the order of its tile's
tables, which differs between a local and the global mesh (rounding order, 1e-16).  Tolerances: those of
tests/test_gpu_parity.py (parity.TOL_STEP in the domain-of-dependence metric, parity.TOL_LEDGER)."""
import numpy as np
import pytest

from paper_2404_17630_b200.inputs import configs as cfg
import parity as P

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("c,n,k,world,mixed", [(0, 12, 20, 2, 0), (1, 16, 20, 2, 0), (2, 10, 15, 2, 0), (3, 10, 12, 3, 0), (4, 9, 12, 2, 0),
                                               (5, 8, 15, 2, 0), (6, 12, 5, 2, 0), (3, 10, 12, 2, 1), (4, 32, 8, 4, 0),
                                               (0, 32, 20, 3, 0), (2, 64, 6, 2, 0)])   # the last two: configs 0 and 2 at BASELINE.json's full size
def test_sharded_step_from_developed_state(oracle_mod, c, n, k, world, mixed):
    from paper_2404_17630_b200 import shard as S
    w = cfg.get(c, n)
    w.params.mixed = mixed
    g = S.LocalGroup(w.mesh, w.params, w.state, w.sources, world)
    g.step(w.dt, k)
    dev, _ = g.download()
    dev["nH"] = w.state.nH
    g.step(w.dt, 1)
    got, lg = g.download()
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(P.as_state(dev))
    w.params.mixed = 0
    o.step(w.dt, 1)
    e = P.step_errors(w.mesh, w.params.ctilde, dev, o.get_state(), got)
    print("config %d at %d^3 on %d shards after %d subcycles:" % (c, n, world, k), e, [(s.shard.nown, s.shard.nghost) for s in g.ranks])
    tol = 1e-6 if mixed else P.TOL_STEP
    assert e["N"] <= tol and e["F"] <= tol, e
    assert max(e["xHII"], e["xHeII"], e["xHeIII"]) <= 1e-9 and e["eth"] <= 1e-8, e
    # the photon budget of the whole run: the shards' ledgers summed
    stored0 = (w.state.N * w.mesh.volume).sum(1)
    assert P.budget_residual(lg, stored0).max() <= P.TOL_LEDGER
    assert lg["nsub_done"] == k + 1
    assert all(s.exchanges == 1 + (k + 1) * (4 if w.params.order >= 2 and w.params.heun else 2) for s in g.ranks) or c == 1


@pytest.mark.parametrize("order,heun", [(1, 1), (2, 0), (1, 0)])
def test_sharded_other_integrator_settings(oracle_mod, order, heun):
    """First order has no gradient exchange, Heun off has three phases and swaps the state buffers."""
    from paper_2404_17630_b200 import shard as S
    w = cfg.get(3, 10)
    w.params.order, w.params.heun = order, heun
    g = S.LocalGroup(w.mesh, w.params, w.state, w.sources, 2)
    assert len([1 for _, x in g.ranks[0].phases() if x is not None]) == (2 if heun else 1) * (2 if order >= 2 else 1)
    g.step(w.dt, 9)
    dev, _ = g.download()
    dev["nH"] = w.state.nH
    g.step(w.dt, 1)
    got, lg = g.download()
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(P.as_state(dev))
    o.step(w.dt, 1)
    e = P.step_errors(w.mesh, w.params.ctilde, dev, o.get_state(), got)
    assert e["N"] <= P.TOL_STEP and e["F"] <= P.TOL_STEP, e
    assert max(e["xHII"], e["xHeII"], e["xHeIII"]) <= 1e-9 and e["eth"] <= 1e-8, e
    assert P.budget_residual(lg, (w.state.N * w.mesh.volume).sum(1)).max() <= P.TOL_LEDGER


@pytest.mark.parametrize("c,n", [(2, 10), (3, 10)])
def test_sharded_run_against_the_unsharded_gpu_path(c, n):
    """30 subcycles sharded and unsharded: the same run up to rounding order (ledgers to 1e-12, fractions to 1e-9:
    none of these configurations' cells is in the chaotic sub-stepping regime, tests/test_gpu_parity.py)."""
    from paper_2404_17630_b200 import rt, shard as S
    w = cfg.get(c, n)
    s = rt.Solver(w.mesh, w.params); s.init(w.state, w.sources)
    s.step(w.dt, 30)
    a, la = s.download()
    g = S.LocalGroup(w.mesh, w.params, w.state, w.sources, 2)
    g.step(w.dt, 30)
    b, lb = g.download()
    for f in ("xHII", "xHeII", "xHeIII"):
        assert np.abs(a[f] - b[f]).max() <= 1e-9, f
    sc = P.dependence_max(w.mesh, np.abs(a["N"]).max(0), rings=2)
    assert (np.abs(a["N"] - b["N"]) / np.maximum(sc, 1e-300)).max() <= 1e-9
    assert P.ledger_errors(la, lb) <= 1e-11
    assert P.budget_residual(lb, (w.state.N * w.mesh.volume).sum(1)).max() <= P.TOL_LEDGER


def test_sharded_individual_time_steps(oracle_mod):
    """Active / passive cells (S27) across shards: a ghost carries its owner's active bit."""
    from paper_2404_17630_b200 import shard as S
    w = cfg.get(2, 10)
    g = S.LocalGroup(w.mesh, w.params, w.state, w.sources, 2)
    g.step(w.dt, 8)
    dev, _ = g.download()
    dev["nH"] = w.state.nH
    rs = np.random.RandomState(7)
    seeds = rs.rand(w.mesh.ncell) < 0.02
    active = P.dependence_max(w.mesh, seeds.astype(np.float64), rings=2) > 0     # blobs, cut by the shard boundary
    assert 0.1 < active.mean() < 0.9
    g.set_active(active)
    g.step(w.dt, 1)
    got, lg = g.download()
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(P.as_state(dev))
    o.set_active(active)
    o.step(w.dt, 1)
    ref = o.get_state()
    e = P.step_errors(w.mesh, w.params.ctilde, dev, ref, got)
    assert e["N"] <= P.TOL_STEP and e["F"] <= P.TOL_STEP, e
    assert max(e["xHII"], e["xHeII"], e["xHeIII"]) <= 1e-9
    same = np.all(ref["N"] == dev["N"], axis=0) & np.all(ref["F"] == dev["F"], axis=(0, 1))
    assert same.sum() > 50
    assert np.array_equal(got["N"][:, same], dev["N"][:, same]) and np.array_equal(got["F"][:, :, same], dev["F"][:, :, same])
    assert P.budget_residual(lg, (w.state.N * w.mesh.volume).sum(1)).max() <= P.TOL_LEDGER


def test_phases_back_to_back_are_one_step_bit_for_bit():
    """rt_step_phase x 5 = rt_step(dt, 1); out-of-order phases and rt_step inside a subcycle are refused."""
    from paper_2404_17630_b200 import rt
    w = cfg.get(3, 8)
    a = rt.Solver(w.mesh, w.params); a.init(w.state, w.sources)
    b = rt.Solver(w.mesh, w.params); b.init(w.state, w.sources)
    for _ in range(3):
        a.step(w.dt, 1)
        for ph in range(5):
            b.step_phase(w.dt, ph)
    sa, la = a.download()
    sb, lb = b.download()
    for k in sa:
        assert np.array_equal(sa[k], sb[k]), k
    for k in ("stored", "injected", "absorbed", "outflow", "floor_added"):
        assert np.array_equal(la[k], lb[k]), k
    assert lb["nsub_done"] == 3
    b.step_phase(w.dt, 0)
    with pytest.raises(rt.RTError, match="out of order"):
        b.step_phase(w.dt, 2)
    with pytest.raises(rt.RTError, match="inside a subcycle"):
        b.step(w.dt, 1)
