"""GPU <-> oracle parity through the C ABI (run with -m gpu on the B200 box)."""
import numpy as np
import pytest

from paper_2404_17630_b200.inputs import configs as cfg
from paper_2404_17630_b200.inputs import mesh as M
import parity as P

pytestmark = pytest.mark.gpu


def _pair(oracle_mod, w, tuning=None):
    from paper_2404_17630_b200 import rt
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(w.state)
    s = rt.Solver(w.mesh, w.params, tuning=tuning); s.init(w.state, w.sources)
    return o, s


CASES = [(0, 12), (1, 24), (2, 10), (3, 10), (4, 9), (5, 10)]   # 5: H II region, SURVEY.md 8(f)2


@pytest.mark.parametrize("c,n", CASES)
def test_first_subcycle(oracle_mod, c, n):
    w = cfg.get(c, n)
    o, s = _pair(oracle_mod, w)
    prev = o.get_state()
    o.step(w.dt, 1); s.step(w.dt, 1)
    got, lg = s.download()
    e = P.step_errors(w.mesh, w.params.ctilde, prev, o.get_state(), got)
    assert e["N"] <= P.TOL_STEP and e["F"] <= P.TOL_STEP, e
    assert max(e["xHII"], e["xHeII"], e["xHeIII"]) <= 1e-10 and e["eth"] <= 1e-9, e
    assert P.ledger_errors(o.ledger(), lg) <= P.TOL_LEDGER


# (the last three: configs 0, 1 and 2 at BASELINE.json's full size, every cell compared)
@pytest.mark.parametrize("c,n,k", [(0, 12, 40), (1, 24, 40), (2, 10, 30), (3, 10, 20), (4, 9, 20), (5, 10, 30),
                                   (0, 32, 80), (1, 128, 100), (2, 64, 30)])
def test_step_from_developed_state(oracle_mod, c, n, k):
    """GPU runs k subcycles and downloads; the oracle advances that state by one subcycle and is
    compared with the GPU's k+1 (SURVEY.md 8(c) parity metric)."""
    from paper_2404_17630_b200 import rt
    w = cfg.get(c, n)
    s = rt.Solver(w.mesh, w.params); s.init(w.state, w.sources)
    s.step(w.dt, k)
    dev, _ = s.download()
    dev["nH"] = w.state.nH
    s.step(w.dt, 1)
    got, _ = s.download()
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(P.as_state(dev))
    o.step(w.dt, 1)
    e = P.step_errors(w.mesh, w.params.ctilde, dev, o.get_state(), got)
    print("config %d at %d^3 after %d subcycles:" % (c, n, k), e)     # N1, F1: the one-ring scale, reported beside the metric
    assert e["N"] <= P.TOL_STEP and e["F"] <= P.TOL_STEP, e
    assert max(e["xHII"], e["xHeII"], e["xHeIII"]) <= 1e-9 and e["eth"] <= 1e-8, e


@pytest.mark.parametrize("k", [2, 30])
def test_hii_region_full_size_outside_the_chaotic_cells(oracle_mod, k):
    """Config 5 at the paper's size (44^3 generators).  In the few strongly irradiated
    cells around the sources the oracle's own sub-stepping is chaotic (parity.chaotic_cells,
    tests/test_oracle_conditioning.py): there both sides must agree at the integration-error level;
    every cell outside those cells' domain of dependence is compared at the usual tolerances."""
    from paper_2404_17630_b200 import rt
    w = cfg.get(5, 44)
    s = rt.Solver(w.mesh, w.params); s.init(w.state, w.sources)
    s.step(w.dt, k)
    dev, _ = s.download()
    dev["nH"] = w.state.nH
    s.step(w.dt, 1)
    got, lg = s.download()
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(P.as_state(dev))
    o.step(w.dt, 1)
    ref = o.get_state()
    bad = P.chaotic_cells(oracle_mod, w, dev)
    reach = P.dependence_max(w.mesh, bad.astype(np.float64), rings=P.DEPENDENCE_RINGS) > 0
    C = w.mesh.ncell
    print("config 5 at 44^3, k = %d: %d chaotic cells, %d cells in their domain of dependence of %d" % (k, bad.sum(), reach.sum(), C))
    assert bad.sum() <= 0.002 * C and reach.sum() <= 0.1 * C
    e = P.cell_errors(w.mesh, w.params.ctilde, dev, ref, got, np.flatnonzero(~reach))
    assert e["N"] <= P.TOL_STEP and e["F"] <= P.TOL_STEP, e
    assert max(e["xHII"], e["xHeII"], e["xHeIII"]) <= 1e-9 and e["eth"] <= 1e-8, e
    for f in ("xHII", "xHeII", "xHeIII"):
        assert np.max(np.abs(got[f] - ref[f])) <= 5e-3, f
    assert np.max(np.abs(got["eth"] - ref["eth"]) / ref["eth"]) <= 2e-2
    assert lg["cells_hit_cap"] == 0 and got["N"].min() >= 0.0


# (0, 32) and (2, 64): configs 0 and 2 of BASELINE.json in full; (4, 24): the recipe of the timed config
@pytest.mark.parametrize("c,n", [(0, 12), (2, 10), (3, 10), (5, 10), (0, 32), (4, 24), (2, 64)])
def test_100_subcycles_fractions_and_ledger(oracle_mod, c, n):
    """north_star: ionised fractions within 1e-6 absolute after 100 subcycles, photon budget to 1e-12.
    Where the bound fails, the test asks the oracle whether the METHOD fixes the answer that well: it is
    run a second time from the same state with 1e-13 relative noise.  Around bright sources the adaptive
    sub-stepping of PAPER.md:238 is chaotic (every rejection is a discontinuity) and 100
    subcycles carry the difference across the box; the CUDA path must then lie within the oracle's own
    spread (counts printed).  Configs 0, 2, 3, 5 meet the 1e-6 bound outright."""
    w = cfg.get(c, n)
    o, s = _pair(oracle_mod, w)
    stored0 = (w.state.N * w.mesh.volume).sum(1)
    o.step(w.dt, 100); s.step(w.dt, 100)
    got, lg = s.download()
    ref = o.get_state()
    C = w.mesh.ncell
    fr = ("xHII", "xHeII", "xHeIII")
    dx = np.max([np.abs(got[k] - ref[k]) for k in fr], axis=0)
    off = dx > P.TOL_X
    nchaos, led_spread = 0, 0.0
    if off.any():
        # is it the method?  The ORACLE ALONE, started from the same state with 1e-13 relative noise, must
        # show the same kind of spread; the CUDA path has to land inside that family
        rs = np.random.RandomState(11)
        st2 = w.state.copy()
        for k in ("N", "xHII", "xHeII", "xHeIII", "eth"):
            a = getattr(st2, k)
            a *= 1.0 + 1e-13 * rs.randn(*a.shape)
        o2 = oracle_mod.Oracle(w.mesh, w.params); o2.set_sources(w.sources); o2.set_state(st2)
        o2.step(w.dt, 100)
        ref2 = o2.get_state()
        doo = np.max([np.abs(ref2[k] - ref[k]) for k in fr], axis=0)
        nchaos = int((doo > P.TOL_X).sum())
        print("config %d at %d^3 after 100 subcycles: CUDA vs oracle: %d of %d cells off by more than 1e-6 (max %.2e); the oracle "
              "against itself with 1e-13 input noise: %d cells (max %.2e): chaotic sub-stepping (DESIGN.md 6)"
              % (c, n, int(off.sum()), C, dx.max(), nchaos, doo.max()))
        assert nchaos > 0, "the oracle is well conditioned here: the CUDA path is wrong"
        assert dx.max() <= 10.0 * doo.max() and dx.max() <= 5e-3
        assert off.sum() <= 3 * nchaos + 0.01 * C
        assert np.median(dx) <= 10.0 * np.median(doo) + P.TOL_X
        led_spread = P.ledger_errors(o.ledger(), o2.ledger())      # how far the absorbed / stored split moves in the oracle itself
    else:
        print("config %d at %d^3 after 100 subcycles: max fraction error %.2e" % (c, n, dx.max()))
    lo = o.ledger()
    assert P.ledger_errors(lo, lg) <= (1e-11 if nchaos == 0 else 10.0 * led_spread)
    assert P.budget_residual(lg, stored0).max() <= P.TOL_LEDGER    # the CUDA path's own budget closes regardless
    if nchaos == 0:
        assert lg["substeps_total"] == lo["substeps_total"] and lg["substeps_max"] == lo["substeps_max"]
    assert got["N"].min() >= w.params.n_floor and lg["cells_hit_cap"] == 0
    for g in range(w.params.ngroup):
        fn = np.sqrt((got["F"][g] ** 2).sum(0))
        assert np.all(fn <= w.params.ctilde * got["N"][g] * (1 + 1e-14))


@pytest.mark.parametrize("order,heun", [(2, 0), (1, 1)])
def test_other_integrator_settings(oracle_mod, order, heun):
    """Second order with forward Euler, first order with Heun (the default is 2 / Heun; 1 / Euler is in
    test_restart_bit_exact_and_first_order_euler)."""
    w = cfg.get(2, 8)
    w.params.order, w.params.heun = order, heun
    o, s = _pair(oracle_mod, w)
    prev = o.get_state()
    for _ in range(5):
        prev = o.get_state()
        o.step(w.dt, 1); s.step(w.dt, 1)
    got, lg = s.download()
    e = P.step_errors(w.mesh, w.params.ctilde, prev, o.get_state(), got)
    assert e["N"] <= P.TOL_STEP and e["F"] <= P.TOL_STEP, e
    assert P.ledger_errors(o.ledger(), lg) <= 1e-11


def test_substep_cap_is_hit_alike(oracle_mod):
    """max_substeps small enough that the stiff cells run into it (PAPER.md:238's loop is cut): both
    sides count the same cells and leave them in the same state."""
    w = cfg.get(2, 8)
    w.params.max_substeps = 6
    o, s = _pair(oracle_mod, w)
    o.step(w.dt, 8); s.step(w.dt, 8)
    got, lg = s.download()
    lo, ref = o.ledger(), o.get_state()
    assert lo["cells_hit_cap"] > 0 and lg["cells_hit_cap"] == lo["cells_hit_cap"]
    assert lg["substeps_total"] == lo["substeps_total"] and lg["substeps_max"] == lo["substeps_max"] == 6
    for k in ("xHII", "xHeII", "xHeIII"):
        assert np.max(np.abs(got[k] - ref[k])) <= 1e-9, k
    assert P.ledger_errors(lo, lg) <= 1e-11


def test_gradients_match_oracle(oracle_mod):
    w = cfg.get(2, 8)
    rs = np.random.RandomState(0)
    C = w.mesh.ncell
    w.state.N[:] = rs.uniform(0.5, 2, (3, C))
    w.state.F[:] = rs.randn(3, 3, C) * 0.1
    o, s = _pair(oracle_mod, w)
    gN, gF = o.gradients()
    hN, hF = s.gradients()
    sc = np.abs(gN).max()
    assert np.max(np.abs(gN - hN)) <= 1e-12 * sc
    assert np.max(np.abs(gF - hF)) <= 1e-12 * np.abs(gF).max()


@pytest.mark.parametrize("kind", ["open2", "periodic2", "mixed_bc3"])
def test_tiny_meshes_and_boundaries(oracle_mod, kind):
    ct = 0.8
    ghost = np.array([[1.3, 0.5, 0.1, -0.2]])
    mesh = {"open2": lambda: M.cartesian(2, 1.0, periodic=False), "periodic2": lambda: M.cartesian(2, 1.0, periodic=True),
            "mixed_bc3": lambda: M.cartesian(3, 1.5, periodic=False, bc=(-2, -1, -3, -2, -1, -3))}[kind]()
    rs = np.random.RandomState(3)
    C = mesh.ncell
    N = rs.uniform(0.5, 2.0, (1, C)); F = rs.randn(1, 3, C) * 0.2
    st = cfg.State(N, F, np.zeros(C), np.zeros(C), np.zeros(C), np.ones(C), np.ones(C))
    p = cfg.Params(ngroup=1, ctilde=ct, ghost_state=ghost)
    w = cfg.Workload(kind, mesh, p, st, cfg.Sources(np.zeros(0, np.int32), np.zeros((1, 0))), cfg.cfl_dt(mesh, ct))
    o, s = _pair(oracle_mod, w)
    prev = o.get_state()
    o.step(w.dt, 3); s.step(w.dt, 3)
    got, lg = s.download()
    e = P.step_errors(mesh, ct, prev, o.get_state(), got)
    assert e["N"] <= 1e-12 and e["F"] <= 1e-12, e
    assert P.ledger_errors(o.ledger(), lg) <= P.TOL_LEDGER


def test_restart_bit_exact_and_first_order_euler(oracle_mod):
    from paper_2404_17630_b200 import rt
    w = cfg.get(2, 8)
    a = rt.Solver(w.mesh, w.params); a.init(w.state, w.sources); a.step(w.dt, 6)
    b = rt.Solver(w.mesh, w.params); b.init(w.state, w.sources); b.step(w.dt, 3)
    mid, _ = b.download(); mid["nH"] = w.state.nH
    c = rt.Solver(w.mesh, w.params); c.init(mid, w.sources); c.step(w.dt, 3)
    sa, _ = a.download(); sc, _ = c.download()
    for k in sa:
        assert np.array_equal(sa[k], sc[k]), k                       # P13
    w.params.order, w.params.heun = 1, 0
    o, s = _pair(oracle_mod, w)
    prev = o.get_state()
    o.step(w.dt, 5); s.step(w.dt, 5)
    got, lg = s.download()
    e = P.step_errors(w.mesh, w.params.ctilde, prev, o.get_state(), got)
    assert e["N"] <= 1e-9 and e["F"] <= 1e-9, e


def test_device_resident_inputs_and_outputs(oracle_mod):
    import torch
    from paper_2404_17630_b200 import rt
    w = cfg.get(3, 8)
    h = rt.Solver(w.mesh, w.params); h.init(w.state, w.sources); h.step(w.dt, 4)
    ref, _ = h.download()
    dm = M.Mesh(w.mesh.ncell, w.mesh.nface, w.mesh.box, w.mesh.periodic,
                *[torch.as_tensor(getattr(w.mesh, k)).cuda() for k in
                  ("volume", "centroid", "area", "normal", "fcentroid", "left", "right")])
    ds = {k: torch.as_tensor(getattr(w.state, k)).cuda() for k in ("N", "F", "xHII", "xHeII", "xHeIII", "eth", "nH")}
    d = rt.Solver(dm, w.params); d.init(ds, w.sources); d.step(w.dt, 4)
    got, _ = d.download(device=True)
    for k in ref:
        assert np.array_equal(ref[k], got[k].cpu().numpy()), k


def test_errors_are_reported_not_thrown_across_the_abi():
    import torch
    from paper_2404_17630_b200 import rt
    mesh = M.cartesian(3, 1.0)
    p = cfg.Params(ngroup=1)
    bad = M.cartesian(3, 1.0)
    bad.right[0] = 10 ** 6
    with pytest.raises(rt.RTError, match="right index"):
        rt.Solver(bad, p)
    bad = M.cartesian(3, 1.0)
    bad.area[5] *= 1.5
    with pytest.raises(rt.RTError, match="not closed"):
        rt.Solver(bad, p)
    h = rt.rt_create(0, None)
    with pytest.raises(rt.RTError, match="rt_mesh_upload first"):
        rt.rt_state_init(h, p, cfg._uniform_state(1, 27, 1.0, 1.0, 1.0, (0, 0, 0), 0.0))
    with pytest.raises(rt.RTError, match="rt_state_init first"):
        rt.rt_step(h, 0.1, 1)
    with pytest.raises(rt.RTError, match="tile_cells"):
        rt.rt_set_tuning(h, tile_cells=3)
    ok = rt.Solver(mesh, p)
    twice = cfg.Sources(np.array([4, 7, 4], dtype=np.int32), np.ones((1, 3)))
    with pytest.raises(rt.RTError, match="listed twice"):
        ok.init(cfg._uniform_state(1, 27, 1.0, 1.0, 1.0, (0, 0, 0), 0.0), twice)
    ws = torch.empty(16, dtype=torch.float64, device="cuda")
    with pytest.raises(rt.RTError, match="workspace has"):
        rt.rt_mesh_upload(h, mesh, 1, None, ws)
    rt.rt_destroy(h)


def _regroup(w, G):
    """The config-2 workload with G frequency groups: cross-sections, heating energies and source
    shares of the three stock groups spread over G (input generation only, no method arithmetic)."""
    rs = np.random.RandomState(100 + G)
    C = w.mesh.ncell
    pick = np.arange(G) % 3
    scale = rs.uniform(0.6, 1.4, (G, 1))
    p = w.params
    p.ngroup = G
    p.sigma = cfg.SIGMA3[pick] * scale
    p.eps_heat = cfg.EPS3[pick] * rs.uniform(0.8, 1.2, (G, 1))
    share = rs.uniform(0.2, 1.0, G); share /= share.sum()
    total = w.sources.rate.sum(0)
    src = cfg.Sources(w.sources.cell, share[:, None] * total[None, :])
    N = np.repeat(w.state.N[:1], G, 0) * rs.uniform(0.5, 2.0, (G, C))
    F = rs.randn(G, 3, C) * 0.05 * p.ctilde * N[:, None, :]
    st = cfg.State(N, F, w.state.xHII, w.state.xHeII, w.state.xHeIII, w.state.eth, w.state.nH)
    return cfg.Workload(w.name + "_G%d" % G, w.mesh, p, st, src, w.dt)


@pytest.mark.parametrize("G", [2, 4, 5, 8])
def test_other_group_counts(oracle_mod, G):
    """The kernels are instantiated for 1..8 groups; configs 0-4 only use 1 and 3."""
    from paper_2404_17630_b200 import rt
    w = _regroup(cfg.get(2, 8), G)
    s = rt.Solver(w.mesh, w.params); s.init(w.state, w.sources)
    s.step(w.dt, 6)
    dev, _ = s.download(); dev["nH"] = w.state.nH
    s.step(w.dt, 1)
    got, lg = s.download()
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(P.as_state(dev))
    o.step(w.dt, 1)
    e = P.step_errors(w.mesh, w.params.ctilde, dev, o.get_state(), got)
    assert e["N"] <= P.TOL_STEP and e["F"] <= P.TOL_STEP, e
    assert max(e["xHII"], e["xHeII"], e["xHeIII"]) <= 1e-9 and e["eth"] <= 1e-8, e
    stored0 = (w.state.N * w.mesh.volume).sum(1)
    assert P.budget_residual(lg, stored0).max() <= P.TOL_LEDGER


@pytest.mark.parametrize("tc", [8, 12, 20])
def test_small_tiles_many_halos(oracle_mod, tc):
    """Forces small tiles (rt_tuning.tile_cells): most faces then cross tile boundaries, so the exchange
    of fluxes through xphi / k_finish and the halo tables carry the result; ragged last tile."""
    w = cfg.get(3, 9)                      # 729 cells: not a multiple of any tile size used here
    o, s = _pair(oracle_mod, w, tuning={"tile_cells": tc})
    assert s.tile_info()["cells_per_tile"] <= tc
    prev = o.get_state()
    for _ in range(4):
        prev = o.get_state()
        o.step(w.dt, 1); s.step(w.dt, 1)
    got, lg = s.download()
    e = P.step_errors(w.mesh, w.params.ctilde, prev, o.get_state(), got)
    assert e["N"] <= 1e-9 and e["F"] <= 1e-9, e
    assert P.ledger_errors(o.ledger(), lg) <= 1e-11


def test_chemistry_passes_keep_the_per_cell_trial_sequence(oracle_mod):
    """The sub-stepping runs in passes over compacted lists of unfinished cells (a scheduling choice):
    every cell must still go through the oracle's sequence of trials, so the counts agree exactly."""
    from paper_2404_17630_b200 import rt
    w = cfg.get(2, 8)
    a = rt.Solver(w.mesh, w.params); a.init(w.state, w.sources); a.step(w.dt, 12)
    _, la = a.download()
    o = oracle_mod.Oracle(w.mesh, w.params); o.set_sources(w.sources); o.set_state(w.state)
    o.step(w.dt, 12)
    assert la["substeps_total"] == o.ledger()["substeps_total"]
    assert la["substeps_max"] == o.ledger()["substeps_max"] > 2      # later passes were exercised


def test_zero_subcycles_and_zero_sources_leave_the_state_alone():
    from paper_2404_17630_b200 import rt
    w = cfg.get(2, 8)
    none = cfg.Sources(np.zeros(0, np.int32), np.zeros((w.params.ngroup, 0)))
    s = rt.Solver(w.mesh, w.params); s.init(w.state, none)
    s.step(w.dt, 0)
    got, lg = s.download()
    assert np.array_equal(got["N"], w.state.N) and np.array_equal(got["F"], w.state.F)
    assert np.array_equal(got["xHII"], w.state.xHII) and np.array_equal(got["eth"], w.state.eth)
    assert lg["nsub_done"] == 0 and np.all(lg["injected"] == 0.0)
    s.step(w.dt, 2)                              # no sources: nothing is injected, the budget still closes
    _, lg = s.download()
    stored0 = (w.state.N * w.mesh.volume).sum(1)
    assert np.all(lg["injected"] == 0.0) and P.budget_residual(lg, stored0).max() <= P.TOL_LEDGER


@pytest.mark.parametrize("c,n,mixed", [(3, 256, 0), (4, 384, 0), (3, 256, 1)])
def test_full_size_sampled_cells(oracle_mod, c, n, mixed):
    """BASELINE.json's configs 3 and 4 at their full sizes (16.8 M and 56.6 M cells; for config 4 the
    mesh and launch configuration `bench.py` times): the oracle cannot run the whole mesh in seconds, so it computes sampled
    cells one by one.  After three subcycles on the GPU the state is downloaded; the oracle advances
    the 5-ring patches around the sampled cells (sources and cells away from them) by one subcycle
    from that state and is compared, on the samples and their face neighbours, with the GPU's
    fourth subcycle.  `tests/test_patch_oracle.py` shows on the CPU that such a patch reproduces the
    whole-mesh oracle exactly on those cells.  mixed = 1: rt_params.mixed against the oracle's mixed mode
    (tests/test_gpu_mixed.py for the tolerance)."""
    import torch
    from paper_2404_17630_b200 import rt
    from paper_2404_17630_b200.inputs import device as devin
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info(0)
    if free < (160e9 if n == 384 else 60e9):
        pytest.skip("needs a whole 180 GB B200 (%.0f GB free)" % (free / 1e9))
    w = devin.config34_device(n, c, "cuda:0")
    w.params.mixed = mixed
    C = w.mesh.ncell
    s = rt.Solver(w.mesh, w.params)
    # 64+ samples, stratified over what could go wrong at size (rt_debug_tiles): cells of class-B flux tiles
    # (second launch, larger capacities), of the tiles with the largest tables / forward halo / face count,
    # of the first and the last (ragged) tile, the brightest and faintest sources, and cells anywhere
    of_cell, desc = s.tiles()
    T = desc.shape[0]
    rs = np.random.RandomState(7)
    pick = lambda tile: int(rs.choice(np.flatnonzero(of_cell == tile)))
    strata = {}
    classB = np.flatnonzero(desc[:, 3] == 1)
    strata["class B"] = [pick(t) for t in rs.choice(classB, min(12, classB.size), replace=False)] if classB.size else []
    strata["largest tables"] = [pick(int(np.argmax(desc[:, 2])))]
    strata["largest forward halo"] = [pick(int(np.argmax(desc[:, 1])))]
    strata["most owned faces"] = [pick(int(np.argmax(desc[:, 0])))]
    strata["first tile"] = [pick(0)]
    strata["last tile"] = [pick(T - 1)]
    order = np.argsort(w.sources.rate.sum(0))
    strata["sources"] = [int(x) for x in w.sources.cell[order[[0, 1, 2, -3, -2, -1]]]]
    strata["anywhere"] = [int(x) for x in rs.randint(0, C, 44)]
    seeds = np.unique(np.concatenate([np.asarray(v, dtype=np.int64) for v in strata.values()]))
    for name, v in strata.items():
        print("stratum %-22s cells %s  tiles %s  class %s" % (name, v[:6], [int(of_cell[x]) for x in v[:6]],
                                                             ["AB"[desc[of_cell[x], 3]] for x in v[:6]]))
    assert seeds.size >= 60 and len(strata["class B"]) >= min(8, classB.size)
    del of_cell
    pm, cells, ring = P.patch_around(w.mesh, seeds, xp=torch)
    assert seeds.size * 300 < pm.ncell < seeds.size * 3000 and ring.max() == P.PATCH_RINGS
    w.mesh = None
    torch.cuda.empty_cache()
    s.init(w.state, w.sources)
    nH = w.state.nH.cpu().numpy()
    w.state = None
    torch.cuda.empty_cache()
    k = 3
    s.step(w.dt, k)
    prev, _ = s.download()
    s.step(w.dt, 1)
    got, lg = s.download()
    assert lg["cells_hit_cap"] == 0
    o = oracle_mod.Oracle(pm, w.params)
    o.set_sources(P.restrict_sources(w.sources, cells))
    o.set_state(P.restrict_state(prev, cells, nH))
    o.step(w.dt, 1)
    ref = o.get_state()
    sub = lambda st: {"N": st["N"][:, cells], "F": st["F"][:, :, cells], "xHII": st["xHII"][cells],
                      "xHeII": st["xHeII"][cells], "xHeIII": st["xHeIII"][cells], "eth": st["eth"][cells]}
    which = np.flatnonzero(ring <= 1)
    pprev, pgot = sub(prev), sub(got)
    assert np.abs(pprev["N"][:, which]).max() > 0 and np.any(pgot["N"][:, which] != pprev["N"][:, which])
    e = P.cell_errors(pm, w.params.ctilde, pprev, ref, pgot, which)
    print("full-size sampled parity: config %d, n = %d, %d seeds, %d patch cells, %d compared:" % (c, n, seeds.size, pm.ncell, which.size), e)
    tol = 1e-6 if mixed else P.TOL_STEP
    assert e["N"] <= tol and e["F"] <= tol, e
    assert max(e["xHII"], e["xHeII"], e["xHeIII"]) <= 1e-9 and e["eth"] <= 1e-8, e
    s.close()
    del s, w
    gc.collect()
    torch.cuda.empty_cache()


# ------------------------------------------------------------------ individual time steps
def _untouched(mesh, active):
    t = active.copy()
    ok = mesh.right >= 0
    l, r = mesh.left[ok], mesh.right[ok]
    np.logical_or.at(t, l, active[r]); np.logical_or.at(t, r, active[l])
    return ~t


@pytest.mark.parametrize("c,n,frac", [(2, 10, 0.4), (3, 10, 0.15), (0, 12, 0.5), (1, 24, 0.3)])
def test_active_sets_match_the_oracle(oracle_mod, c, n, frac):
    """rt_set_active (reading S27): a random subset of the cells takes the RT step;
    half of the sources sit in passive cells.  Per-step parity, the ledger, and the cells without an active
    neighbour bit for bit."""
    w = cfg.get(c, n)
    C = w.mesh.ncell
    rs = np.random.RandomState(5)
    # blobs of active cells (so that whole tiles are passive) plus scattered ones
    cen = w.mesh.centroid / np.asarray(w.mesh.box)[:, None]
    active = (np.sin(5.0 * cen[0]) * np.cos(4.0 * cen[1] + 1.0) + 0.3 * rs.rand(C) > 1.0 - 2.0 * frac)
    if len(w.sources.cell):
        active[w.sources.cell[::2]] = True
        active[w.sources.cell[1::2]] = False
    assert 0.02 * C < active.sum() < 0.9 * C
    o, s = _pair(oracle_mod, w)
    o.step(w.dt, 3); s.step(w.dt, 3)                            # develop a little with every cell active
    o.set_active(active); s.set_active(active)
    start, _ = s.download()
    o.step(w.dt, 2); s.step(w.dt, 2)
    # per-step parity from the CUDA path's own state (the protocol of test_step_from_developed_state: a cell the
    # donor cap has just drained holds rounding noise around zero, which one side floors and the other keeps;
    # run in lockstep, that noise would become the whole stencil of the cells ahead of the front)
    dev, _ = s.download(); dev["nH"] = w.state.nH
    o.step(w.dt, 1); s.step(w.dt, 1)
    got, lg = s.download()
    o1 = oracle_mod.Oracle(w.mesh, w.params); o1.set_sources(w.sources); o1.set_state(P.as_state(dev)); o1.set_active(active)
    o1.step(w.dt, 1)
    e = P.step_errors(w.mesh, w.params.ctilde, dev, o1.get_state(), got)
    assert e["N"] <= P.TOL_STEP and e["F"] <= P.TOL_STEP, e
    assert max(e["xHII"], e["xHeII"], e["xHeIII"]) <= 1e-9 and e["eth"] <= 1e-8, e
    assert P.ledger_errors(o.ledger(), lg) <= 1e-11
    stored0 = (w.state.N * w.mesh.volume).sum(1)
    assert P.budget_residual(lg, stored0).max() <= P.TOL_LEDGER
    far = _untouched(w.mesh, active)
    assert far.sum() > 0.05 * C
    for k in ("N", "F", "xHII", "xHeII", "xHeIII", "eth"):
        assert np.array_equal(got[k][..., far], start[k][..., far]), k
    # back to every cell: the next subcycle is again the plain one
    s.set_active(None)
    dev, _ = s.download(); dev["nH"] = w.state.nH
    s.step(w.dt, 1)
    got, _ = s.download()
    o1 = oracle_mod.Oracle(w.mesh, w.params); o1.set_sources(w.sources); o1.set_state(P.as_state(dev))
    o1.step(w.dt, 1)
    e = P.step_errors(w.mesh, w.params.ctilde, dev, o1.get_state(), got)
    assert e["N"] <= P.TOL_STEP and e["F"] <= P.TOL_STEP, e


def test_all_active_mask_is_bit_identical_and_device_masks_work():
    import torch
    from paper_2404_17630_b200 import rt
    w = cfg.get(2, 8)
    a = rt.Solver(w.mesh, w.params); a.init(w.state, w.sources); a.step(w.dt, 4)
    b = rt.Solver(w.mesh, w.params); b.init(w.state, w.sources)
    b.set_active(torch.ones(w.mesh.ncell, dtype=torch.bool, device="cuda")); b.step(w.dt, 4)
    sa, la = a.download(); sb, lb = b.download()
    for k in sa:
        assert np.array_equal(sa[k], sb[k]), k
    assert np.array_equal(la["injected"], lb["injected"]) and np.array_equal(la["absorbed"], lb["absorbed"])
    mask = np.arange(w.mesh.ncell) % 3 == 0
    c = rt.Solver(w.mesh, w.params); c.init(w.state, w.sources); c.set_active(mask); c.step(w.dt, 2)
    d = rt.Solver(w.mesh, w.params); d.init(w.state, w.sources); d.set_active(torch.as_tensor(mask).cuda()); d.step(w.dt, 2)
    sc, _ = c.download(); sd, _ = d.download()
    for k in sc:
        assert np.array_equal(sc[k], sd[k]), k


def test_power_of_two_schedule_matches_the_oracle(oracle_mod):
    """Three levels of a power-of-two hierarchy (inputs.configs.active_at): level-l cells are active every
    2^(lmax - l) fine steps; two full cycles on both sides."""
    w = cfg.get(3, 10)
    lmax = 2
    level = cfg.levels_by_density(w.state.nH, lmax)
    o, s = _pair(oracle_mod, w)
    prev = o.get_state()
    for k in range(2 * (1 << lmax)):
        act = cfg.active_at(level, k, lmax)
        o.set_active(act); s.set_active(act)
        prev = o.get_state()
        o.step(w.dt, 1); s.step(w.dt, 1)
    got, lg = s.download()
    e = P.step_errors(w.mesh, w.params.ctilde, prev, o.get_state(), got)
    assert e["N"] <= P.TOL_STEP and e["F"] <= P.TOL_STEP, e
    assert max(e["xHII"], e["xHeII"], e["xHeIII"]) <= 1e-9
    lo = o.ledger()
    assert P.ledger_errors(lo, lg) <= 1e-11 and lg["substeps_total"] == lo["substeps_total"]
    stored0 = (w.state.N * w.mesh.volume).sum(1)
    assert P.budget_residual(lg, stored0).max() <= P.TOL_LEDGER
