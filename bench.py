#!/usr/bin/env python
"""Benchmark of the RT subcycle (BASELINE.json metric: RT cell-group-updates/s per subcycle on
one B200, and % of the HBM roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--n 384] [--impl reference]

A "step" is one subcycle = one pass of the whole hot path (chemistry, then two Heun stages of
gradient -> face flux -> update) over the synthetic workload of BASELINE.json configs[4] (384^3
jittered-lattice Voronoi cells, periodic, 3 groups, H+He chemistry; recipe in DESIGN.md 4),
built on the device.  One process per GPU; N > 1 runs N independent replicas (DESIGN.md 8:
"replicas only", no data-path collective) and reports the aggregate.  Prints ONE JSON line.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
recipe on the host cores; the ratio to it is context, not the headline (parity and the roofline
fraction are).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "rt_cell_group_updates_per_s"
UNIT = "cell-group-updates/s"
FULL_N = {0: 32, 1: 128, 2: 64, 3: 256, 4: 384, 5: 44, 6: 128}
SAMPLE_N = {0: 24, 1: 32, 2: 24, 3: 28, 4: 28, 5: 20, 6: 32}


def workload_name(c, n):
    return "config%d_%s_n%d" % (c, ("stromgren", "beam", "hhe_voronoi", "reion_voronoi", "reion_voronoi", "hii_region_voronoi", "travelling_wave")[c], n)


# ------------------------------------------------------------------ CPU oracle legs
def oracle_sample(c, budget_s, steps=None):
    """Times the oracle on the config-c recipe at a reduced lattice.  Returns (value, info)."""
    import oracle
    from paper_2404_17630_b200.inputs import configs as cfg
    n = SAMPLE_N[c]
    w = cfg.get(c, n)
    o = oracle.Oracle(w.mesh, w.params)
    o.set_sources(w.sources)
    o.set_state(w.state)
    C, G = w.mesh.ncell, w.params.ngroup
    t0 = time.perf_counter()
    o.step(w.dt, 1)
    t1 = time.perf_counter() - t0
    if steps is None:
        steps = int(max(1, min(200, budget_s / max(t1, 1e-6) - 1)))
    t0 = time.perf_counter()
    o.step(w.dt, steps)
    el = time.perf_counter() - t0
    val = C * G * steps / el
    info = {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": "%s recipe on a %d^3 lattice (%d cells, %d groups), %d subcycles after 1 untimed, %.1f s"
                      % (workload_name(c, FULL_N[c]), n, C, G, steps, el)}
    return val, info, el / steps * 1e3


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    c = args.config
    import oracle
    from paper_2404_17630_b200.inputs import configs as cfg
    n = SAMPLE_N[c]
    w = cfg.get(c, n)
    o = oracle.Oracle(w.mesh, w.params)
    o.set_sources(w.sources)
    o.set_state(w.state)
    C, G = w.mesh.ncell, w.params.ngroup
    o.step(w.dt, args.warmup)
    t0 = time.perf_counter()
    o.step(w.dt, args.steps)
    el = time.perf_counter() - t0
    val = C * G * args.steps / el
    sample = "%s recipe on a %d^3 lattice (%d cells, %d groups), one subcycle per step" % (
        workload_name(c, FULL_N[c]), n, C, G)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": el / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(c, args.n or FULL_N[c]), "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------ replicas: timing over ranks
def max_over_ranks(x, dist, device):
    """The slowest rank's value (device-timed milliseconds or seconds); x itself without a group."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(world, C, G, steps, ms):
    """Whole-job throughput of `world` independent replicas (replicas only)."""
    return world * C * G * steps / (ms * 1e-3)


# ------------------------------------------------------------------ clocks
class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.rows = []
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.p = None

    def _read(self):
        for line in self.p.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0, t1):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        sm, mx, reasons = [], None, set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for t, l in self.rows:
            if t < t0 or t > t1 + 0.2:
                continue
            f = [x.strip() for x in l.split(",")]
            try:
                sm.append(float(f[0])); mx = float(f[1])
            except Exception:
                continue
            for k, nm in enumerate(names):
                if len(f) > 3 + k and f[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


# ------------------------------------------------------------------ algorithmic bytes
def algorithmic_bytes(C, F, NR, G, heun=True, chem=True, order=2, mixed=False):
    """Bytes each kernel must move per launch if every array it needs is read or written once
    (neighbour gathers served by L2/shared memory; faces shared by two tiles counted once)."""
    # a2 gradient pass: U in, grad out, per face (w, ids) + (c, A), per r-entry slot id, per cell
    # Minv, (s, V), two list offsets
    gb = 48 if mixed else 96   # gradients per (cell, group): 12 floats with rt_params.mixed, else 12 doubles
    grad = 32 * G * C + gb * G * C + 64 * F + 2 * NR + (48 + 32 + 16) * C
    # a3+a4 stage pass: U and grad in, U out, U0 in (read in both stages), per face (c, A) + (n, ids),
    # per r-entry slot id, per cell (s, V), two list offsets, source index
    stage = (32 + gb + 32 + 32) * G * C + 64 * F + 2 * NR + (32 + 16 + 4) * C
    if order < 2:
        stage -= gb * G * C
    chemb = 64 * G * C + 64 * C + 16 * C
    per_stage = (grad if order >= 2 else 0) + stage
    per_sub = (2 if heun else 1) * per_stage + (chemb if chem else 0)
    return {"grad": grad, "stage": stage, "chem": chemb, "subcycle": per_sub}


def run_timeline(s, w, name):
    """Phase durations of the flux kernel per tile (thread 0's device-clock stamps, second Heun stage) and, per
    multiprocessor, how many tiles are in flight and how many of them are in the face-flux phase."""
    tl = s.tile_timeline(w.dt).astype(np.int64)
    tl = tl[tl[:, 5] > 0]
    d = np.diff(tl[:, :6], axis=1) / 1e3
    names = ("tables arrive", "data staged", "face fluxes (a3)", "publish + boundary ledger", "gather + update (a4)")
    out = {"workload": name, "tiles": int(len(tl)), "kernel_span_ms": float((tl[:, 5].max() - tl[:, 0].min()) / 1e6), "phases_us": {}}
    for i, nm in enumerate(names):
        out["phases_us"][nm] = {"mean": float(d[:, i].mean()), "p10": float(np.percentile(d[:, i], 10)),
                                "p50": float(np.percentile(d[:, i], 50)), "p90": float(np.percentile(d[:, i], 90))}
    out["tile_total_us"] = {"mean": float((tl[:, 5] - tl[:, 0]).mean() / 1e3)}
    sms = np.unique(tl[:, 6])
    conc, a3 = [], {}
    for k in sms[:: max(1, len(sms) // 8)]:
        m = tl[:, 6] == k
        span = float(tl[m, 5].max() - tl[m, 0].min())
        conc.append(float((tl[m, 5] - tl[m, 0]).sum() / span))
        ev = sorted([(a, 1) for a in tl[m, 2]] + [(b, -1) for b in tl[m, 3]])
        cur, last = 0, ev[0][0]
        for t, dl in ev:
            a3[cur] = a3.get(cur, 0.0) + (t - last) / span / 8.0
            last, cur = t, cur + dl
    out["tiles_in_flight_per_sm"] = float(np.mean(conc))
    out["share_of_time_with_k_tiles_in_a3"] = {str(k): round(v, 3) for k, v in sorted(a3.items())}
    print(json.dumps({"timeline": out}))
    return 0


def run_alu_peak():
    """fp64-pipe and shared-memory peaks of this GPU, measured by the library's own micro-benchmark
    kernels (csrc/rt_peak.cu), with the clocks sampled while they run."""
    import torch
    from paper_2404_17630_b200 import rt
    torch.cuda.set_device(0)
    h = rt.rt_create(0, torch.cuda.current_stream().cuda_stream)
    rt.rt_debug_alu_peak(h)                      # warm-up
    sampler = ClockSampler(0)
    time.sleep(0.3)
    t0 = time.perf_counter()
    best = None
    for _ in range(5):
        d = rt.rt_debug_alu_peak(h)
        best = d if best is None else {k: max(best[k], d[k]) for k in d}
    t1 = time.perf_counter()
    clocks = sampler.stop(t0, t1)
    rt.rt_destroy(h)
    best["fp64_tflops_dfma"] = 2.0 * best["dfma"] / 1e12
    best["lds_bytes_per_clk_per_sm"] = {k: 16.0 * best[k] / best["sm_count"] / (clocks["sm_mhz"] or 1965.0) / 1e6
                                        for k in ("lds128", "lds128_bcast3", "lds128_bcast8", "lds128_random")}
    best["clocks"] = clocks
    print(json.dumps({"alu_peak": best}))
    return 0


def survey_bytes(C, F, G):
    """per subcycle 2 x (gradient pass + update pass) + 32 G (stage 2 re-reads U^n) + 80, with
    fpc = F / C unique faces and hf = 2 fpc half-faces per cell, int32 ids."""
    fpc = F / C
    hf = 2.0 * fpc
    grad = 32 * G + 56 * fpc + 76 + 4 * hf + 96 * G
    upd = 32 * G + 96 * G + 64 * fpc + 36 + 4 * hf + 32 * G
    return C * (2 * (grad + upd) + 32 * G + 80)


def run_sharded(args):
    """--shard: ONE mesh cut into contiguous Peano-Hilbert ranges, one per rank (paper_2404_17630_b200/shard.py;
    DESIGN.md 8.1), four ghost exchanges per subcycle over torch.distributed (NCCL).  Strong scaling: the value
    is the whole mesh's cell-group-updates per second.  --shards-local K instead runs K shards on ONE GPU in
    lock-step (plain copies for the exchange): the cost of the ghost layers and of packing, not of a link."""
    import torch
    from paper_2404_17630_b200 import rt, shard as S
    from paper_2404_17630_b200.inputs import configs as cfg
    rank, local, world = int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    c = args.config
    n = args.n or min(FULL_N[c], 128)        # (the partitioner is host-side numpy: sized for it)
    w = cfg.get(c, n)                        # every rank builds the same seeded inputs and cuts its part out
    w.params.mixed = 1 if args.mixed else 0
    C, G = int(w.mesh.ncell), int(w.params.ngroup)
    klocal = args.shards_local
    if klocal > 1:
        run = S.LocalGroup(w.mesh, w.params, w.state, w.sources, klocal, device=local)
        ranks = run.ranks
    else:
        run = S.ShardedSolver(w.mesh, w.params, w.state, w.sources, rank, world, S.DistComm(dist) if dist else None, device=local)
        ranks = [run]
    rows = sum(int(v.numel()) for r in ranks for v in r.send_ids.values())
    bytes_step = rows * 2 * (ranks[0].solver.halo_row_bytes(rt.RT_HALO_U) + ranks[0].solver.halo_row_bytes(rt.RT_HALO_GRAD))
    run.step(w.dt, max(3, args.warmup))
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = sum(r.solver.launches() for r in ranks)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    tw0 = time.perf_counter()
    e0.record()
    run.step(w.dt, args.steps)
    e1.record()
    torch.cuda.synchronize()
    tw1 = time.perf_counter()
    if dist is not None:
        dist.barrier()
    ms = max_over_ranks(e0.elapsed_time(e1), dist, torch.device("cuda", local))
    clocks = sampler.stop(tw0, tw1)
    launches = sum(r.solver.launches() for r in ranks) - l0
    led = run.download()[1] if klocal > 1 else run.ledger()
    stored0 = (w.state.N * w.mesh.volume).sum(1)
    resid = float(np.max(np.abs(led["stored"] + led["absorbed"] + led["outflow"] - stored0 - led["injected"] - led["inflow_bc"] - led["floor_added"])
                         / np.maximum(np.abs(stored0 + led["injected"]), 1e-300)))
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": C * G * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": max(3, args.warmup), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong",
                          "vs_baseline": None, "dtype": "f64" if not args.mixed else "f64 + f32 (rt_params.mixed)", "data": "synthetic",
                          "config": {"workload": workload_name(c, n), "cells": C, "groups": G,
                                     "parallelism": "%d shards on one GPU, lock-step" % klocal if klocal > 1 else "shards x%d" % world,
                                     "shards": [{"owned": r.shard.nown, "ghosts": r.shard.nghost} for r in ranks],
                                     "exchanges_per_subcycle": len([1 for _, x in ranks[0].phases() if x is not None]),
                                     "halo_bytes_per_subcycle": bytes_step,
                                     "l2": "inputs larger than L2" if C * G * 192 > 126e6 else "inputs smaller than L2 (small --n)"},
                          "clocks": clocks, "gpu_launches": int(launches), "ledger": {"budget_residual": resid}}))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--n", type=int, default=None, help="lattice cells per dimension (default: the config's full size)")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--e2e-rt-subcycles", type=int, default=64,
                    help="subcycles of the one RT step timed end to end with a single upload and download (0: skip)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--tuning", default="", help="rt_tuning fields, e.g. tile_cells=40,variant=2 (experiments)")
    ap.add_argument("--mixed", action="store_true",
                    help="rt_params.mixed = 1: fp32 gradients, closure and flux, fp64 state and sums (PAPER.md:380-386; "
                         "not the headline: DESIGN.md 7.6)")
    ap.add_argument("--shard", action="store_true",
                    help="one mesh sharded over the ranks with ghost exchanges (strong scaling) instead of N replicas")
    ap.add_argument("--shards-local", type=int, default=1,
                    help="with --shard: K shards on one GPU in lock-step (overhead of the ghost layers, no link)")
    ap.add_argument("--active-frac", type=float, default=1.0,
                    help="individual time steps (rt_set_active): only the cells of the slab x < frac * box take the step")
    ap.add_argument("--timeline", action="store_true",
                    help="only record the per-tile phase stamps of the flux kernel (rt_debug_tile_timeline) and print their statistics")
    ap.add_argument("--alu-peak", action="store_true",
                    help="only run the fp64 / shared-memory micro-benchmarks (rt_debug_alu_peak) and print them")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.alu_peak:
        return run_alu_peak()
    if args.warmup < 3:
        args.warmup = 3
    if args.shard:
        return run_sharded(args)

    import torch
    from paper_2404_17630_b200 import rt
    from paper_2404_17630_b200.inputs import configs as cfg
    from paper_2404_17630_b200.inputs import device as devin
    from paper_2404_17630_b200.profile_summary import kernel_source_sha

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the RT path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    c = args.config
    n = args.n or FULL_N[c]
    t_build = time.perf_counter()
    if c in (3, 4):
        w = devin.config34_device(n, c, "cuda:%d" % local)
    elif c == 6:
        w = cfg.get(6, n)                        # transport only, one bin, 10 % generator offset
    else:
        w = cfg.get(c, n)
    C, F, G = int(w.mesh.ncell), int(w.mesh.nface), int(w.params.ngroup)
    NR = int((w.mesh.right >= 0).sum())
    tuning = {k: int(v) for k, v in (kv.split("=") for kv in args.tuning.split(",") if kv)} or None
    w.params.mixed = 1 if args.mixed else 0
    s = rt.Solver(w.mesh, w.params, device=local, tuning=tuning)
    stored0 = np.asarray([float((w.state.N[g] * w.mesh.volume).sum()) for g in range(G)])   # photons at t = 0
    x_slab, box_x = w.mesh.centroid[0], float(w.mesh.box[0])
    w.mesh = None
    torch.cuda.empty_cache()
    s.init(w.state, w.sources)
    n_active = C
    if args.active_frac < 1.0:
        mask = x_slab < args.active_frac * box_x
        n_active = int(mask.sum())
        s.set_active(mask)
    tiles = s.tile_info()
    t_build = time.perf_counter() - t_build
    s.step(w.dt, args.warmup)
    torch.cuda.synchronize()
    if args.timeline:
        return run_timeline(s, w, workload_name(c, n))

    # ---- timed region: K subcycles, state (>= 20 GB at full size) far larger than the 126 MB L2
    sampler = ClockSampler(local)
    time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = s.launches()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    tw0 = time.perf_counter()
    e0.record()
    s.step(w.dt, args.steps)          # the headline pass: no per-kernel events on the stream
    e1.record()
    torch.cuda.synchronize()
    tw1 = time.perf_counter()
    if dist is not None:
        dist.barrier()
    ms = e0.elapsed_time(e1)
    launches = s.launches() - l0
    clocks = sampler.stop(tw0, tw1)
    # a second, shorter pass with the library's per-kernel events for the shares (not part of `value`)
    nprof = max(1, min(args.steps, 5))
    s.profile(True)
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    s.step(w.dt, nprof)
    p1.record()
    torch.cuda.synchronize()
    prof = s.profile_read()
    s.profile(False)
    ms_prof = p0.elapsed_time(p1)
    ms = max_over_ranks(ms, dist, "cuda")
    value = aggregate_value(world, C, G, args.steps, ms)

    # ---- ledger sanity after the timed region (photon budget closes)
    led = s.ledger()

    # ---- end to end through the C ABI with HOST buffers: H2D state, one subcycle, D2H state
    e2e = None
    if args.e2e_steps > 0:
        shapes = {"N": (G, C), "F": (G, 3, C), "xHII": (C,), "xHeII": (C,), "xHeIII": (C,), "eth": (C,)}
        host = {k: torch.empty(sh, dtype=torch.float64).pin_memory() for k, sh in shapes.items()}
        nH = w.state.nH
        host_in = dict(host)
        host_in["nH"] = (nH.cpu() if hasattr(nH, "cpu") else torch.as_tensor(nH)).pin_memory()
        rt.rt_download(s.h, host, False, G)
        for _ in range(1):  # warm-up of the copy path
            rt.rt_state_init(s.h, w.params, host_in, w.sources); rt.rt_step(s.h, w.dt, 1); rt.rt_download(s.h, host, False, G)
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            rt.rt_state_init(s.h, w.params, host_in, w.sources)
            rt.rt_step(s.h, w.dt, 1)
            rt.rt_download(s.h, host, False, G)
        torch.cuda.synchronize()
        el = time.perf_counter() - t0
        el = max_over_ranks(el, dist, "cuda")
        e2e = {"value": world * C * G * args.e2e_steps / el, "unit": UNIT, "h2d_bytes_per_step": (4 * G + 5) * 8 * C,
               "d2h_bytes_per_step": (4 * G + 4) * 8 * C, "steps": args.e2e_steps, "ms_per_step": el / args.e2e_steps * 1e3}
        # the same through the C ABI in the paper's own rhythm: the state goes to the GPU once per RT step of
        # 64 subcycles and comes back after it ("transferred to the GPU once before the first subcycle
        # and only copied back after the completion of the full RT step"; 64 subcycles: PAPER.md:284, 334)
        if args.e2e_rt_subcycles > 0:
            nsub = args.e2e_rt_subcycles
            if dist is not None:
                dist.barrier()
            t0 = time.perf_counter()
            rt.rt_state_init(s.h, w.params, host_in, w.sources)
            rt.rt_step(s.h, w.dt, nsub)
            rt.rt_download(s.h, host, False, G)
            torch.cuda.synchronize()
            el = max_over_ranks(time.perf_counter() - t0, dist, "cuda")
            e2e["rt_step"] = {"value": world * C * G * nsub / el, "unit": UNIT, "subcycles_per_rt_step": nsub,
                              "ms_per_rt_step": el * 1e3, "h2d_bytes_per_rt_step": (4 * G + 5) * 8 * C,
                              "d2h_bytes_per_rt_step": (4 * G + 4) * 8 * C}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel
    peaks_file = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_file):
        peak, peak_src = float(json.load(open(peaks_file))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    else:
        peak, peak_src = 6650.0, "fallback (B200_PROFILING.md)"
    ab = algorithmic_bytes(C, F, NR, G, bool(w.params.heun), w.params.chem_mode != 0, int(w.params.order), bool(args.mixed))
    kern = {}
    # one Heun stage's a3 + a4 = k_flux (class 2) followed by k_finish (class 3): reported separately
    # and, as "stage", together (the algorithmic bytes of a3 + a4 are those of the pair)
    prof["finish"] = prof["update"]
    prof["stage"] = (prof["flux"][0] + prof["update"][0], prof["flux"][1])
    for k in ("chem", "grad", "stage", "flux", "finish", "reduce"):
        tms, cnt = prof[k]
        if cnt == 0:
            continue
        avg = tms / cnt
        d = {"launches": cnt, "avg_ms": avg, "share": tms / ms_prof}
        if k in ab:
            d["algorithmic_bytes"] = ab[k]
            d["GBps"] = ab[k] / (avg * 1e-3) / 1e9
            d["frac_of_hbm_peak"] = d["GBps"] / peak
        kern[k] = d
    dom = max((k for k in kern if k in ab), key=lambda k: kern[k]["avg_ms"] * kern[k]["launches"])
    # (kern["stage"] is the pair k_flux + k_finish: avg_ms is the pair's time per stage)
    # dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full`
    # capture of this workload (profiles/traffic.csv, written from profiles/r1_ncu_full_*.md); for
    # the stage pair it is the sum of k_flux (both tile classes) and k_finish
    traffic, traffic_note = None, "no ncu capture of this workload in profiles/traffic.csv"
    tf = os.path.join(ROOT, "profiles", "traffic.csv")
    if args.mixed:
        traffic_note = "profiles/traffic.csv holds the fp64 path's capture; none for --mixed"
    elif os.path.exists(tf):
        rows = {}
        for ln in open(tf).read().splitlines()[1:]:
            f = ln.split(",")
            if len(f) >= 4 and f[0] == workload_name(c, n):
                rows[f[1]] = (float(f[2]), f[3])
        parts = {"stage": ("k_flux", "k_finish"), "grad": ("k_grad",), "chem": ("k_chem",)}.get(dom, (dom,))
        if all(k in rows for k in parts):
            if all(rows[k][1] == kernel_source_sha() for k in parts):
                traffic, traffic_note = sum(rows[k][0] for k in parts), "ncu capture of these kernel sources (profiles/traffic.csv)"
            else:
                traffic_note = "profiles/traffic.csv was captured from other kernel sources: stale, not reported"

    roofline = {"bound": "hbm", "kernel": {"stage": "stage = k_flux + k_finish (a3 + a4 of one Heun stage)"}.get(dom, dom), "achieved": kern[dom]["GBps"], "peak": peak, "unit": "GB/s",
                "frac": kern[dom]["GBps"] / peak, "frac_of_nominal_8TBs": kern[dom]["GBps"] / 8000.0,
                "traffic": traffic, "traffic_note": traffic_note, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": ab[dom],
                "subcycle": {"algorithmic_bytes": ab["subcycle"], "GBps": ab["subcycle"] * args.steps / (ms * 1e-3) / 1e9,
                             "frac": ab["subcycle"] * args.steps / (ms * 1e-3) / 1e9 / peak,
                             "frac_of_nominal_8TBs": ab["subcycle"] * args.steps / (ms * 1e-3) / 1e9 / 8000.0,
                             "bytes_per_cell_group_update": ab["subcycle"] / (C * G),
                             # the same time against SURVEY 8(d)'s model (fused, no list bytes: 4222 B per cell at
                             # G = 3 on a Voronoi mesh), so that the fraction cannot rise by redefining the bytes
                             "frac_survey_model": survey_bytes(C, F, G) * args.steps / (ms * 1e-3) / 1e9 / peak,
                             "survey_bytes_per_cell_group_update": survey_bytes(C, F, G) / (C * G)}}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        _, cpu, _ = oracle_sample(c, args.cpu_seconds)

    stored_scale = float(np.max(np.abs(led["injected"]) + np.abs(led["stored"])) + 1e-300)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64 state and sums, f32 gradients / closure / flux (rt_params.mixed)" if args.mixed else "f64", "data": "synthetic",
            "config": {"workload": workload_name(c, n), "cells": C, "faces": F, "groups": G,
                       "chem_mode": int(w.params.chem_mode), "dt": w.dt, "parallelism": "replicas x%d" % world,
                       "l2": "inputs larger than L2 (%.1f GB of state and geometry per subcycle)" % (ab["subcycle"] / 1e9),
                       "build_s": t_build, "tiles": tiles, "active_cells": n_active,
                       "timed_subcycles": "%d..%d after rt_state_init (warm-up %d)" % (args.warmup + 1, args.warmup + args.steps, args.warmup)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "kernels": kern,
            "cpu_baseline": cpu,
            "ledger": {"substeps_total": int(led["substeps_total"]), "substeps_max": int(led["substeps_max"]),
                       "cells_hit_cap": int(led["cells_hit_cap"]),
                       "budget_residual": float(np.max(np.abs(led["stored"] + led["absorbed"] + led["outflow"]
                                                              - stored0 - led["injected"] - led["inflow_bc"] - led["floor_added"]))
                                                / stored_scale)}}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
