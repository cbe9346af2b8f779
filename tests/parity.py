"""Helpers shared by the GPU parity tests: run the oracle and the CUDA path on the same inputs."""
import numpy as np

from paper_2404_17630_b200.inputs import configs as cfg

TOL_STEP = 1e-10      # north_star: max relative error per step on N and F
TOL_X = 1e-6          # north_star: absolute error on ionised fractions after 100 subcycles
TOL_LEDGER = 1e-12    # north_star: photon budget, relative


def stencil_max(mesh, a):
    """max of |a| over each cell and its face neighbours (a: (C,))."""
    m = np.abs(a).copy()
    ok = mesh.right >= 0
    l, r = mesh.left[ok], mesh.right[ok]
    np.maximum.at(m, l, np.abs(a)[r])
    np.maximum.at(m, r, np.abs(a)[l])
    return m


def dependence_max(mesh, a, rings=1):
    """max of |a| over `rings` rings of face neighbours."""
    m = np.abs(a)
    for _ in range(rings):
        m = stencil_max(mesh, m)
    return m


def step_errors(mesh, ct, ref_prev, ref, got, rings=1):
    """Normalised errors of N and F (north_star metric): |dN_i| / max over i's
    stencil (the cell and its face neighbours) of N^n and of the result; F likewise, scaled by c~.
    tests/test_oracle_conditioning.py checks that the oracle itself is conditioned to ~1e-15 in
    this metric, so 1e-10 is a meaningful bar."""
    errs = {}
    G = ref["N"].shape[0]
    eN = eF = 0.0
    for g in range(G):
        scale = np.maximum(dependence_max(mesh, ref_prev["N"][g], rings), np.abs(ref["N"][g]))
        # cells whose whole stencil lies > 100 decades below the peak are compared on the peak's
        # scale: there |F|^2 is subnormal and both sides lose digits (parity metric)
        scale = np.maximum(scale, max(1e-100 * np.abs(ref["N"][g]).max(), 1e-300))
        eN = max(eN, np.max(np.abs(got["N"][g] - ref["N"][g]) / scale))
        eF = max(eF, np.max(np.abs(got["F"][g] - ref["F"][g]) / (ct * scale[None, :])))
    errs["N"], errs["F"] = eN, eF
    for k in ("xHII", "xHeII", "xHeIII"):
        errs[k] = float(np.max(np.abs(got[k] - ref[k])))
    errs["eth"] = float(np.max(np.abs(got["eth"] - ref["eth"]) / np.maximum(np.abs(ref["eth"]), 1e-300)))
    return errs


def as_state(d):
    return cfg.State(d["N"], d["F"], d["xHII"], d["xHeII"], d["xHeIII"], d["eth"], d["nH"])


def budget_residual(led, stored0):
    lhs = led["stored"] + led["absorbed"] + led["outflow"]
    rhs = stored0 + led["injected"] + led["inflow_bc"] + led["floor_added"]
    return np.abs(lhs - rhs) / np.maximum(np.abs(rhs), 1e-300)


def ledger_errors(lo, lg):
    """Relative to the budget scale (stored + injected + inflow) of each group."""
    scale = np.abs(lo["stored"]) + np.abs(lo["injected"]) + np.abs(lo["inflow_bc"]) + np.abs(lo["absorbed"]) + 1e-300
    return max(float(np.max(np.abs(lo[k] - lg[k]) / scale)) for k in
               ("stored", "injected", "absorbed", "outflow", "inflow_bc", "floor_added"))
