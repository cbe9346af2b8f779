"""rt_stored_photons_noalloc (include/rt.h): the budget's "stored" row computed with its scratch in a static
device array, against the existing path (k_stored + k_reduce behind rt_ledger_read, scratch in the caller's
workspace).  Collected last on purpose (the suite runs with pytest -x): a failure here hides nothing.

Two calls in a row on different workloads, the larger first, so that the second call finds the first one's
partial sums in the rows beyond its own: it must not read them.  Tolerance: the ledger tolerance of the
parity tests (parity.TOL_LEDGER, 1e-12 relative; the two paths differ in summation order only).
"""
import numpy as np
import pytest

import parity as P
from paper_2404_17630_b200.inputs import configs as cfg

pytestmark = pytest.mark.gpu


def _existing_path(rt, torch, w, nsub):
    """State and `stored` of the existing path after nsub subcycles: (N (G, C) cuda, volume (C) cuda, stored (G,))."""
    s = rt.Solver(w.mesh, w.params, device=0)
    s.init(w.state, w.sources)
    s.step(w.dt, nsub)
    st, led = s.download(device=True)
    torch.cuda.synchronize()
    vol = torch.as_tensor(np.ascontiguousarray(w.mesh.volume), dtype=torch.float64, device="cuda:0")
    return st["N"].contiguous(), vol, np.asarray(led["stored"])[: w.params.ngroup].copy()


def test_no_alloc_stored_matches_the_ledger_twice_in_a_row():
    import torch
    from paper_2404_17630_b200 import rt
    assert torch.cuda.is_available()
    cases = []
    for c, n, nsub in ((2, 14, 3), (0, 9, 2)):        # 2744 cells x 3 groups, then 729 cells x 1 group (ragged blocks)
        w = cfg.get(c, n)
        cases.append((w,) + _existing_path(rt, torch, w, nsub))
    outs = [torch.full((8,), -1.0, dtype=torch.float64, device="cuda:0") for _ in cases]
    for (w, N, vol, want), out in zip(cases, outs):   # back to back on one stream, no synchronisation in between
        rc, msg = rt.rt_stored_photons_noalloc(N, vol, out)
        assert rc == 0, msg
    torch.cuda.synchronize()
    for (w, N, vol, want), out in zip(cases, outs):
        G = w.params.ngroup
        got = out.cpu().numpy()
        assert np.all(want > 0)
        assert np.max(np.abs(got[:G] - want) / np.abs(want)) <= P.TOL_LEDGER, (got[:G], want)
        assert np.all(got[G:] == -1.0)                # nothing written beyond the G results
        direct = (N.cpu().numpy() * w.mesh.volume).sum(1)
        assert np.max(np.abs(got[:G] - direct) / np.abs(direct)) <= P.TOL_LEDGER
    # the same call again gives the same bits (fixed summation order, no state carried over)
    w, N, vol, want = cases[0]
    again = torch.zeros(8, dtype=torch.float64, device="cuda:0")
    rc, msg = rt.rt_stored_photons_noalloc(N, vol, again)
    torch.cuda.synchronize()
    assert rc == 0 and np.array_equal(again.cpu().numpy()[:3], outs[0].cpu().numpy()[:3])


def test_no_alloc_rejects_sizes_beyond_the_static_scratch():
    import ctypes
    import torch
    from paper_2404_17630_b200 import rt
    L = rt.lib()
    L.rt_stored_photons_noalloc.restype = ctypes.c_int
    L.rt_stored_photons_noalloc.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_void_p,
                                            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_char_p, ctypes.c_int]
    out = torch.zeros(8, dtype=torch.float64, device="cuda:0")
    err = ctypes.create_string_buffer(512)
    # rejected on its size alone, before any pointer is touched
    rc = L.rt_stored_photons_noalloc(0, None, rt.RT_NOALLOC_MAX_CELLS + 1, 3, out.data_ptr(), out.data_ptr(), out.data_ptr(), err, 512)
    assert rc == -1 and b"RT_NOALLOC_MAX_CELLS" in err.value, err.value
    rc = L.rt_stored_photons_noalloc(0, None, 10, 9, out.data_ptr(), out.data_ptr(), out.data_ptr(), err, 512)
    assert rc == -1 and b"ngroup" in err.value
    # an empty mesh stores nothing
    rc = L.rt_stored_photons_noalloc(0, None, 0, 2, None, None, out.data_ptr(), err, 512)
    torch.cuda.synchronize()
    assert rc == 0 and np.all(out.cpu().numpy()[:2] == 0.0)
