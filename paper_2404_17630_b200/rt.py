"""Thin ctypes binding of librt.so (include/rt.h): argument marshalling only.

The functions carry the ABI's names (rt_create, rt_workspace_bytes, rt_mesh_upload, rt_state_init,
rt_step, rt_download, rt_destroy, rt_last_error); `Solver` strings them together and owns the
torch tensor that backs the device workspace.  torch is used for device memory and streams only.
There is no fallback: a missing or unloadable librt.so raises.
"""
import ctypes
import os

import numpy as np

RT_MAXG = 8
RT_MEM_HOST, RT_MEM_DEVICE = 0, 1
RT_WS_DEVICE_MESH, RT_WS_ALL_FACES_CROSS = 1, 2
LEDGER_ROWS = ("stored", "injected", "absorbed", "outflow", "inflow_bc", "floor_added")
_vp = ctypes.c_void_p


class rt_mesh(ctypes.Structure):
    _fields_ = [("ncell", ctypes.c_int64), ("nface", ctypes.c_int64), ("box", ctypes.c_double * 3),
                ("periodic", ctypes.c_int32 * 3), ("mem_kind", ctypes.c_int32), ("volume", _vp), ("centroid", _vp),
                ("area", _vp), ("normal", _vp), ("fcentroid", _vp), ("left", _vp), ("right", _vp),
                ("nghost", ctypes.c_int32), ("ngroup", ctypes.c_int32), ("ghost_state", _vp)]


class rt_state(ctypes.Structure):
    _fields_ = [("mem_kind", ctypes.c_int32), ("pad", ctypes.c_int32), ("N", _vp), ("F", _vp), ("xHII", _vp),
                ("xHeII", _vp), ("xHeIII", _vp), ("eth", _vp), ("nH", _vp)]


class rt_sources(ctypes.Structure):
    _fields_ = [("nsrc", ctypes.c_int32), ("pad", ctypes.c_int32), ("cell", _vp), ("rate", _vp)]


class rt_params(ctypes.Structure):
    _fields_ = [("ngroup", ctypes.c_int32), ("chem_mode", ctypes.c_int32), ("order", ctypes.c_int32),
                ("heun", ctypes.c_int32), ("ctilde", ctypes.c_double), ("sigma", (ctypes.c_double * 3) * RT_MAXG),
                ("eps_heat", (ctypes.c_double * 3) * RT_MAXG), ("T_fixed", ctypes.c_double),
                ("alphaB_override", ctypes.c_double), ("y_he", ctypes.c_double), ("f_accept", ctypes.c_double),
                ("f_target", ctypes.c_double), ("x_floor_rel", ctypes.c_double), ("n_floor", ctypes.c_double),
                ("max_substeps", ctypes.c_int64), ("kappa_mem_kind", ctypes.c_int32), ("mixed", ctypes.c_int32),
                ("kappa", _vp)]


class rt_tuning(ctypes.Structure):
    _fields_ = [("tile_cells", ctypes.c_int32), ("tile_faces", ctypes.c_int32), ("tile_blocks", ctypes.c_int32),
                ("tile_classes", ctypes.c_int32), ("flux_threads", ctypes.c_int32), ("grad_threads", ctypes.c_int32),
                ("prefetch_tiles", ctypes.c_int32), ("chem_caps", ctypes.c_int32 * 6), ("variant", ctypes.c_int32),
                ("reserved", ctypes.c_int32 * 9)]


class rt_ledger(ctypes.Structure):
    _fields_ = [(k, ctypes.c_double * RT_MAXG) for k in LEDGER_ROWS] + \
               [("substeps_total", ctypes.c_int64), ("substeps_max", ctypes.c_int64), ("cells_hit_cap", ctypes.c_int64),
                ("nsub_done", ctypes.c_int64)]


_lib = None


def lib():
    """Loads librt.so (building it in-tree if the sources are newer).  Raises if that fails."""
    global _lib
    if _lib is None:
        from .build import build_rt
        so = build_rt()
        L = ctypes.CDLL(so)
        L.rt_create.restype = ctypes.c_int
        L.rt_create.argtypes = [ctypes.POINTER(_vp), ctypes.c_int, _vp]
        L.rt_set_tuning.restype = ctypes.c_int
        L.rt_set_tuning.argtypes = [_vp, ctypes.POINTER(rt_tuning)]
        L.rt_workspace_bytes.restype = ctypes.c_size_t
        L.rt_workspace_bytes.argtypes = [ctypes.c_int64, ctypes.c_int64, ctypes.c_int, ctypes.c_int]
        L.rt_mesh_upload.restype = ctypes.c_int
        L.rt_mesh_upload.argtypes = [_vp, ctypes.POINTER(rt_mesh), _vp, ctypes.c_size_t]
        L.rt_state_init.restype = ctypes.c_int
        L.rt_state_init.argtypes = [_vp, ctypes.POINTER(rt_params), ctypes.POINTER(rt_state), ctypes.POINTER(rt_sources)]
        L.rt_set_active.restype = ctypes.c_int
        L.rt_set_active.argtypes = [_vp, ctypes.c_int, _vp]
        L.rt_step.restype = ctypes.c_int
        L.rt_step.argtypes = [_vp, ctypes.c_double, ctypes.c_int]
        L.rt_download.restype = ctypes.c_int
        L.rt_download.argtypes = [_vp, ctypes.POINTER(rt_state), ctypes.POINTER(rt_ledger)]
        L.rt_kernel_launches.restype = ctypes.c_int64
        L.rt_kernel_launches.argtypes = [_vp]
        L.rt_tile_info.restype = ctypes.c_int
        L.rt_tile_info.argtypes = [_vp, _vp]
        L.rt_debug_gradients.restype = ctypes.c_int
        L.rt_debug_gradients.argtypes = [_vp, ctypes.c_int, _vp, _vp]
        L.rt_profile.restype = ctypes.c_int
        L.rt_profile.argtypes = [_vp, ctypes.c_int]
        L.rt_profile_read.restype = ctypes.c_int
        L.rt_profile_read.argtypes = [_vp, _vp, _vp]
        L.rt_debug_tiles.restype = ctypes.c_int
        L.rt_debug_tiles.argtypes = [_vp, ctypes.c_int, _vp, _vp]
        L.rt_debug_tile_timeline.restype = ctypes.c_int
        L.rt_debug_tile_timeline.argtypes = [_vp, ctypes.c_double, ctypes.c_int64, _vp]
        L.rt_debug_alu_peak.restype = ctypes.c_int
        L.rt_debug_alu_peak.argtypes = [_vp, _vp]
        L.rt_last_error.restype = ctypes.c_char_p
        L.rt_last_error.argtypes = [_vp]
        L.rt_destroy.restype = None
        L.rt_destroy.argtypes = [_vp]
        _lib = L
    return _lib


class RTError(RuntimeError):
    pass


def _is_torch(a):
    return hasattr(a, "data_ptr")


def _addr(a):
    if a is None:
        return None
    return a.data_ptr() if _is_torch(a) else a.ctypes.data


def _kind(a):
    return RT_MEM_DEVICE if (_is_torch(a) and a.is_cuda) else RT_MEM_HOST


def _prep(a, dtype):
    """Contiguous array of the ABI's dtype; numpy or torch (host or cuda) pass through."""
    if _is_torch(a):
        import torch
        td = {np.float64: torch.float64, np.int32: torch.int32}[dtype]
        return a.to(td).contiguous()
    return np.ascontiguousarray(a, dtype=dtype)


# ------------------------------------------------------------------ the ABI, name for name
def rt_create(device=0, stream=None):
    h = _vp()
    rc = lib().rt_create(ctypes.byref(h), int(device), _vp(stream) if stream else None)
    if rc != 0:
        raise RTError("rt_create failed with code %d (no usable CUDA device %d?)" % (rc, device))
    return h


def rt_set_tuning(h, **kw):
    """Fields of rt_tuning by name (chem_caps: a sequence); unnamed fields keep the default 0."""
    t = rt_tuning()
    for k, v in kw.items():
        if k == "chem_caps":
            for i, x in enumerate(v):
                t.chem_caps[i] = int(x)
        else:
            setattr(t, k, int(v))
    _check(h, lib().rt_set_tuning(h, ctypes.byref(t)), "rt_set_tuning")


def rt_workspace_bytes(ncell, nface, ngroup, flags=0):
    return int(lib().rt_workspace_bytes(ncell, nface, ngroup, flags))


def rt_last_error(h):
    return lib().rt_last_error(h).decode()


def _check(h, rc, what):
    if rc != 0:
        raise RTError("%s failed (%d): %s" % (what, rc, rt_last_error(h)))


def _on_device(mesh):
    return _kind(mesh.volume) == RT_MEM_DEVICE


def rt_mesh_upload(h, mesh, ngroup, ghost_state, workspace):
    """mesh: object with the attributes of inputs.mesh.Mesh (numpy or torch arrays)."""
    keep = [_prep(getattr(mesh, k), np.float64) for k in ("volume", "centroid", "area", "normal", "fcentroid")]
    keep += [_prep(mesh.left, np.int32), _prep(mesh.right, np.int32)]
    kinds = {_kind(a) for a in keep}
    if len(kinds) != 1:
        raise RTError("mesh arrays must all live on the host or all on the device")
    m = rt_mesh()
    m.ncell, m.nface = int(mesh.ncell), int(mesh.nface)
    m.box[:] = [float(x) for x in mesh.box]
    m.periodic[:] = [int(x) for x in mesh.periodic]
    m.mem_kind = kinds.pop()
    for name, a in zip(("volume", "centroid", "area", "normal", "fcentroid", "left", "right"), keep):
        setattr(m, name, _addr(a))
    gs = None if ghost_state is None else np.ascontiguousarray(ghost_state, dtype=np.float64)
    m.nghost = 0 if gs is None else int(gs.shape[0])
    m.ngroup = int(ngroup)
    m.ghost_state = _addr(gs)
    _check(h, lib().rt_mesh_upload(h, ctypes.byref(m), _vp(workspace.data_ptr()),
                                   workspace.numel() * workspace.element_size()), "rt_mesh_upload")


def make_params(p):
    """inputs.configs.Params (or alike) -> rt_params plus the arrays it borrows."""
    q = rt_params()
    q.ngroup, q.chem_mode, q.order, q.heun = int(p.ngroup), int(p.chem_mode), int(p.order), int(p.heun)
    q.ctilde = float(p.ctilde)
    sg, ep = np.asarray(p.sigma, dtype=np.float64), np.asarray(p.eps_heat, dtype=np.float64)
    for g in range(p.ngroup):
        for j in range(3):
            q.sigma[g][j] = sg[g, j]
            q.eps_heat[g][j] = ep[g, j]
    q.T_fixed, q.alphaB_override, q.y_he = float(p.T_fixed), float(p.alphaB_override), float(p.y_he)
    q.f_accept, q.f_target, q.x_floor_rel = float(p.f_accept), float(p.f_target), float(p.x_floor_rel)
    q.n_floor, q.max_substeps = float(p.n_floor), int(p.max_substeps)
    q.mixed = int(getattr(p, "mixed", 0))
    kp = None
    if p.kappa is not None:
        kp = _prep(p.kappa, np.float64)
        q.kappa_mem_kind = _kind(kp)
        q.kappa = _addr(kp)
    return q, kp


def make_state(s, need_nH=True):
    names = ("N", "F", "xHII", "xHeII", "xHeIII", "eth") + (("nH",) if need_nH else ())
    keep = {k: _prep(s[k] if isinstance(s, dict) else getattr(s, k), np.float64) for k in names}
    kinds = {_kind(a) for a in keep.values()}
    if len(kinds) != 1:
        raise RTError("state arrays must all live on the host or all on the device")
    st = rt_state()
    st.mem_kind = kinds.pop()
    for k, a in keep.items():
        setattr(st, k, _addr(a))
    return st, keep


def rt_state_init(h, params, state, sources=None):
    q, kp = make_params(params)
    st, keep = make_state(state)
    src = None
    if sources is not None and len(sources.cell) > 0:
        cell = np.ascontiguousarray(sources.cell, dtype=np.int32)
        rate = np.ascontiguousarray(sources.rate, dtype=np.float64)
        src = rt_sources(int(cell.size), 0, _addr(cell), _addr(rate))
    _check(h, lib().rt_state_init(h, ctypes.byref(q), ctypes.byref(st), ctypes.byref(src) if src else None),
           "rt_state_init")


def rt_set_active(h, active=None):
    """active: (C,) mask (numpy or torch, host or cuda) of the cells taking part in the next rt_step calls, or None."""
    if active is None:
        _check(h, lib().rt_set_active(h, RT_MEM_HOST, None), "rt_set_active")
        return
    if _is_torch(active):
        import torch
        a = active.to(torch.uint8).contiguous()
    else:
        a = np.ascontiguousarray(active, dtype=np.uint8)
    _check(h, lib().rt_set_active(h, _kind(a), _vp(_addr(a))), "rt_set_active")


def rt_step(h, dt, nsub=1):
    _check(h, lib().rt_step(h, float(dt), int(nsub)), "rt_step")


RT_PHASE_CHEM, RT_PHASE_GRAD1, RT_PHASE_FLUX1, RT_PHASE_GRAD2, RT_PHASE_FLUX2 = range(5)
RT_HALO_U, RT_HALO_GRAD = 0, 1


def rt_step_phase(h, dt, phase):
    L = lib()
    L.rt_step_phase.restype = ctypes.c_int
    L.rt_step_phase.argtypes = [_vp, ctypes.c_double, ctypes.c_int]
    _check(h, L.rt_step_phase(h, float(dt), int(phase)), "rt_step_phase")


def rt_halo_row_bytes(h, what):
    L = lib()
    L.rt_halo_row_bytes.restype = ctypes.c_int
    L.rt_halo_row_bytes.argtypes = [_vp, ctypes.c_int]
    n = L.rt_halo_row_bytes(h, int(what))
    if n <= 0:
        raise RTError("rt_halo_row_bytes: no state yet, or unknown field")
    return n


def _halo(name, h, what, cells, buf):
    """cells: int32 CUDA tensor (local cell numbers); buf: CUDA tensor of len(cells) * rt_halo_row_bytes bytes."""
    if not (_is_torch(cells) and cells.is_cuda and cells.element_size() == 4 and cells.is_contiguous() and
            _is_torch(buf) and buf.is_cuda and buf.is_contiguous()):
        raise RTError(name + " takes contiguous CUDA tensors (int32 cells)")
    n = int(cells.numel())
    if buf.numel() * buf.element_size() < n * rt_halo_row_bytes(h, what):
        raise RTError(name + ": buffer too small")
    L = lib()
    f = getattr(L, name)
    f.restype = ctypes.c_int
    f.argtypes = [_vp, ctypes.c_int, ctypes.c_int64, _vp, _vp]
    _check(h, f(h, int(what), n, _vp(cells.data_ptr()) if n else None, _vp(buf.data_ptr()) if n else None), name)


def rt_halo_pack(h, what, cells, buf):
    _halo("rt_halo_pack", h, what, cells, buf)


def rt_halo_unpack(h, what, cells, buf):
    _halo("rt_halo_unpack", h, what, cells, buf)


def rt_download(h, out=None, want_ledger=True, ngroup=1):
    """out: dict of preallocated arrays (N, F, xHII, xHeII, xHeIII, eth; any subset), or None."""
    st = None
    if out is not None:
        st = rt_state()
        kinds = {_kind(a) for a in out.values()}
        if len(kinds) != 1:
            raise RTError("output arrays must all live on the host or all on the device")
        st.mem_kind = kinds.pop()
        for k, a in out.items():
            setattr(st, k, _addr(a))
    led = rt_ledger() if want_ledger else None
    _check(h, lib().rt_download(h, ctypes.byref(st) if st else None, ctypes.byref(led) if led else None), "rt_download")
    if led is None:
        return None
    d = {k: np.array(getattr(led, k)[:ngroup]) for k in LEDGER_ROWS}
    d.update(substeps_total=led.substeps_total, substeps_max=led.substeps_max, cells_hit_cap=led.cells_hit_cap,
             nsub_done=led.nsub_done)
    return d


def rt_debug_alu_peak(h):
    """Measured operations per second of the fp64 pipe and of shared memory (include/rt.h)."""
    out = np.zeros(14)
    _check(h, lib().rt_debug_alu_peak(h, _vp(out.ctypes.data)), "rt_debug_alu_peak")
    names = ("dfma", "dadd", "dmul", "dmax", "rcp_seed", "rcp_newton2", "rsqrt_seed", "ddiv", "dsqrt", "lds128",
             "lds128_bcast3", "lds128_bcast8", "lds128_random")
    d = {k: float(out[i]) for i, k in enumerate(names)}
    d["sm_count"] = int(out[13])
    return d


RT_NOALLOC_MAX_CELLS = 1 << 24


def rt_stored_photons_noalloc(N, volume, out, stream=None):
    """Sum over cells of V N per group into `out` without any device allocation (include/rt.h): N (G, C),
    volume (C) and out (G) are contiguous float64 CUDA tensors on one device; nothing is copied or converted
    here.  Returns the ABI's return code and message (0, "" on success): the call does not synchronise."""
    for a in (N, volume, out):
        if not (_is_torch(a) and a.is_cuda and a.is_contiguous() and a.element_size() == 8 and a.is_floating_point()):
            raise RTError("rt_stored_photons_noalloc takes contiguous float64 CUDA tensors")
    G, C = int(N.shape[0]), int(N.shape[1])
    if volume.numel() != C or out.numel() < G:
        raise RTError("rt_stored_photons_noalloc: volume must have C and out at least G elements")
    L = lib()
    L.rt_stored_photons_noalloc.restype = ctypes.c_int
    L.rt_stored_photons_noalloc.argtypes = [ctypes.c_int, _vp, ctypes.c_int64, ctypes.c_int, _vp, _vp, _vp, ctypes.c_char_p,
                                            ctypes.c_int]
    err = ctypes.create_string_buffer(512)
    rc = L.rt_stored_photons_noalloc(N.device.index or 0, _vp(stream) if stream else None, C, G, _vp(N.data_ptr()),
                                     _vp(volume.data_ptr()), _vp(out.data_ptr()), err, 512)
    return rc, err.value.decode()


def rt_destroy(h):
    lib().rt_destroy(h)


# ------------------------------------------------------------------ convenience wrapper
class Solver:
    """Owns a context and its workspace tensor.  Every computation happens inside librt.so."""

    def __init__(self, mesh, params, device=0, stream=None, tuning=None):
        import torch
        if not torch.cuda.is_available():
            raise RTError("no CUDA device: the RT path has no CPU fallback")
        lib()
        self.torch = torch
        self.dev = torch.device("cuda", device)
        self.C, self.F, self.G = int(mesh.ncell), int(mesh.nface), int(params.ngroup)
        if stream is None:
            stream = torch.cuda.current_stream(self.dev).cuda_stream
        self.h = rt_create(device, stream)
        flags = RT_WS_DEVICE_MESH if _on_device(mesh) else 0
        if tuning:
            rt_set_tuning(self.h, **tuning)
            if 0 < tuning.get("tile_cells", 0) < 32 or 0 < tuning.get("tile_faces", 0) < 240:
                flags |= RT_WS_ALL_FACES_CROSS
        nbytes = rt_workspace_bytes(self.C, self.F, self.G, flags)
        if nbytes == 0:
            raise RTError("rt_workspace_bytes rejected the sizes")
        self.workspace = torch.empty((nbytes + 7) // 8, dtype=torch.float64, device=self.dev)
        rt_mesh_upload(self.h, mesh, self.G, params.ghost_state, self.workspace)
        self.params = params

    def init(self, state, sources=None, params=None):
        if params is not None:
            self.params = params
        rt_state_init(self.h, self.params, state, sources)

    def set_active(self, active=None):
        rt_set_active(self.h, active)

    def step(self, dt, nsub=1):
        rt_step(self.h, dt, nsub)

    def step_phase(self, dt, phase):
        rt_step_phase(self.h, dt, phase)

    def halo_row_bytes(self, what):
        return rt_halo_row_bytes(self.h, what)

    def halo_pack(self, what, cells, buf):
        rt_halo_pack(self.h, what, cells, buf)

    def halo_unpack(self, what, cells, buf):
        rt_halo_unpack(self.h, what, cells, buf)

    def download(self, device=False):
        """Returns (state dict, ledger dict); arrays are numpy, or cuda tensors if device=True."""
        C, G = self.C, self.G
        shapes = {"N": (G, C), "F": (G, 3, C), "xHII": (C,), "xHeII": (C,), "xHeIII": (C,), "eth": (C,)}
        if device:
            out = {k: self.torch.empty(s, dtype=self.torch.float64, device=self.dev) for k, s in shapes.items()}
        else:
            out = {k: np.empty(s) for k, s in shapes.items()}
        led = rt_download(self.h, out, True, G)
        return out, led

    def ledger(self):
        return rt_download(self.h, None, True, self.G)

    def gradients(self):
        gN = np.empty((self.G, 3, self.C))
        gF = np.empty((self.G, 3, 3, self.C))
        _check(self.h, lib().rt_debug_gradients(self.h, RT_MEM_HOST, _vp(gN.ctypes.data), _vp(gF.ctypes.data)),
               "rt_debug_gradients")
        return gN, gF

    def tiles(self):
        """(tile of every cell in the caller's order (C,), per-tile (owned faces, forward halo, table words,
        flux launch class) (T, 4)) as numpy int32 arrays (rt_debug_tiles)."""
        T = self.tile_info()["tiles"]
        of_cell = np.zeros(self.C, dtype=np.int32)
        desc = np.zeros((T, 4), dtype=np.int32)
        _check(self.h, lib().rt_debug_tiles(self.h, RT_MEM_HOST, _vp(of_cell.ctypes.data), _vp(desc.ctypes.data)), "rt_debug_tiles")
        return of_cell, desc

    def tile_timeline(self, dt):
        """One subcycle with per-tile time stamps of the flux kernel: (T, 8) uint64 array (include/rt.h)."""
        T = self.tile_info()["tiles"]
        out = np.zeros((T, 8), dtype=np.uint64)
        _check(self.h, lib().rt_debug_tile_timeline(self.h, float(dt), T, _vp(out.ctypes.data)), "rt_debug_tile_timeline")
        return out

    def profile(self, enable):
        _check(self.h, lib().rt_profile(self.h, int(bool(enable))), "rt_profile")

    def profile_read(self):
        ms = np.zeros(6)
        cnt = np.zeros(6, dtype=np.int64)
        _check(self.h, lib().rt_profile_read(self.h, _vp(ms.ctypes.data), _vp(cnt.ctypes.data)), "rt_profile_read")
        names = ("chem", "grad", "flux", "update", "reduce", "other")
        return {k: (float(ms[i]), int(cnt[i])) for i, k in enumerate(names)}

    def tile_info(self):
        out = np.zeros(16, dtype=np.int64)
        _check(self.h, lib().rt_tile_info(self.h, _vp(out.ctypes.data)), "rt_tile_info")
        return {"cells_per_tile": int(out[0]), "tiles": int(out[1]), "max_slots": int(out[2]), "refaces": int(out[3]),
                "max_halo": int(out[4]), "halo_cells": int(out[5]), "max_table_words": int(out[6]),
                "table_words": int(out[7]), "max_owned": int(out[8]), "max_forward_halo": int(out[9]),
                "smem_grad": int(out[10]), "smem_flux": int(out[11]),
                "flux_class_a": {"tiles": int(out[12]), "max_owned": int(out[13]), "max_forward_halo": int(out[14]),
                                 "smem": int(out[15])}}

    def launches(self):
        return int(lib().rt_kernel_launches(self.h))

    def close(self):
        if getattr(self, "h", None):
            rt_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:      # interpreter shutdown: module globals may already be gone
            pass
