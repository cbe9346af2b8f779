"""TEST INFRASTRUCTURE — NOT THE PRODUCT.  ctypes front end of oracle/rt_oracle.c.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2404_17630_b200 (inputs arrive as numpy
arrays / duck-typed objects with the attributes named below).
"""
import ctypes

import numpy as np

from .build import build_oracle

_lib = None
LEDGER_ROWS = ("stored", "injected", "absorbed", "outflow", "inflow_bc", "floor_added")


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build_oracle())
        vp, i64, i32, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
        L.oracle_create.restype = vp
        L.oracle_create.argtypes = [i64, i64, i32] + [vp] * 9 + [i32, vp]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_set_params.argtypes = [vp, dbl, vp, vp, i32, vp, dbl, dbl, dbl, dbl, dbl, dbl, dbl, i64, i32, i32]
        L.oracle_set_sources.argtypes = [vp, i32, vp, vp]
        L.oracle_set_active.argtypes = [vp, vp]
        L.oracle_set_precision.argtypes = [vp, i32]
        L.oracle_set_state.argtypes = [vp] * 8
        L.oracle_get_state.argtypes = [vp] * 7
        L.oracle_get_ledger.argtypes = [vp, vp, vp]
        L.oracle_step.argtypes = [vp, dbl, i32]
        L.oracle_transport_only.argtypes = [vp, dbl]
        L.oracle_chemistry_only.argtypes = [vp, dbl]
        L.oracle_gradients.argtypes = [vp, vp, vp]
        L.oracle_chi.restype = dbl
        L.oracle_chi.argtypes = [dbl]
        L.oracle_eddington.argtypes = [dbl, vp, dbl, vp]
        L.oracle_riemann.argtypes = [vp, vp, vp, dbl, vp]
        L.oracle_rates.argtypes = [dbl, vp]
        L.oracle_chem_cell.restype = i64
        L.oracle_chem_cell.argtypes = [vp, vp, vp, vp, dbl, dbl, vp, i64, vp, vp]
        L.oracle_nhalf.restype = i64
        L.oracle_nhalf.argtypes = [vp]
        L.oracle_get_geometry.argtypes = [vp] * 6
        _lib = L
    return _lib


def _p(a):
    return ctypes.c_void_p(a.ctypes.data) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def chi(f):
    return lib().oracle_chi(float(f))


def eddington(N, F, ctilde):
    D = np.zeros(9)
    Fv = _f64(F)
    lib().oracle_eddington(float(N), _p(Fv), float(ctilde), _p(D))
    return D.reshape(3, 3)


def riemann(UL, UR, n, ctilde):
    out = np.zeros(4)
    a, b, c = _f64(UL), _f64(UR), _f64(n)
    lib().oracle_riemann(_p(a), _p(b), _p(c), float(ctilde), _p(out))
    return out


def rates(T):
    r = np.zeros(15)
    lib().oracle_rates(float(T), _p(r))
    return r


class Oracle:
    """mesh: attributes ncell, nface, box, periodic, volume, centroid(3,C), area, normal(3,F),
    fcentroid(3,F), left, right.  params: attributes of inputs.configs.Params."""

    def __init__(self, mesh, params):
        self.L = lib()
        self.C, self.F, self.G = int(mesh.ncell), int(mesh.nface), int(params.ngroup)
        gs = params.ghost_state
        ng = 0 if gs is None else int(np.asarray(gs).shape[0])
        gs = _f64(gs) if ng else None
        arrs = [_f64(mesh.box), np.ascontiguousarray(mesh.periodic, dtype=np.int32), _f64(mesh.volume),
                _f64(mesh.centroid), _f64(mesh.area), _f64(mesh.normal), _f64(mesh.fcentroid),
                np.ascontiguousarray(mesh.left, dtype=np.int32), np.ascontiguousarray(mesh.right, dtype=np.int32)]
        self.h = self.L.oracle_create(self.C, self.F, self.G, *[_p(a) for a in arrs], ng, _p(gs))
        self.set_params(params)

    def __del__(self):
        if getattr(self, "h", None):
            self.L.oracle_destroy(self.h)
            self.h = None

    def set_params(self, p):
        sg, ep = _f64(p.sigma), _f64(p.eps_heat)
        kp = _f64(p.kappa) if p.kappa is not None else None
        self.L.oracle_set_params(self.h, p.ctilde, _p(sg), _p(ep), p.chem_mode, _p(kp), p.T_fixed, p.alphaB_override,
                                 p.y_he, p.f_accept, p.f_target, p.x_floor_rel, p.n_floor, p.max_substeps, p.order,
                                 p.heun)
        self.L.oracle_set_precision(self.h, int(getattr(p, "mixed", 0)))

    def set_sources(self, src):
        cell = np.ascontiguousarray(src.cell, dtype=np.int32)
        rate = _f64(src.rate)
        self.L.oracle_set_sources(self.h, int(cell.size), _p(cell), _p(rate))

    def set_active(self, active):
        """active: (C,) boolean mask of the cells taking part in the RT step, or None for all."""
        a = None if active is None else np.ascontiguousarray(active, dtype=np.uint8)
        assert a is None or a.shape == (self.C,)
        self.L.oracle_set_active(self.h, _p(a))

    def set_state(self, s):
        a = [_f64(s.N), _f64(s.F), _f64(s.xHII), _f64(s.xHeII), _f64(s.xHeIII), _f64(s.eth), _f64(s.nH)]
        assert a[0].shape == (self.G, self.C) and a[1].shape == (self.G, 3, self.C)
        self.L.oracle_set_state(self.h, *[_p(x) for x in a])
        self._nH = a[6]

    def get_state(self):
        """dict of numpy arrays N(G,C), F(G,3,C), xHII, xHeII, xHeIII, eth, nH."""
        C, G = self.C, self.G
        o = {"N": np.zeros((G, C)), "F": np.zeros((G, 3, C)), "xHII": np.zeros(C), "xHeII": np.zeros(C),
             "xHeIII": np.zeros(C), "eth": np.zeros(C)}
        self.L.oracle_get_state(self.h, *[_p(o[k]) for k in ("N", "F", "xHII", "xHeII", "xHeIII", "eth")])
        o["nH"] = self._nH.copy()
        return o

    def ledger(self):
        led = np.zeros((self.G, 6))
        cnt = np.zeros(3, dtype=np.int64)
        self.L.oracle_get_ledger(self.h, _p(led), _p(cnt))
        d = {k: led[:, i].copy() for i, k in enumerate(LEDGER_ROWS)}
        d.update(substeps_total=int(cnt[0]), substeps_max=int(cnt[1]), cells_hit_cap=int(cnt[2]))
        return d

    def step(self, dt, nsub=1):
        self.L.oracle_step(self.h, float(dt), int(nsub))

    def transport_only(self, dt):
        self.L.oracle_transport_only(self.h, float(dt))

    def chemistry_only(self, dt):
        self.L.oracle_chemistry_only(self.h, float(dt))

    def gradients(self):
        gN = np.zeros((self.G, 3, self.C))
        gF = np.zeros((self.G, 3, 3, self.C))
        self.L.oracle_gradients(self.h, _p(gN), _p(gF))
        return gN, gF

    def chem_cell(self, N, F, xHII, xHeII, xHeIII, eth, nH, dt, ntrace=100000):
        N = _f64(N).copy()
        F = _f64(F).copy().reshape(-1)
        x = np.array([xHII, xHeII, xHeIII, eth], dtype=np.float64)
        tr = np.zeros((ntrace, 3))
        nt = ctypes.c_int64(0)
        cap = ctypes.c_int(0)
        att = self.L.oracle_chem_cell(self.h, _p(N), _p(F), _p(x), float(nH), float(dt), _p(tr), ntrace,
                                      ctypes.byref(nt), ctypes.byref(cap))
        return {"N": N, "F": F.reshape(-1, 3), "xHII": x[0], "xHeII": x[1], "xHeIII": x[2], "eth": x[3],
                "attempts": int(att), "trace": tr[:nt.value].copy(), "hit_cap": bool(cap.value)}

    def geometry(self):
        nhf = self.L.oracle_nhalf(self.h)
        off = np.zeros(self.C + 1, dtype=np.int64)
        hf = np.zeros(nhf, dtype=np.int32)
        w = np.zeros((nhf, 3)); r = np.zeros((nhf, 3)); Mi = np.zeros((self.C, 3, 3))
        self.L.oracle_get_geometry(self.h, _p(off), _p(hf), _p(w), _p(r), _p(Mi))
        return off, hf, w, r, Mi
