"""Mesh inputs: Cartesian face lists (configs 0, 1) and jittered-lattice Voronoi meshes
(configs 2-4) in the layout of `rt_mesh` (include/rt.h).

Input generators only; none of the RT method's arithmetic lives here.  Faces are stored
once, unit normal pointing from `left` to `right`; `right < 0` encodes a boundary:
-1 outflow, -2 reflective, -3-k Dirichlet ghost state k.
"""
import ctypes
import os
from dataclasses import dataclass, field

import numpy as np

BC_OUTFLOW = -1
BC_REFLECT = -2
BC_DIRICHLET0 = -3


@dataclass
class Mesh:
    ncell: int
    nface: int
    box: np.ndarray          # (3,)
    periodic: np.ndarray     # (3,) int32
    volume: np.ndarray       # (C,)
    centroid: np.ndarray     # (3, C)
    area: np.ndarray         # (F,)
    normal: np.ndarray       # (3, F)
    fcentroid: np.ndarray    # (3, F)   in the left cell's frame
    left: np.ndarray         # (F,) int32
    right: np.ndarray        # (F,) int32
    meta: dict = field(default_factory=dict)


def cartesian(n, box=1.0, periodic=False, bc=(BC_OUTFLOW,) * 6):
    """n^3 regular mesh as an unstructured face list.  Cell id = (ix*n+iy)*n+iz.

    bc = codes for (xlo, xhi, ylo, yhi, zlo, zhi) when not periodic.  Boundary faces have the
    boundary cell as `left` and the outward normal.
    """
    h = box / n
    C = n ** 3
    idx = np.arange(C, dtype=np.int64).reshape(n, n, n)
    g = (np.arange(n) + 0.5) * h
    cx, cy, cz = np.meshgrid(g, g, g, indexing="ij")
    centroid = np.stack([cx.ravel(), cy.ravel(), cz.ravel()])
    L, R, NRM, FC = [], [], [], []
    for ax in range(3):
        e = np.zeros(3)
        e[ax] = 1.0
        sl_lo = [slice(None)] * 3
        sl_hi = [slice(None)] * 3
        sl_lo[ax] = slice(0, n - 1)
        sl_hi[ax] = slice(1, n)
        l = idx[tuple(sl_lo)].ravel()
        r = idx[tuple(sl_hi)].ravel()
        fc = centroid[:, l].copy()
        fc[ax] += 0.5 * h
        L.append(l); R.append(r); NRM.append(np.tile(e[:, None], (1, l.size))); FC.append(fc)
        sl_a = [slice(None)] * 3
        sl_b = [slice(None)] * 3
        sl_a[ax] = n - 1
        sl_b[ax] = 0
        hi_cells = idx[tuple(sl_a)].ravel()
        lo_cells = idx[tuple(sl_b)].ravel()
        if periodic:
            fc = centroid[:, hi_cells].copy()
            fc[ax] += 0.5 * h
            L.append(hi_cells); R.append(lo_cells); NRM.append(np.tile(e[:, None], (1, hi_cells.size))); FC.append(fc)
        else:
            fc = centroid[:, lo_cells].copy()
            fc[ax] -= 0.5 * h
            L.append(lo_cells); R.append(np.full(lo_cells.size, bc[2 * ax], dtype=np.int64))
            NRM.append(np.tile(-e[:, None], (1, lo_cells.size))); FC.append(fc)
            fc = centroid[:, hi_cells].copy()
            fc[ax] += 0.5 * h
            L.append(hi_cells); R.append(np.full(hi_cells.size, bc[2 * ax + 1], dtype=np.int64))
            NRM.append(np.tile(e[:, None], (1, hi_cells.size))); FC.append(fc)
    left = np.concatenate(L).astype(np.int32)
    right = np.concatenate(R).astype(np.int32)
    normal = np.ascontiguousarray(np.concatenate(NRM, axis=1))
    fcentroid = np.ascontiguousarray(np.concatenate(FC, axis=1))
    F = left.size
    return Mesh(C, F, np.full(3, float(box)), np.full(3, int(bool(periodic)), dtype=np.int32),
                np.full(C, h ** 3), np.ascontiguousarray(centroid), np.full(F, h * h), normal, fcentroid,
                left, right, {"kind": "cartesian", "n": n, "h": h})


# ----------------------------------------------------------------------------- Voronoi
class _MgParams(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int32), ("periodic", ctypes.c_int32), ("bc_code", ctypes.c_int32),
                ("stagger", ctypes.c_int32), ("box", ctypes.c_double), ("jitter", ctypes.c_double),
                ("seed", ctypes.c_uint64)]


_lib = None


def meshgen_lib():
    global _lib
    if _lib is None:
        from ..build import build_meshgen, MESHGEN_SO
        if not os.path.exists(MESHGEN_SO):
            build_meshgen()
        _lib = ctypes.CDLL(MESHGEN_SO)
        _lib.mg_voronoi_cells.restype = ctypes.c_int
        _lib.mg_voronoi_cells.argtypes = [ctypes.POINTER(_MgParams), ctypes.c_int, ctypes.c_void_p] + [ctypes.c_void_p] * 4
        _lib.mg_voronoi_faces.restype = ctypes.c_int
        _lib.mg_voronoi_faces.argtypes = [ctypes.POINTER(_MgParams), ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
                                          ctypes.c_int64] + [ctypes.c_void_p] * 6
        _lib.mg_u01_c.restype = ctypes.c_double
        _lib.mg_u01_c.argtypes = [ctypes.c_uint64] * 3
    return _lib


def _ptr(a):
    return ctypes.c_void_p(a.ctypes.data)


def voronoi(n, box, jitter, seed, periodic, bc_code=BC_OUTFLOW, stagger=False):
    """Host build (OpenMP) of the Voronoi mesh of n^3 jittered-lattice generators, or of 2 n^3 generators
    on two interleaved lattices (stagger=True: the "2 x N^3 staggered grid" of PAPER.md:180, 290)."""
    lib = meshgen_lib()
    P = _MgParams(n, int(bool(periodic)), bc_code, int(bool(stagger)), box, jitter, seed)
    C = n ** 3 * (2 if stagger else 1)
    counts = np.zeros(C, dtype=np.int32)
    volume = np.zeros(C)
    centroid = np.zeros((3, C))
    st = np.zeros(2, dtype=np.int32)
    rc = lib.mg_voronoi_cells(ctypes.byref(P), 0, None, _ptr(counts), _ptr(volume), _ptr(centroid), _ptr(st))
    if rc != 0:
        raise RuntimeError("meshgen pass 1 failed rc=%d status=%s" % (rc, st))
    offsets = np.zeros(C, dtype=np.int64)
    np.cumsum(counts[:-1], out=offsets[1:])
    F = int(offsets[-1] + counts[-1])
    area = np.zeros(F)
    normal = np.zeros((3, F))
    fcen = np.zeros((3, F))
    left = np.zeros(F, dtype=np.int32)
    right = np.zeros(F, dtype=np.int32)
    rc = lib.mg_voronoi_faces(ctypes.byref(P), 0, None, _ptr(offsets), F, _ptr(area), _ptr(normal), _ptr(fcen),
                              _ptr(left), _ptr(right), _ptr(st))
    if rc != 0:
        raise RuntimeError("meshgen pass 2 failed rc=%d status=%s" % (rc, st))
    return Mesh(C, F, np.full(3, float(box)), np.full(3, int(bool(periodic)), dtype=np.int32), volume, centroid,
                area, normal, fcen, left, right, {"kind": "voronoi", "n": n, "h": box / n, "jitter": jitter, "seed": seed,
                                                  "stagger": bool(stagger)})


def voronoi_device(n, box, jitter, seed, periodic, bc_code=BC_OUTFLOW, device="cuda:0"):
    """Same mesh built directly in device memory; returns a Mesh whose arrays are torch tensors."""
    import torch
    lib = meshgen_lib()
    P = _MgParams(n, int(bool(periodic)), bc_code, 0, box, jitter, seed)
    C = n ** 3
    dev = torch.device(device)
    stream = torch.cuda.current_stream(dev).cuda_stream
    counts = torch.zeros(C, dtype=torch.int32, device=dev)
    volume = torch.zeros(C, dtype=torch.float64, device=dev)
    centroid = torch.zeros((3, C), dtype=torch.float64, device=dev)
    st = np.zeros(2, dtype=np.int32)
    vp = lambda t: ctypes.c_void_p(t.data_ptr())
    rc = lib.mg_voronoi_cells(ctypes.byref(P), 1, ctypes.c_void_p(stream), vp(counts), vp(volume), vp(centroid), _ptr(st))
    if rc != 0:
        raise RuntimeError("meshgen pass 1 failed rc=%d status=%s" % (rc, st))
    incl = torch.cumsum(counts, 0, dtype=torch.int64)
    F = int(incl[-1].item())
    offsets = incl - counts.to(torch.int64)
    del incl, counts
    area = torch.zeros(F, dtype=torch.float64, device=dev)
    normal = torch.zeros((3, F), dtype=torch.float64, device=dev)
    fcen = torch.zeros((3, F), dtype=torch.float64, device=dev)
    left = torch.zeros(F, dtype=torch.int32, device=dev)
    right = torch.zeros(F, dtype=torch.int32, device=dev)
    rc = lib.mg_voronoi_faces(ctypes.byref(P), 1, ctypes.c_void_p(stream), vp(offsets), F, vp(area), vp(normal),
                              vp(fcen), vp(left), vp(right), _ptr(st))
    if rc != 0:
        raise RuntimeError("meshgen pass 2 failed rc=%d status=%s" % (rc, st))
    del offsets
    return Mesh(C, F, np.full(3, float(box)), np.full(3, int(bool(periodic)), dtype=np.int32), volume, centroid,
                area, normal, fcen, left, right,
                {"kind": "voronoi", "n": n, "h": box / n, "jitter": jitter, "seed": seed, "device": str(dev)})
