"""Brute-force numpy evaluation of one transport subcycle on a tiny mesh (pin P5).

Independent of oracle/rt_oracle.c in structure: dense cell x face incidence matrices instead of
CSR loops, the lab-frame form of the GLF/M1 flux instead of the rotation into the face frame
(PAPER.md:155), gradients by numpy.linalg.lstsq on the weighted system of eq (14)
 instead of the normal equations (15).  Only for meshes of a few cells.
"""
import numpy as np


def _minimg(d, box, per):
    d = d.copy()
    for a in range(3):
        if per[a]:
            d[a] -= box[a] * np.rint(d[a] / box[a])
    return d


def _chi(f):
    f = np.clip(f, 0.0, 1.0)
    return (3 + 4 * f * f) / (5 + 2 * np.sqrt(4 - 3 * f * f))


def _Pn(U, n, ct):
    """c^2 P.n in the lab frame for state U=(N,Fx,Fy,Fz), unit normal n."""
    N, F = U[0], U[1:]
    fn = np.linalg.norm(F)
    chi = _chi(fn / max(ct * N, 1e-300))
    out = 0.5 * (1 - chi) * n
    if fn > 0:
        nh = F / fn
        out = out + 0.5 * (3 * chi - 1) * np.dot(nh, n) * nh
    return N * out


def _glf(UL, UR, n, ct):
    ph = np.zeros(4)
    ph[0] = 0.5 * np.dot(UL[1:] + UR[1:], n) - 0.5 * ct * (UR[0] - UL[0])
    ph[1:] = 0.5 * ct * ct * (_Pn(UL, n, ct) + _Pn(UR, n, ct)) - 0.5 * ct * (UR[1:] - UL[1:])
    return ph


def _ghost(U, code, n, ghost, for_flux):
    if code == -1:
        return np.zeros(4) if for_flux else U.copy()
    if code == -2:
        G = U.copy()
        G[1:] -= 2 * np.dot(U[1:], n) * n
        return G
    return ghost[-3 - code].copy()


CAPPED = []   # faces whose number flux the donor cap clamped, appended by rhs() (tests clear and read it)


def rhs(mesh, U, ct, dt, ghost, order):
    """U: (C,4). Returns R (C,4) without sources, and boundary N-fluxes {face: A*Phi_N}."""
    C, F = mesh.ncell, mesh.nface
    box, per = mesh.box, mesh.periodic
    s, cf = mesh.centroid.T, mesh.fcentroid.T
    nrm = mesh.normal.T
    grad = np.zeros((C, 4, 3))
    faces_of = [[] for _ in range(C)]
    for f in range(F):
        faces_of[mesh.left[f]].append((f, 1))
        if mesh.right[f] >= 0:
            faces_of[mesh.right[f]].append((f, -1))
    if order >= 2:
        for i in range(C):
            rows, rhs_, vals, rs = [], [], [], []
            for f, sd in faces_of[i]:
                j = mesh.right[f] if sd > 0 else mesh.left[f]
                ri = _minimg(cf[f] - s[i], box, per)
                nout = sd * nrm[f]
                if j >= 0:
                    d = ri - _minimg(cf[f] - s[j], box, per)
                    Uj = U[j]
                else:
                    d = 2 * np.dot(ri, nout) * nout
                    Uj = _ghost(U[i], j, nrm[f], ghost, False)
                wgt = np.sqrt(mesh.area[f]) / np.linalg.norm(d)   # sqrt of the weight in eq (14)
                rows.append(wgt * d)
                rhs_.append(wgt * (Uj - U[i]))
                vals.append(Uj)
                rs.append(ri)
            A = np.array(rows); B = np.array(rhs_); vals = np.array(vals); rs = np.array(rs)
            g = np.linalg.lstsq(A, B, rcond=None)[0].T          # (4,3)
            for q in range(4):
                hi = max(U[i, q], vals[:, q].max()); lo = min(U[i, q], vals[:, q].min())
                dl = rs @ g[q]
                psi = np.ones(len(dl))
                psi[dl > 0] = (hi - U[i, q]) / dl[dl > 0]
                psi[dl < 0] = (lo - U[i, q]) / dl[dl < 0]
                grad[i, q] = min(1.0, psi.min()) * g[q]
    R = np.zeros((C, 4))
    bnd = {}
    for f in range(F):
        L, Rr = mesh.left[f], mesh.right[f]
        n = nrm[f]
        UL = U[L] + grad[L] @ _minimg(cf[f] - s[L], box, per)
        if Rr >= 0:
            UR = U[Rr] + grad[Rr] @ _minimg(cf[f] - s[Rr], box, per)
        else:
            UR = _ghost(UL, Rr, n, ghost, True)
        ph = _glf(UL, UR, n, ct)
        d = L if ph[0] > 0 else (Rr if ph[0] < 0 else -1)
        if d >= 0:
            lim = U[d, 0] * mesh.volume[d] / (dt * mesh.area[f])
            if abs(ph[0]) > lim:
                ph[0] = np.sign(ph[0]) * lim
                CAPPED.append(f)
        R[L] -= mesh.area[f] * ph / mesh.volume[L]
        if Rr >= 0:
            R[Rr] += mesh.area[f] * ph / mesh.volume[Rr]
        else:
            bnd[f] = mesh.area[f] * ph[0]
    return R, bnd


def _enforce(U, ct, n_floor):
    U = U.copy()
    U[:, 0] = np.maximum(U[:, 0], n_floor)
    fn = np.linalg.norm(U[:, 1:], axis=1)
    lim = ct * U[:, 0]
    sc = np.where(fn > lim, lim / np.maximum(fn, 1e-300), 1.0)
    U[:, 1:] *= sc[:, None]
    return U


def heun_step(mesh, U, ct, dt, ghost=None, order=2, n_floor=0.0, src=None):
    """One transport subcycle (reading S3): U1 = enforce(U + dt R(U)); U' = enforce((U + U1 + dt R(U1))/2)."""
    S = np.zeros_like(U)
    if src is not None:
        S[:, 0] = src / mesh.volume
    R0, _ = rhs(mesh, U, ct, dt, ghost, order)
    U1 = _enforce(U + dt * (R0 + S), ct, n_floor)
    R1, _ = rhs(mesh, U1, ct, dt, ghost, order)
    return _enforce(0.5 * U + 0.5 * (U1 + dt * (R1 + S)), ct, n_floor)
