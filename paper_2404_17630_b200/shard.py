"""Sharded runs: one process per GPU, each with a contiguous range of
the Peano-Hilbert order of the cells plus one layer of ghost cells.

Host logic and plumbing only: every step of the path runs in librt.so's kernels (include/rt.h, "sharded runs").
Per subcycle the ranks exchange the ghosts' primitive variables before each gradient pass and the ghosts'
gradients before each flux pass; the fluxes of cross-shard faces are computed on both sides
(PAPER.md:258), so no flux travels and the update needs no third exchange.

  hilbert_keys(mesh)            Peano-Hilbert key of every cell (numpy)
  partition(mesh, world)        owner rank of every cell: equal contiguous ranges of the curve
  Shard(mesh, owner, rank)      the local mesh of a rank (owned cells, then ghosts; every ghost closed by
                                reflective faces), the send / receive lists per peer
  ShardedSolver                 rt.Solver on a shard + the exchange; transports: DistComm (torch.distributed:
                                NCCL on GPUs, gloo for the CPU tests of the plan) and LocalGroup (several shards
                                on ONE device in one process, run in lock-step with plain copies: the
                                single-GPU parity test of the sharded path)
"""
import numpy as np

from .inputs import mesh as M
from .inputs.mesh import BC_REFLECT

HILBERT_BITS = 16


def hilbert_keys(mesh, bits=HILBERT_BITS):
    """Key of every cell along the 3-D Peano-Hilbert curve through the box (Skilling's transpose algorithm,
    vectorised over the cells): (C,) uint64."""
    x = np.empty((3, mesh.ncell), dtype=np.uint64)
    for a in range(3):
        q = np.floor(np.asarray(mesh.centroid[a]) / float(mesh.box[a]) * (1 << bits))
        x[a] = np.clip(q, 0, (1 << bits) - 1).astype(np.uint64)
    one = np.uint64(1)
    top = one << np.uint64(bits - 1)
    qb = top
    while qb > one:                                    # undo the excess work of the Gray code
        p = qb - one
        for i in range(3):
            hit = (x[i] & qb) != 0
            x[0] = np.where(hit, x[0] ^ p, x[0])
            t = np.where(hit, np.uint64(0), (x[0] ^ x[i]) & p)
            x[0] ^= t
            x[i] ^= t
        qb >>= one
    for i in range(1, 3):                              # Gray encode
        x[i] ^= x[i - 1]
    t = np.zeros(mesh.ncell, dtype=np.uint64)
    qb = top
    while qb > one:
        t = np.where((x[2] & qb) != 0, t ^ (qb - one), t)
        qb >>= one
    x ^= t
    key = np.zeros(mesh.ncell, dtype=np.uint64)        # interleave: bit b of x[0], x[1], x[2], from the top
    for b in range(bits - 1, -1, -1):
        for i in range(3):
            key = (key << one) | ((x[i] >> np.uint64(b)) & one)
    return key


def partition(mesh, world, keys=None):
    """owner[C]: rank r owns the r-th of `world` equal contiguous ranges of the Peano-Hilbert order."""
    keys = hilbert_keys(mesh) if keys is None else keys
    order = np.argsort(keys, kind="stable")
    owner = np.empty(mesh.ncell, dtype=np.int32)
    bounds = (np.arange(world + 1, dtype=np.int64) * mesh.ncell) // world
    for r in range(world):
        owner[order[bounds[r]:bounds[r + 1]]] = r
    return owner


class Shard:
    """The part of `mesh` that rank `rank` works on.

    cells        global ids of the local cells: the `nown` owned ones (ascending), then the ghosts (ascending)
    mesh         the local mesh in local numbering.  Faces: every face with a local cell.  A ghost keeps all its
                 faces, so that it is a closed cell: those to other local cells as they are, those to cells that
                 are not local - and its boundary faces, which are its owner's business - as reflective
                 boundary faces with the ghost on the left (no ledger row, and the ghost is never updated here)
    flags        rt_set_active bytes: 1 owned, 3 ghost (see active_flags for individual time steps)
    send[q]      local ids of the owned cells that are ghosts on rank q, in ascending global id
    recv[q]      local ids of the ghosts owned by rank q, in ascending global id (= rank q's send[rank] order)
    """

    def __init__(self, mesh, owner, rank):
        owner = np.asarray(owner)
        L, R = np.asarray(mesh.left, dtype=np.int64), np.asarray(mesh.right, dtype=np.int64)
        inner = R >= 0
        Rs = np.where(inner, R, 0)
        mine = owner == rank
        # ghosts: the cells of other ranks across a face of an owned cell
        cross = inner & (mine[L] != mine[Rs])
        other = np.where(mine[L[cross]], Rs[cross], L[cross])
        ghosts = np.unique(other)
        owned = np.flatnonzero(mine)
        self.rank, self.nown, self.nghost = int(rank), int(owned.size), int(ghosts.size)
        self.cells = np.concatenate([owned, ghosts]).astype(np.int64)
        loc = np.full(mesh.ncell, -1, dtype=np.int64)
        loc[self.cells] = np.arange(self.cells.size)
        is_ghost = np.zeros(mesh.ncell, dtype=bool)
        is_ghost[ghosts] = True
        lL, lR = loc[L], np.where(inner, loc[Rs], -1)
        keep = (lL >= 0) | (lR >= 0)
        f = np.flatnonzero(keep)
        fl, fr, code = lL[f], lR[f], R[f]
        normal = np.asarray(mesh.normal)[:, f].copy()
        fcen = np.asarray(mesh.fcentroid)[:, f].copy()
        left = fl.copy()
        right = np.where(code >= 0, fr, code)                 # local right id, or the boundary code
        # 1. boundary faces of ghosts are the owner's: reflective here
        gb = (code < 0) & is_ghost[L[f]]
        right[gb] = BC_REFLECT
        # 2. the right cell is not local (then the left one is a ghost): reflective
        right[(code >= 0) & (fr < 0)] = BC_REFLECT
        # 3. the left cell is not local (the right one is a ghost): turn the face round
        flip = fl < 0
        if flip.any():
            cl, cr = np.asarray(mesh.centroid)[:, L[f][flip]], np.asarray(mesh.centroid)[:, Rs[f][flip]]
            d = cr - cl
            for a in range(3):                                 # the face centre in the right cell's frame
                if mesh.periodic[a]:
                    fcen[a, flip] += d[a] - (d[a] - mesh.box[a] * np.rint(d[a] / mesh.box[a]))
            left[flip] = fr[flip]
            right[flip] = BC_REFLECT
            normal[:, flip] *= -1.0
        self.faces = f
        self.mesh = M.Mesh(ncell=int(self.cells.size), nface=int(f.size), box=np.asarray(mesh.box, dtype=np.float64).copy(),
                           periodic=np.asarray(mesh.periodic, dtype=np.int32).copy(),
                           volume=np.ascontiguousarray(np.asarray(mesh.volume)[self.cells]),
                           centroid=np.ascontiguousarray(np.asarray(mesh.centroid)[:, self.cells]),
                           area=np.ascontiguousarray(np.asarray(mesh.area)[f]), normal=np.ascontiguousarray(normal),
                           fcentroid=np.ascontiguousarray(fcen), left=left.astype(np.int32), right=right.astype(np.int32),
                           meta={"shard": int(rank)})
        self.flags = np.where(np.arange(self.cells.size) < self.nown, 1, 3).astype(np.uint8)
        # who sends what: for every cross-rank face, each side's cell goes to the other side's rank
        a, b = L[inner], R[inner]
        x = owner[a] != owner[b]
        a, b = a[x], b[x]
        self.send, self.recv = {}, {}
        for src, dst in ((a, b), (b, a)):
            s = owner[src] == rank                              # my cell `src` is a ghost on owner[dst]
            for q in np.unique(owner[dst[s]]):
                ids = np.unique(src[s][owner[dst[s]] == q])
                self.send[int(q)] = np.union1d(self.send.get(int(q), np.zeros(0, np.int64)), ids)
            r = owner[dst] == rank                              # `src` is my ghost, owned by owner[src]
            for q in np.unique(owner[src[r]]):
                ids = np.unique(src[r][owner[src[r]] == q])
                self.recv[int(q)] = np.union1d(self.recv.get(int(q), np.zeros(0, np.int64)), ids)
        self.send_global = {q: v.astype(np.int64) for q, v in self.send.items()}
        self.recv_global = {q: v.astype(np.int64) for q, v in self.recv.items()}
        self.send = {q: loc[v].astype(np.int32) for q, v in self.send_global.items()}
        self.recv = {q: loc[v].astype(np.int32) for q, v in self.recv_global.items()}
        self.peers = sorted(set(self.send) | set(self.recv))

    def active_flags(self, active=None):
        """rt_set_active bytes of the local cells for a global active mask (individual time steps):
        bit 0 = the cell is active (at its owner too), bit 1 = ghost."""
        if active is None:
            return self.flags
        a = np.asarray(active)[self.cells].astype(bool).astype(np.uint8)
        return (a | np.where(np.arange(self.cells.size) < self.nown, 0, 2)).astype(np.uint8)

    def local_state(self, state):
        """The rows of a global inputs.configs.State (or dict) that belong to the local cells."""
        get = (lambda k: state[k]) if isinstance(state, dict) else (lambda k: getattr(state, k))
        out = {k: np.ascontiguousarray(np.asarray(get(k))[..., self.cells]) for k in ("N", "F", "xHII", "xHeII", "xHeIII", "eth", "nH")}
        return out

    def local_sources(self, sources):
        """(cell, rate) of the sources in OWNED cells, in local numbering (a ghost's source is its owner's)."""
        cell = np.asarray(sources.cell, dtype=np.int64)
        if cell.size == 0:
            return np.zeros(0, dtype=np.int32), np.zeros((np.asarray(sources.rate).shape[0], 0))
        loc = np.full(int(max(self.cells.max(), cell.max())) + 1, -1, dtype=np.int64)
        loc[self.cells[: self.nown]] = np.arange(self.nown)
        k = np.flatnonzero(loc[cell] >= 0)
        return loc[cell[k]].astype(np.int32), np.ascontiguousarray(np.asarray(sources.rate)[:, k])


# ------------------------------------------------------------------ transports
class DistComm:
    """Pairwise exchange over torch.distributed (NCCL for CUDA tensors, gloo for the CPU tests of the plan):
    one batch of isend / irecv per exchange, peers in ascending rank order on both sides."""

    def __init__(self, dist, group=None):
        self.dist, self.group = dist, group

    def exchange(self, send, recv):
        """send, recv: {peer rank: contiguous tensor}.  Returns when the receive buffers are complete (for CUDA
        tensors: complete in stream order on the current stream)."""
        ops = []
        for q in sorted(set(send) | set(recv)):
            if q in send and send[q].numel():
                ops.append(self.dist.P2POp(self.dist.isend, send[q], q, self.group))
            if q in recv and recv[q].numel():
                ops.append(self.dist.P2POp(self.dist.irecv, recv[q], q, self.group))
        if ops:
            for w in self.dist.batch_isend_irecv(ops):
                w.wait()

    def allreduce_sum(self, x):
        """Sum of a float64 numpy array over the ranks, added in rank order (deterministic)."""
        import torch
        world = self.dist.get_world_size(self.group)
        parts = [torch.zeros(x.size, dtype=torch.float64) for _ in range(world)]
        mine = torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64).ravel())
        backend = self.dist.get_backend(self.group)
        if backend == "nccl":
            dev = torch.device("cuda", torch.cuda.current_device())
            parts = [p.to(dev) for p in parts]
            mine = mine.to(dev)
        self.dist.all_gather(parts, mine, group=self.group)
        tot = np.zeros(x.size)
        for p in parts:
            tot = tot + p.cpu().numpy()
        return tot.reshape(x.shape)


# ------------------------------------------------------------------ one rank's solver
LEDGER_SUMS = ("stored", "injected", "absorbed", "outflow", "inflow_bc", "floor_added")


class ShardedSolver:
    """rt.Solver on this rank's shard, advanced phase by phase with the ghost exchanges in between.

    All ranks hold the global (synthetic) inputs and cut their part out of them: `mesh`, `state`, `sources` are
    global.  comm: DistComm, or None when a LocalGroup drives several of these in one process."""

    def __init__(self, mesh, params, state, sources, rank, world, comm=None, device=0, tuning=None, owner=None):
        import torch
        from . import rt
        self.rt, self.torch = rt, torch
        self.rank, self.world, self.comm = int(rank), int(world), comm
        self.owner = partition(mesh, world) if owner is None else np.asarray(owner)
        self.shard = sh = Shard(mesh, self.owner, rank)
        if getattr(params, "kappa", None) is not None:       # FIXED_OPACITY: the local cells' opacities
            import copy
            params = copy.copy(params)
            params.kappa = np.ascontiguousarray(np.asarray(params.kappa)[sh.cells])
        self.params = params
        self.heun = bool(params.heun)
        self.second_order = int(params.order) >= 2
        self.solver = rt.Solver(sh.mesh, params, device=device, tuning=tuning)
        self.dev = self.solver.dev
        from .inputs import configs as cfg
        cell, rate = sh.local_sources(sources)
        self.solver.init(sh.local_state(state), cfg.Sources(cell, rate))
        self.solver.set_active(sh.flags)
        i32 = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.int32), device=self.dev)
        self.send_ids = {q: i32(v) for q, v in sh.send.items()}
        self.recv_ids = {q: i32(v) for q, v in sh.recv.items()}
        self.bufs = {}
        for what in (rt.RT_HALO_U, rt.RT_HALO_GRAD):
            rb = self.solver.halo_row_bytes(what)
            self.bufs[what] = ({q: torch.empty(v.numel() * rb // 8, dtype=torch.float64, device=self.dev) for q, v in self.send_ids.items()},
                               {q: torch.empty(v.numel() * rb // 8, dtype=torch.float64, device=self.dev) for q, v in self.recv_ids.items()})
        self.exchanges = 0
        self.exchange(rt.RT_HALO_U)      # (nothing to do for identical inputs; keeps the ghosts valid for restarts from a gathered state)

    # --- the exchange, in three steps so that a LocalGroup can interleave the ranks
    def pack(self, what):
        send, _ = self.bufs[what]
        for q, ids in self.send_ids.items():
            self.solver.halo_pack(what, ids, send[q])
        return send

    def unpack(self, what):
        _, recv = self.bufs[what]
        for q, ids in self.recv_ids.items():
            self.solver.halo_unpack(what, ids, recv[q])

    def exchange(self, what):
        if self.comm is None:
            return
        send = self.pack(what)
        self.comm.exchange(send, self.bufs[what][1])
        self.unpack(what)
        self.exchanges += 1

    def set_active(self, active=None):
        """Global active mask of the next steps (individual time steps), or None for every cell."""
        self.solver.set_active(self.shard.active_flags(active))

    def phases(self):
        """(phase, field to exchange after it or None) of one subcycle."""
        rt = self.rt
        g = rt.RT_HALO_GRAD if self.second_order else None
        out = [(rt.RT_PHASE_CHEM, rt.RT_HALO_U), (rt.RT_PHASE_GRAD1, g)]
        if self.heun:
            out += [(rt.RT_PHASE_FLUX1, rt.RT_HALO_U), (rt.RT_PHASE_GRAD2, g), (rt.RT_PHASE_FLUX2, None)]
        else:
            out += [(rt.RT_PHASE_FLUX1, None)]
        return out

    def step(self, dt, nsub=1):
        for _ in range(nsub):
            for phase, what in self.phases():
                self.solver.step_phase(dt, phase)
                if what is not None:
                    self.exchange(what)

    def download_owned(self):
        """(global ids of the owned cells, their state rows, this rank's ledger)."""
        st, led = self.solver.download()
        n = self.shard.nown
        return self.shard.cells[:n], {k: v[..., :n] for k, v in st.items()}, led

    def ledger(self):
        """The run's ledger: the sum of the shards' (needs a comm)."""
        led = self.solver.ledger()
        if self.comm is None:
            return led
        x = np.stack([np.asarray(led[k], dtype=np.float64) for k in LEDGER_SUMS])
        tot = self.comm.allreduce_sum(x)
        out = dict(led)
        for i, k in enumerate(LEDGER_SUMS):
            out[k] = tot[i]
        cnt = self.comm.allreduce_sum(np.asarray([led["substeps_total"], led["cells_hit_cap"]], dtype=np.float64))
        out["substeps_total"], out["cells_hit_cap"] = int(cnt[0]), int(cnt[1])
        return out


class LocalGroup:
    """`world` shards on ONE device in one process, advanced in lock-step: every rank runs a phase, every rank packs,
    the send buffers are copied into the peers' receive buffers, every rank unpacks.  No rank's kernels wait on
    another's: the test harness of the sharded path where there is one GPU (tests/test_gpu_shard.py)."""

    def __init__(self, mesh, params, state, sources, world, device=0, tuning=None):
        owner = partition(mesh, world)
        self.ranks = [ShardedSolver(mesh, params, state, sources, r, world, None, device, tuning, owner) for r in range(world)]
        self.ncell = int(mesh.ncell)
        self.exchange(self.ranks[0].rt.RT_HALO_U)

    def exchange(self, what):
        sent = [s.pack(what) for s in self.ranks]
        for s in self.ranks:
            for q, buf in s.bufs[what][1].items():
                buf.copy_(sent[q][s.rank])
        for s in self.ranks:
            s.unpack(what)
            s.exchanges += 1

    def set_active(self, active=None):
        for s in self.ranks:
            s.set_active(active)

    def step(self, dt, nsub=1):
        for _ in range(nsub):
            for phase, what in self.ranks[0].phases():
                for s in self.ranks:
                    s.solver.step_phase(dt, phase)
                if what is not None:
                    self.exchange(what)

    def download(self):
        """(global state dict assembled from the owners, summed ledger)."""
        out, led = None, None
        for s in self.ranks:
            ids, st, l = s.download_owned()
            if out is None:
                out = {k: np.zeros(v.shape[:-1] + (self.ncell,)) for k, v in st.items()}
                led = {k: np.zeros_like(np.asarray(l[k], dtype=np.float64)) for k in LEDGER_SUMS}
                led.update({"substeps_total": 0, "cells_hit_cap": 0, "substeps_max": 0, "nsub_done": l["nsub_done"]})
            for k, v in st.items():
                out[k][..., ids] = v
            for k in LEDGER_SUMS:
                led[k] = led[k] + np.asarray(l[k], dtype=np.float64)
            led["substeps_total"] += l["substeps_total"]
            led["cells_hit_cap"] += l["cells_hit_cap"]
            led["substeps_max"] = max(led["substeps_max"], l["substeps_max"])
        return out, led
