"""Host logic of the sharded path (paper_2404_17630_b200/shard.py): the
Peano-Hilbert partition, the local meshes with their closed ghosts, the send / receive plan, and the pairwise
exchange over a world_size-2 gloo group.  CPU only; the kernels' side is tests/test_gpu_shard.py."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2404_17630_b200 import shard as S
from paper_2404_17630_b200.inputs import configs as cfg
from paper_2404_17630_b200.inputs import mesh as M


def _meshes():
    return [M.voronoi(8, 1.0, 0.3, 11, periodic=True), M.voronoi(7, 2.0, 0.2, 12, periodic=False),
            M.cartesian(6, 1.0, periodic=False)]


def test_hilbert_keys_are_a_space_filling_order():
    m = M.cartesian(16, 1.0, periodic=False)
    k = S.hilbert_keys(m)
    assert np.unique(k).size == m.ncell
    c = m.centroid[:, np.argsort(k)]
    step = np.sqrt((np.diff(c, axis=1) ** 2).sum(0))
    assert np.allclose(step, 1.0 / 16)            # consecutive cells of the curve share a face: the Hilbert property
    # contiguous ranges are compact: an eighth of the curve is an octant of the box
    o = S.partition(m, 8, k)
    for r in range(8):
        ext = np.ptp(m.centroid[:, o == r], axis=1)
        assert np.all(ext < 0.5)


@pytest.mark.parametrize("world", [2, 3])
def test_partition_and_local_meshes(world):
    for m in _meshes():
        owner = S.partition(m, world)
        cnt = np.bincount(owner, minlength=world)
        assert cnt.sum() == m.ncell and cnt.max() - cnt.min() <= 1
        shards = [S.Shard(m, owner, r) for r in range(world)]
        seen = np.zeros(m.ncell, int)
        flux_faces = np.zeros(m.nface, int)
        for s in shards:
            lm = s.mesh
            seen[s.cells[: s.nown]] += 1
            assert np.all(owner[s.cells[: s.nown]] == s.rank) and np.all(owner[s.cells[s.nown:]] != s.rank)
            # every local cell, ghosts included, is closed: sum of outward A n vanishes
            acc = np.zeros((3, lm.ncell))
            np.add.at(acc, (slice(None), lm.left), lm.area * lm.normal)
            inner = lm.right >= 0
            np.subtract.at(acc, (slice(None), lm.right[inner]), (lm.area * lm.normal)[:, inner])
            tot = np.zeros(lm.ncell)
            np.add.at(tot, lm.left, lm.area)
            np.add.at(tot, lm.right[inner], lm.area[inner])
            assert np.all(np.sqrt((acc ** 2).sum(0)) <= 1e-10 * tot)
            # an owned cell has exactly its global faces, with its global boundary codes
            gl, gr = np.asarray(m.left)[s.faces], np.asarray(m.right)[s.faces]
            own_l = lm.left < s.nown
            own_r = inner & (lm.right < s.nown)
            flux_faces[s.faces[own_l | own_r]] += 1
            bnd_owned = (lm.right < 0) & own_l
            assert np.array_equal(lm.right[bnd_owned], gr[bnd_owned])
            # reflective faces added by the sharding sit on ghosts only
            added = (lm.right == M.BC_REFLECT) & ~((gr == M.BC_REFLECT) & (owner[gl] == s.rank))
            assert np.all(lm.left[added] >= s.nown)
            # volumes, areas and centres are the global ones
            assert np.array_equal(lm.volume, np.asarray(m.volume)[s.cells]) and np.array_equal(lm.area, np.asarray(m.area)[s.faces])
        assert np.all(seen == 1)
        # a face is evaluated by the owners of its cells: once inside a shard, on both sides across shards
        gR = np.asarray(m.right)
        innerg = gR >= 0
        crossg = innerg & (owner[np.asarray(m.left)] != owner[np.where(innerg, gR, 0)])
        assert np.all(flux_faces[crossg] == 2) and np.all(flux_faces[~crossg] == 1)
        # the plan: what r sends to q is what q expects from r, in the same order; ghosts = everything received
        for s in shards:
            got = np.concatenate([s.recv_global[q] for q in sorted(s.recv_global)]) if s.recv_global else np.zeros(0, np.int64)
            assert np.array_equal(np.sort(got), s.cells[s.nown:])
            for q, ids in s.send_global.items():
                assert np.array_equal(ids, shards[q].recv_global[s.rank])
                assert np.all(owner[ids] == s.rank)
                assert np.array_equal(s.cells[s.send[q]], ids)
            for q, ids in s.recv_global.items():
                assert np.array_equal(s.cells[s.recv[q]], ids)


def test_sources_and_active_flags_go_to_the_owner():
    w = cfg.get(3, 8)
    owner = S.partition(w.mesh, 2)
    shards = [S.Shard(w.mesh, owner, r) for r in range(2)]
    got = []
    for s in shards:
        cell, rate = s.local_sources(w.sources)
        assert np.all(cell < s.nown) and rate.shape == (w.params.ngroup, cell.size)
        got.append(s.cells[cell])
        st = s.local_state(w.state)
        assert np.array_equal(st["N"], w.state.N[:, s.cells]) and np.array_equal(st["F"], w.state.F[:, :, s.cells])
    assert np.array_equal(np.sort(np.concatenate(got)), np.sort(w.sources.cell))
    active = np.random.RandomState(4).rand(w.mesh.ncell) < 0.5
    for s in shards:
        f = s.active_flags(active)
        assert np.array_equal(f & 1, active[s.cells].astype(np.uint8))
        assert np.array_equal((f >> 1) & 1, (np.arange(s.cells.size) >= s.nown).astype(np.uint8))
        assert np.array_equal(s.active_flags(None), np.where(np.arange(s.cells.size) < s.nown, 1, 3))


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    m = M.voronoi(8, 1.0, 0.3, 11, periodic=True)            # every rank builds the same seeded mesh
    s = S.Shard(m, S.partition(m, world), rank)
    comm = S.DistComm(dist)
    # a field whose value is a function of the global cell id: rows of 3 doubles
    f = lambda ids: np.stack([ids * 1.0, ids * ids * 0.5, np.cos(ids)], axis=1)
    send = {q: torch.as_tensor(f(s.send_global[q])) for q in s.send}
    recv = {q: torch.zeros(len(s.recv[q]), 3, dtype=torch.float64) for q in s.recv}
    comm.exchange(send, recv)
    ok = all(np.array_equal(recv[q].numpy(), f(s.recv_global[q])) for q in s.recv)
    tot = comm.allreduce_sum(np.asarray([[1.0 + rank, 10.0], [0.5, rank]]))
    dist.barrier()
    out.put((rank, ok, tot.tolist(), sorted(s.peers)))
    dist.destroy_process_group()


def test_exchange_over_gloo_world_size_2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ok, tot, peers in got:
        assert ok                                             # every ghost received its owner's row
        assert tot == [[3.0, 20.0], [1.0, 1.0]]
        assert peers == [1 - rank]
