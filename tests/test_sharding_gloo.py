"""World-size-2 CPU test (gloo) of the marker sharding used by bench.py --gpus N.

The push itself has no collective: what can go wrong across ranks is the bookkeeping -- shards that
overlap or repeat, a whole-job figure that is not the max over ranks -- and that is what is checked here."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2107_13663_b200 import shard


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import synth
        w = synth.make_config(0, n_markers=257, nx=8, seed=shard.shard_seed(0, rank))
        ms_local = 3.0 + 2.0 * rank                     # rank 1 is the slow one
        ms, = shard.max_over_ranks([ms_local], dist)
        counts = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(counts, torch.tensor([w.n_markers]))
        rate = shard.whole_job_rate([int(c) for c in counts], 10, ms)
        b, e = shard.shard_range(1000 + 1, rank, world)
        out[rank] = (float(w.markers["x"][:8].sum()), ms, rate, b, e)
    finally:
        dist.destroy_process_group()


def test_two_rank_shards_and_max_over_ranks():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    r0, r1 = out[0], out[1]
    assert r0[0] != r1[0]                                # different seeds: different markers
    assert r0[1] == r1[1] == 5.0                         # max over ranks, seen by both
    assert r0[2] == r1[2] == 2 * 257 * 10 / 5.0e-3       # whole job = all markers / slowest rank
    assert (r0[3], r0[4], r1[3], r1[4]) == (0, 501, 501, 1001)   # contiguous, disjoint, complete


def _worker_moments(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        import synth
        w = synth.make_config(1, n_markers=3001, nx=12, tables=(rank == 0))       # only rank 0 fits the tables
        rng = np.random.Generator(np.random.PCG64(5))
        w.markers["w"] = rng.normal(size=w.n_markers)
        # (1) the field tables travel as one byte image from rank 0 (here: the host tables, pickled to bytes)
        if rank == 0:
            blob = np.concatenate([w.eq_coef.ravel(), w.pert_coef.ravel()]).view(np.uint8)
            buf = torch.from_numpy(blob.copy())
        else:
            buf = None
        buf = shard.broadcast_bytes(buf, dist, 0)
        flat = buf.numpy().view(np.float64)
        n_eq = w.n_elems * 4 * 21
        eq_coef = flat[:n_eq].reshape(w.n_elems, 4, 21)
        pert_coef = flat[n_eq:].reshape(w.n_modes, w.n_elems, 7, 2, 21)
        mesh = oracle.Mesh(w.node_RZ, w.tri, eq_coef, pert_coef, w.n_tor, w.omega)
        sp = oracle.species_of(w)
        # (2) every rank deposits its shard of the SAME global marker set; the tables are summed
        b, e = shard.shard_range(w.n_markers, rank, world)
        mine = {k: v[b:e] for k, v in w.markers.items()}
        rhs, _ = oracle.deposit(mesh, sp, mine, 1, 0.3)
        t = torch.from_numpy(rhs.copy())
        shard.allreduce_moments(t, dist)
        whole, _ = oracle.deposit(mesh, sp, w.markers, 1, 0.3)
        out[rank] = (float(np.abs(t.numpy() - whole).max()), float(np.abs(whole).max()), int(buf.numel()), e - b)
    finally:
        dist.destroy_process_group()


def test_two_rank_field_broadcast_and_moment_allreduce():
    """The two exchange steps around the push: rank 1 never sees the host tables, it receives rank 0's
    byte image; the all-reduced moment table of the two marker shards equals the deposition of the whole marker set."""
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker_moments, args=(world, _free_port(), out), nprocs=world, join=True)
    for r in range(world):
        err, scale, nbytes, n_mine = out[r]
        assert err <= 1e-12 * scale and scale > 0
        assert nbytes == out[0][2] > 0
    assert out[0][3] + out[1][3] == 3001


def test_shard_range_partitions_every_count():
    for n in (0, 1, 7, 64, 1000):
        for world in (1, 2, 3, 8):
            edges = [shard.shard_range(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[k][1] == edges[k + 1][0] for k in range(world - 1))
            sizes = [e - b for b, e in edges]
            assert max(sizes) - min(sizes) <= 1
    assert shard.shard_seed(3, 0) == 1003                # rank 0 draws the documented seed
    assert len({shard.shard_seed(3, r) for r in range(8)}) == 8
