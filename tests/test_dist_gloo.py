"""N>1 paths on CPU: world_size-2 gloo.

Request sharding (no data-path collective): each rank's shard is probed independently (here by the
oracle, standing in for the GPU kernels that a CPU box cannot run) and the gathered outputs must
equal the unsharded result.

Vocabulary sharding (one exchange step): each rank's per-row records over its slice of W (oracle
row_stats_range, standing in for laser_probe_partial) go through parallel.gather_row_stats, and the
gathered [G, N, 4] buffer, merged in rank order with the oracle's merge operator, must give the
unsharded statistics."""
import os
import socket

import numpy as np
import pytest

from paper_2606_31580_b200 import parallel, workloads as wl


def test_shard_requests_partitions_exactly():
    rng = np.random.default_rng(0)
    for trial in range(50):
        R = int(rng.integers(0, 40))
        lens = rng.integers(0, 17, R)
        off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        for world in (1, 2, 3, 8):
            seen_r, seen_rows = [], []
            for rank in range(world):
                r0, r1, row0, row1, local = parallel.shard_requests(off, world, rank)
                assert 0 <= r0 <= r1 <= R and local[0] == 0 and len(local) == r1 - r0 + 1
                assert np.array_equal(local, off[r0:r1 + 1] - off[r0])
                seen_r.extend(range(r0, r1)); seen_rows.extend(range(row0, row1))
            assert seen_r == list(range(R))
            assert seen_rows == list(range(int(off[-1])))


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = wl.scaled("dist", 3000, 64, 0.05, 11, None, seed=77, var_len=(0, 9))
    tp = oracle.TauParams(**w.tau_params)
    r0, r1, row0, row1, local = parallel.shard_requests(w.req_offsets, world, rank)
    res = oracle.probe(w.hidden_f32()[row0:row1], w.W_f32(), local, w.load[r0:r1], tp)
    counts = [0] * world
    for k in range(world):
        a, b, *_ = parallel.shard_requests(w.req_offsets, world, k)
        counts[k] = b - a
    conf, ex = parallel.gather_request_outputs(dist, torch.from_numpy(res.conf.astype(np.float32)),
                                               torch.from_numpy(res.exit), counts)
    # timing reduction used by bench.py: max over ranks
    t = torch.tensor([float(rank + 1)], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    if rank == 0:
        q.put((conf.numpy(), ex.numpy(), float(t[0])))
    dist.barrier()
    dist.destroy_process_group()


def test_world2_gloo_sharded_equals_unsharded():
    import torch.multiprocessing as mp
    import oracle
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    conf, ex, tmax = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = wl.scaled("dist", 3000, 64, 0.05, 11, None, seed=77, var_len=(0, 9))
    full = oracle.probe(w.hidden_f32(), w.W_f32(), w.req_offsets, w.load, oracle.TauParams(**w.tau_params))
    np.testing.assert_allclose(conf, full.conf.astype(np.float32), rtol=0, atol=0)
    assert np.array_equal(ex, full.exit)
    assert tmax == 2.0


# ------------------------------------------------------------------------------- vocabulary sharding
def test_shard_vocab_partitions_exactly():
    for V in (1, 7, 1000, 151936, 128256):
        for world in (1, 2, 3, 8, 16):
            edges = [parallel.shard_vocab(V, world, r) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == V
            assert all(edges[r][1] == edges[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1


def _vp_worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = wl.scaled("vp-dist", 1501, 64, 0.05, 5, 4, seed=78)
    v0, v1 = parallel.shard_vocab(w.V, world, rank)
    N = w.N_alloc
    rec = np.zeros((N, 4), np.float32)          # {m, s, a (int bits), l_tok}: layout of laser_row_stats
    h, W = w.hidden_f32(), w.W_f32()
    for n in range(N):
        m, a, S = oracle.row_stats_range(h[n], W, v0, v1)
        rec[n, 0], rec[n, 1] = m, S
        rec[n, 2:3].view(np.int32)[0] = a
        rec[n, 3] = -np.inf
    local = torch.from_numpy(rec)
    allb = torch.empty((world, N, 4), dtype=torch.float32)
    parallel.gather_row_stats(dist, local, allb)
    if rank == 1:
        q.put(allb.numpy().copy())
    dist.barrier()
    dist.destroy_process_group()


def test_world2_gloo_vocab_parallel_exchange():
    import torch.multiprocessing as mp
    import oracle
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_vp_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    allb = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = wl.scaled("vp-dist", 1501, 64, 0.05, 5, 4, seed=78)
    full = oracle.row_stats(w.hidden_f32(), w.W_f32())
    assert allb.shape == (2, w.N_alloc, 4)
    for n in range(w.N_alloc):
        t = (-np.inf, -1, 0.0)
        for g in range(2):                      # rank order = ascending vocabulary
            t = oracle.merge(t, (float(allb[g, n, 0]), int(allb[g, n, 2:3].view(np.int32)[0]), float(allb[g, n, 1])))
        assert t[1] == full["a"][n]
        # records travel as float32: m and S are rounded once (1e-7 relative)
        assert abs(1.0 / t[2] - full["pmax"][n]) <= 5e-6
        v0, v1 = parallel.shard_vocab(w.V, 2, 1)
        assert v0 <= int(allb[1, n, 2:3].view(np.int32)[0]) < v1
