"""Sharding of a probe batch across ranks (one process per GPU): by requests, or by vocabulary.

The probe's requests are independent (one confidence per request), so the N>1 path
shards REQUESTS: every rank holds a replica of W, probes its own contiguous slice of requests with
laser_probe_confidence, and no collective touches the data path.  torch.distributed (NCCL on GPUs,
gloo in the CPU tests) is used only to gather the small per-request outputs when a caller wants the
whole batch's mask on every rank.  The paper itself is single-GPU.

The second layout is the LM head's tensor-parallel one (SURVEY.md §8 e): every rank holds a slice
of W's rows and the whole batch, computes per-row partial statistics over its slice
(laser_probe_partial), the 16-byte records of all ranks meet on every rank - one all-gather of
N*16 bytes per rank, or peer stores issued by the producing kernel itself (PeerExchange) - and
laser_probe_combine merges them and finishes a3-a5.  This is the path's one real exchange step.

Host logic only: no arithmetic of the method lives here.
"""
from __future__ import annotations

import numpy as np


def shard_requests(req_offsets: np.ndarray, world: int, rank: int):
    """Contiguous request range for `rank`, balanced by ROW count (the unit of work).

    Returns (r0, r1, row0, row1, local_offsets): requests [r0, r1) own rows [row0, row1);
    local_offsets = req_offsets[r0:r1+1] - row0 (int32, starts at 0)."""
    off = np.asarray(req_offsets, np.int64)
    R = off.shape[0] - 1
    total = int(off[-1]) if R > 0 else 0
    # boundary b_k = first request whose start row >= k * total / world
    cuts = [int(np.searchsorted(off[:-1], (k * total) / world, side="left")) if R > 0 else 0
            for k in range(world)] + [R]
    cuts[0] = 0
    for k in range(1, world + 1):
        cuts[k] = max(cuts[k], cuts[k - 1])
    r0, r1 = cuts[rank], cuts[rank + 1]
    row0, row1 = (int(off[r0]), int(off[r1])) if R > 0 else (0, 0)
    local = (off[r0:r1 + 1] - row0).astype(np.int32) if R > 0 else np.zeros(1, np.int32)
    return r0, r1, row0, row1, local


def gather_request_outputs(dist, conf, exit_mask, counts):
    """all_gather of per-request outputs with uneven shard sizes.  `conf` float32 [R_local],
    `exit_mask` uint8 [R_local] torch tensors on the backend's device; `counts[k]` = requests on
    rank k.  Returns (conf_all [R], exit_all [R]) on every rank."""
    import torch
    world = dist.get_world_size()
    m = max(max(counts), 1)
    pc = torch.zeros(m, dtype=torch.float32, device=conf.device)
    pe = torch.zeros(m, dtype=torch.uint8, device=conf.device)
    pc[: conf.numel()] = conf
    pe[: exit_mask.numel()] = exit_mask
    gc = [torch.empty_like(pc) for _ in range(world)]
    ge = [torch.empty_like(pe) for _ in range(world)]
    dist.all_gather(gc, pc)
    dist.all_gather(ge, pe)
    return (torch.cat([g[:c] for g, c in zip(gc, counts)]),
            torch.cat([g[:c] for g, c in zip(ge, counts)]))


# ------------------------------------------------------------------------------- vocabulary-parallel
def shard_vocab(V: int, world: int, rank: int):
    """Contiguous vocabulary range [v0, v1) of `rank`: balanced to within one row, in rank order (so
    that the lowest-index tie-break of the merge is the global one)."""
    base, rem = divmod(int(V), int(world))
    v0 = rank * base + min(rank, rem)
    return v0, v0 + base + (1 if rank < rem else 0)


def gather_row_stats(dist, stats_local, stats_all, group=None):
    """The exchange step as a collective: all-gather of the [N, 4] float32 row records into
    [G, N, 4] (rank-major, the layout laser_probe_combine reads).  NCCL on GPUs, gloo on CPU."""
    dist.all_gather_into_tensor(stats_all.view(-1), stats_local.view(-1), group=group)
    return stats_all


class VocabParallelProbe:
    """One rank of the vocabulary-parallel probe: laser_probe_partial over this rank's rows of W ->
    exchange -> laser_probe_combine.  exchange="collective" all-gathers through torch.distributed
    (NCCL); exchange="peer" pushes the records from the reduce kernel into every rank's buffer over
    NVLink (PeerExchange: symmetric memory, no collective call on the data path)."""

    def __init__(self, dist, N, d, V, R, device, exchange="collective", group=None, debug_outputs=False,
                 w_layout=0):
        """w_layout = binding.W_KBLOCKED: every call's W_shard is binding.pack_w() of this rank's rows."""
        from . import binding as B
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.v0, self.v1 = shard_vocab(V, self.world, self.rank)
        self.shard = B.VocabShardProbe(N, d, self.v1 - self.v0, R, self.v0, self.world, device=device,
                                       debug_outputs=debug_outputs, w_layout=w_layout)
        self.exchange = exchange
        self.peers = PeerExchange(dist, N, self.world, self.rank, device, group) if exchange == "peer" else None

    def __call__(self, hidden, W_shard, req_offsets, load, params, token_ids=None, agg=0, stream=None):
        sh = self.shard
        if self.peers is not None:
            peers, stats_all, flags, epoch = self.peers.next()
            sh.partial(hidden, W_shard, req_offsets, token_ids=token_ids, stream=stream, peers=peers)
            return sh.combine(req_offsets, load, params, stats_all=stats_all, agg=agg,
                              token_prob=token_ids is not None, stream=stream, wait_flags=flags, epoch=epoch)
        sh.partial(hidden, W_shard, req_offsets, token_ids=token_ids, stream=stream)
        if stream is not None:
            # the collective is ordered against torch's CURRENT stream: make that the caller's stream
            import torch
            with torch.cuda.stream(stream):
                gather_row_stats(self.dist, sh.stats_local, sh.stats_all, self.group)
        else:
            gather_row_stats(self.dist, sh.stats_local, sh.stats_all, self.group)
        return sh.combine(req_offsets, load, params, agg=agg, token_prob=token_ids is not None, stream=stream)


class PeerExchange:
    """Two (gathered statistics [G, N, 4], flags [G]) sets per rank in symmetric memory
    (torch.distributed._symmetric_memory: every rank maps every peer's buffer), alternated by epoch
    parity as include/laser_probe.h asks.  next() returns the laser_probe_peers struct for the
    coming exchange together with this rank's own gathered buffer, flag array and the epoch."""

    def __init__(self, dist, N, world, rank, device, group=None):
        import torch
        import torch.distributed._symmetric_memory as symm
        from . import binding as B
        self.B, self.rank, self.world, self.epoch = B, rank, world, 0
        if world > B.MAX_PEERS:
            raise ValueError(f"at most {B.MAX_PEERS} ranks")
        grp = group if group is not None else dist.group.WORLD
        self.sets = []
        for _ in range(2):
            # one allocation per set: [G*N*4 floats of records | G uint32 flags (as 4-byte floats)]
            buf = symm.empty(world * N * 4 + world, dtype=torch.float32, device=device)
            buf.zero_()
            hdl = symm.rendezvous(buf, grp.group_name)
            ptrs = [int(q) for q in hdl.buffer_ptrs]
            stats = buf[: world * N * 4].view(world, N, 4)
            flags = buf[world * N * 4:].view(torch.int32)
            self.sets.append((buf, hdl, ptrs, stats, flags))
        torch.cuda.synchronize(device)
        dist.barrier(group=group)
        self.flag_offset = world * N * 4 * 4

    def next(self):
        self.epoch += 1
        buf, hdl, ptrs, stats, flags = self.sets[self.epoch & 1]
        pe = self.B.Peers()
        pe.rank, pe.world, pe.epoch = self.rank, self.world, self.epoch
        for g in range(self.world):
            pe.peer_stats[g] = ptrs[g]
            pe.peer_flags[g] = ptrs[g] + self.flag_offset
        return pe, stats, flags, self.epoch
