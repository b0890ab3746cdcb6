"""Data-parallel sharding of a probe batch across ranks (one process per GPU).

The probe's requests are independent (one confidence per request), so the N>1 path
shards REQUESTS: every rank holds a replica of W, probes its own contiguous slice of requests with
laser_probe_confidence, and no collective touches the data path.  torch.distributed (NCCL on GPUs,
gloo in the CPU tests) is used only to gather the small per-request outputs when a caller wants the
whole batch's mask on every rank.  The paper itself is single-GPU.

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
