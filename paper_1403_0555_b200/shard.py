"""Host-side logic of the N > 1 launch.

The path shards over starts: a start's trajectory is a pure function of (orbit, seed, start index, omega,
eps), and the paper itself runs its GPUs from a host loop over independent samples.  Every rank
therefore takes a disjoint, contiguous range of start indices of the same orbit and runs the whole hot path on
it; there is NO data-path collective ("replicas only").  What is exchanged is the measurement -- the step time
(max over ranks) and the work counters (sum over ranks) -- and, once at the end, the ranks' distinct-copy tables
(SURVEY section 8(f)-4): `gather_copy_tables` all-gathers {F/(dV), signature, first start, multiplicity} per copy,
`u1gf_merge_copy_tables` (on every rank, or on rank 0) identifies the copies of different ranks with each other, and
`global_copy_ids` turns a rank's local copy ids into ids of the whole job.

This module holds no arithmetic of the method and works on any torch.distributed backend (nccl on the GPUs,
gloo in the CPU tests).
"""
from __future__ import annotations

import os
from dataclasses import dataclass


@dataclass(frozen=True)
class RankInfo:
    rank: int
    world: int
    local_rank: int


def rank_info_from_env(env=None) -> RankInfo:
    """RANK / WORLD_SIZE / LOCAL_RANK as torchrun exports them (1 process = 1 GPU); single process if unset."""
    env = os.environ if env is None else env
    return RankInfo(int(env.get("RANK", "0")), int(env.get("WORLD_SIZE", "1")), int(env.get("LOCAL_RANK", "0")))


def weak_start_range(rank: int, world: int, n_per_rank: int) -> tuple[int, int]:
    """Weak scaling (bench.py): every rank relaxes `n_per_rank` starts; rank r owns [r*n, (r+1)*n)."""
    if not (0 <= rank < world) or n_per_rank < 0:
        raise ValueError("bad rank / world / n_per_rank")
    return rank * n_per_rank, n_per_rank


def strong_start_range(rank: int, world: int, n_total: int) -> tuple[int, int]:
    """Strong scaling: `n_total` starts split into contiguous ranges whose sizes differ by at most one."""
    if not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad rank / world / n_total")
    q, r = divmod(n_total, world)
    first = rank * q + min(rank, r)
    return first, q + (1 if rank < r else 0)


def aggregate(total_ms: float, counters, dist=None, device="cpu"):
    """(max over ranks of total_ms, sum over ranks of each counter).  `dist` is torch.distributed (initialised) or
    None for a single process.  Counters are summed in float64 (exact below 2^53)."""
    counters = [float(c) for c in counters]
    if dist is None:
        return float(total_ms), counters
    import torch
    t = torch.tensor([float(total_ms)], dtype=torch.float64, device=device)
    c = torch.tensor(counters, dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t[0]), [float(x) for x in c]


def gather_copy_tables(F_rep, sig_rep, first_start, multiplicity, dist=None):
    """All-gather the ranks' copy tables (tensors of n_copies_r, [n_copies_r, 4], n_copies_r, n_copies_r entries; the
    first_start entries must be GLOBAL start indices).  Returns (F, sig, first_start, multiplicity, offsets): the tables
    concatenated in rank order and offsets[r] = position of rank r's first entry (length world + 1).  Table sizes differ
    between ranks, so they are padded to the largest for the collective and trimmed afterwards."""
    import torch
    if dist is None:
        return F_rep, sig_rep, first_start, multiplicity, [0, int(F_rep.numel())]
    world = dist.get_world_size()
    dev = F_rep.device
    cnt = torch.tensor([int(F_rep.numel())], dtype=torch.int64, device=dev)
    counts = [torch.zeros_like(cnt) for _ in range(world)]
    dist.all_gather(counts, cnt)
    counts = [int(c[0]) for c in counts]
    m = max(max(counts), 1)

    def gather(t, width, dtype):
        pad = torch.zeros((m, width), dtype=dtype, device=dev)
        pad[:t.shape[0]] = t.reshape(-1, width).to(dtype)
        parts = [torch.zeros_like(pad) for _ in range(world)]
        dist.all_gather(parts, pad)
        return torch.cat([p[:c] for p, c in zip(parts, counts)])
    F = gather(F_rep, 1, torch.float64).reshape(-1)
    S = gather(sig_rep, 4, torch.float64)
    fs = gather(first_start, 1, torch.int64).reshape(-1)
    mu = gather(multiplicity, 1, torch.int64).reshape(-1)
    offsets = [0]
    for c in counts:
        offsets.append(offsets[-1] + c)
    return F, S, fs, mu, offsets


def global_copy_ids(local_copy_id, merged_id, offset):
    """Ids of the whole job for a rank's starts: merged_id[offset + local id], -1 (not converged) kept."""
    import torch
    loc = local_copy_id.long()
    out = torch.full_like(loc, -1)
    ok = loc >= 0
    out[ok] = merged_id.long()[offset + loc[ok]]
    return out
