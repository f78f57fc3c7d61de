"""N > 1 launch logic on CPU (gloo, world_size 2): the path shards over starts with no data-path collective
(DESIGN.md section 9), so what has to hold is
  * the ranks' start ranges are disjoint, contiguous and cover the job;
  * a start's result does not depend on which rank relaxed it (trajectories are pure functions of the start index),
    so the ranks' outputs concatenated equal one process relaxing the whole range (checked with the CPU oracle,
    which is allowed here: this is a test);
  * the measurement aggregation is max over ranks for time and sum over ranks for work.
"""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1403_0555_b200 import shard, synth  # noqa: E402

EXT, SEED, N_PER_RANK = (4, 4), 1, 96


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ri = shard.rank_info_from_env()
        first, n = shard.weak_start_range(ri.rank, ri.world, N_PER_RANK)
        th = synth.uniform_links(EXT, SEED)
        r = oracle.relax(EXT, th, SEED, n, first_start=first)
        ms = 10.0 + 5.0 * rank                                   # pretend rank 1 was the slow one
        t, (sw, conv) = shard.aggregate(ms, [int(r["sweeps"].sum()), int(((r["status"] & 1) == 0).sum())], dist)
        # copy tables of the ranks -> one table of the job.  The identification of copies across ranks is
        # u1gf_merge_copy_tables on the GPU; here (CPU, test) the oracle's count_copies on the gathered entries, ordered by
        # first start, stands in for it -- the host logic under test is the gather, the offsets and the id mapping.
        c = oracle.count_copies(r["F_norm"], r["sig"], r["status"])
        rep = c["rep"]
        F, S, fs, mu, offs = shard.gather_copy_tables(torch.as_tensor(r["F_norm"][rep]), torch.as_tensor(r["sig"][rep]),
                                                      torch.as_tensor(rep + first), torch.as_tensor(c["multiplicity"]), dist)
        order = np.argsort(fs.numpy(), kind="stable")
        mc = oracle.count_copies(F.numpy()[order], S.numpy()[order], np.zeros(order.size, dtype=np.uint8))
        merged_id = np.empty(order.size, dtype=np.int64)
        merged_id[order] = mc["copy_id"]
        gid = shard.global_copy_ids(torch.as_tensor(c["copy_id"]), torch.as_tensor(merged_id), offs[rank]).numpy()
        merged_mult = np.bincount(merged_id, weights=mu.numpy().astype(np.float64), minlength=mc["n_distinct"]).astype(np.int64)
        q.put((rank, first, n, r["sweeps"].copy(), r["F_norm"].copy(), t, sw, conv, gid, mc["n_distinct"], merged_mult,
               r["sig"].copy(), r["status"].copy()))
    finally:
        dist.destroy_process_group()


def test_start_ranges_partition_the_job():
    for world in (1, 2, 3, 8):
        got = []
        for r in range(world):
            f, n = shard.weak_start_range(r, world, 1000)
            got.append((f, n))
        assert got == [(r * 1000, 1000) for r in range(world)]
        for total in (0, 1, 7, 1000, 1 << 22):
            pos = 0
            sizes = []
            for r in range(world):
                f, n = shard.strong_start_range(r, world, total)
                assert f == pos
                pos += n
                sizes.append(n)
            assert pos == total and max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.weak_start_range(2, 2, 10)


def test_single_process_aggregate_is_identity():
    t, c = shard.aggregate(3.5, [7, 9])
    assert t == 3.5 and c == [7.0, 9.0]
    assert shard.rank_info_from_env({}) == shard.RankInfo(0, 1, 0)
    assert shard.rank_info_from_env({"RANK": "3", "WORLD_SIZE": "8", "LOCAL_RANK": "3"}) == shard.RankInfo(3, 8, 3)


def test_two_ranks_gloo(oracle):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=120) for _ in procs], key=lambda x: x[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, f0, n0, sw0, F0, t0, s0, c0, g0, nm0, mm0, sg0, st0), (r1, f1, n1, sw1, F1, t1, s1, c1, g1, nm1, mm1, sg1, st1) = res
    assert (f0, n0, f1, n1) == (0, N_PER_RANK, N_PER_RANK, N_PER_RANK)
    # the same job in one process
    th = synth.uniform_links(EXT, SEED)
    whole = oracle.relax(EXT, th, SEED, 2 * N_PER_RANK)
    assert (np.concatenate([sw0, sw1]) == whole["sweeps"]).all()
    assert (np.concatenate([F0, F1]) == whole["F_norm"]).all()       # bit-identical: same code, same start index
    # aggregation: max of the times, sum of the work, identical on both ranks
    assert t0 == t1 == 15.0
    assert s0 == s1 == float(whole["sweeps"].sum())
    assert c0 == c1 == float(((whole["status"] & 1) == 0).sum())
    # merged copy tables: every start gets the id one process over all starts gives it; multiplicities add up
    oc = oracle.count_copies(whole["F_norm"], whole["sig"], whole["status"])
    assert nm0 == nm1 == oc["n_distinct"]
    assert (np.concatenate([g0, g1]) == oc["copy_id"]).all()
    assert (mm0 == oc["multiplicity"]).all() and (mm1 == oc["multiplicity"]).all()
