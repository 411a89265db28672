"""Multi-GPU path = replicas only: the protein list is sharded across ranks by
pf_sched_partition, every rank batches its own shard with the bucket scheduler, and the only cross-rank traffic is the
timing reduction bench.py does (MAX over ranks).  Covered here with world_size 2 on the gloo backend, CPU only."""
import os
import socket

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

import paper_2111_06340_b200 as pf
import pf_synth as ps

BUCKETS = list(ps.CFG5_BUCKETS)


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2111_06340_b200 import build
    build.build()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, lengths, S, q):
    import torch
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ranks = pf.partition(lengths, BUCKETS, S, world)          # every rank computes the same assignment, no talking
        mine = [i for i, r in enumerate(ranks) if r == rank]
        sched = pf.Scheduler(BUCKETS, 8 << 30, S)
        for i in mine:
            sched.add(i, lengths[i])
        done, cost = [], 0.0
        for ids, lens, bucket in sched.batches():
            done += ids
            cost += len(ids) * pf.sched_cost(bucket, S)
        # what bench.py does with its per-rank time: MAX over ranks; and the whole-job unit count: SUM
        t = torch.tensor([cost], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        n = torch.tensor([len(done)], dtype=torch.int64)
        dist.all_reduce(n, op=dist.ReduceOp.SUM)
        gathered = [None] * world
        dist.all_gather_object(gathered, sorted(done))
        q.put((rank, ranks, sorted(done), cost, float(t[0]), int(n[0]), gathered))
    finally:
        dist.destroy_process_group()


def test_list_sharding_world2_gloo():
    world, S = 2, 512
    lengths = [int(x) for x in ps.cfg5_lengths(5, 200)]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, lengths, S, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, ranks0, done0, cost0, tmax0, n0, g0), (_, ranks1, done1, cost1, tmax1, n1, g1) = res
    assert ranks0 == ranks1                                        # deterministic: identical on both ranks
    assert sorted(done0 + done1) == list(range(len(lengths)))      # every protein exactly once
    assert not set(done0) & set(done1)
    assert n0 == n1 == len(lengths)
    assert tmax0 == tmax1 == max(cost0, cost1)
    assert g0 == g1 == [done0, done1]
    # LPT guarantee: the heavier rank exceeds the mean by at most one protein's cost
    worst_item = max(pf.sched_cost(b, S) for b in BUCKETS)
    assert max(cost0, cost1) - (cost0 + cost1) / 2 <= worst_item


def test_partition_properties():
    lengths = [int(x) for x in ps.cfg5_lengths(3, 500)]
    for world in (1, 2, 4, 8):
        ranks = pf.partition(lengths, BUCKETS, 512, world)
        assert len(ranks) == len(lengths) and set(ranks) <= set(range(world))
        load = np.zeros(world)
        for L, r in zip(lengths, ranks):
            b = min(x for x in BUCKETS if x >= L)
            load[r] += pf.sched_cost(b, 512)
        assert load.max() - load.mean() <= pf.sched_cost(BUCKETS[-1], 512)
    with pytest.raises(pf.PfError):
        pf.partition([400], BUCKETS, 512, 2)                       # longer than the largest bucket
    assert pf.partition([], BUCKETS, 512, 2) == []


def test_cost_model_matches_flop_formula():
    """pf_sched_cost restates SURVEY.md §8(d) F(S, N); pf_synth.gemm_flops_per_block is the bench's copy of it."""
    for N in BUCKETS:
        assert pf.sched_cost(N, 512) == pytest.approx(ps.gemm_flops_per_block(512, N), rel=1e-12)
