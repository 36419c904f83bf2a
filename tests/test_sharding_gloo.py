"""The N > 1 path on CPU: world_size-2 gloo processes shard the job the way bench.py does under
torchrun (rank r owns shots [r*S, (r+1)*S), no data-path collective — DESIGN.md §8) and reduce the
timing / unit counts with the same collectives. The per-rank "device work" is played by the oracle
(tests may call it); what is under test is the host logic: disjoint contiguous shot ranges whose
union is the whole job, results identical to the unsharded run, max-over-ranks time, summed units."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SHOTS_PER_RANK = 40
CFG = 2


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    import torch
    import torch.distributed as dist

    import bench
    import oracle

    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert bench.dist_env() == (rank, world, rank)
        w = bench.make_workload("cfg%d" % CFG, SHOTS_PER_RANK, rank)       # bench.py's sharding rule
        o = oracle.run(w.x, w.y, w.toa, w.tot, w.toa_window_ticks, w.shot_period_ticks)
        dist.barrier()
        fake_ms = 10.0 + 5.0 * rank                                         # rank 1 is the slow one
        t = torch.tensor([fake_ms], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        tot = torch.tensor([w.n, o["n_clusters"]], dtype=torch.int64)
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
        q.put((rank, w.shot_begin, w.shots, w.n, o["n_clusters"], int(w.toa.min()), int(w.toa.max()),
               float(t.item()), int(tot[0]), int(tot[1]), o["c_sum_tot"].sum(), o["c_cx"].tobytes()))
    finally:
        dist.destroy_process_group()


def test_two_rank_shot_sharding():
    import torch.multiprocessing as mp

    sys.path.insert(0, ROOT)
    import gen
    import oracle

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    r0, r1 = res
    # contiguous, disjoint shot ranges covering the whole job
    assert (r0[1], r0[2]) == (0, SHOTS_PER_RANK) and (r1[1], r1[2]) == (SHOTS_PER_RANK, SHOTS_PER_RANK)
    assert r0[6] < r1[5]                      # every ToA of rank 0 precedes every ToA of rank 1
    assert r0[6] // gen.SHOT_PERIOD_TICKS < SHOTS_PER_RANK <= r1[5] // gen.SHOT_PERIOD_TICKS
    # reductions as bench.py does them: max over ranks of the time, sum of the units
    assert r0[7] == r1[7] == 15.0
    assert r0[8] == r1[8] == r0[3] + r1[3]
    assert r0[9] == r1[9] == r0[4] + r1[4]
    # sharded == unsharded: no link crosses a shot, so the union of the ranks' hits is the whole job's
    w = gen.generate(CFG, shots=2 * SHOTS_PER_RANK)
    o = oracle.run(w.x, w.y, w.toa, w.tot, w.toa_window_ticks, w.shot_period_ticks)
    assert w.n == r0[3] + r1[3]
    assert o["n_clusters"] == r0[4] + r1[4]
    assert int(o["c_sum_tot"].sum()) == int(r0[10]) + int(r1[10])
    assert o["c_cx"].tobytes() == r0[11] + r1[11]
