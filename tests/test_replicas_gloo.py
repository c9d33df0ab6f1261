"""N > 1 launch path on CPU: world_size = 2, `gloo` backend ("replicas only").
The hot path has no data-path collective; what is distributed is the assignment of configurations
to ranks and the timing reduction bench.py reports (max over ranks, whole-job throughput)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1208_1186_b200 import replicas


def _free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank: int, world: int, port: int, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import lgf_inputs as gi
        # every rank makes ITS OWN lattice (distinct seed), as bench.py does under torchrun
        seed = replicas.rank_seed(gi.CONFIG_SEED, rank)
        U = gi.make_config((4, 4, 4, 4), seed, 0.59)
        checksum = float(U.real.sum())
        mine = replicas.assign_configs(7, world, rank)
        ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
        mx = replicas.max_over_ranks(ms)
        total_iters = replicas.sum_over_ranks(100.0)
        rows = replicas.gather_results([checksum, float(len(mine)), ms])
        out.put((rank, seed, mine, mx, total_iters, rows, replicas.job_throughput(total_iters, mx)))
    finally:
        dist.destroy_process_group()


def test_two_rank_replicas_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=120) for _ in range(world)])
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    (r0, s0, m0, mx0, t0, rows0, v0), (r1, s1, m1, mx1, t1, rows1, v1) = res
    assert (r0, r1) == (0, 1) and s0 != s1
    assert sorted(m0 + m1) == list(range(7)) and not set(m0) & set(m1)      # a partition of the ensemble
    assert abs(len(m0) - len(m1)) <= 1
    assert mx0 == mx1 == 15.0                                               # max over ranks, same on both
    assert t0 == t1 == 200.0
    assert v0 == v1 == pytest.approx(200.0 / 15e-3)
    assert rows0 == rows1 and len(rows0) == 2
    assert rows0[0][0] != rows0[1][0]                                       # different lattices per rank
    assert rows0[0][2] == 10.0 and rows0[1][2] == 15.0                      # rank-ordered


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.sum_over_ranks(2.0) == 2.0
    assert replicas.assign_configs(5, 1, 0) == [0, 1, 2, 3, 4]
    assert replicas.gather_results([1.0, 2.0]) == [[1.0, 2.0]]
    with pytest.raises(ValueError):
        replicas.assign_configs(5, 2, 2)
    with pytest.raises(ValueError):
        replicas.job_throughput(1.0, 0.0)
