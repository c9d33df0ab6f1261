"""Host-side logic of the N > 1 launch: "replicas only".

Gauge fixing is run once per configuration of an ensemble, so the hot path shards by giving every
rank (= GPU) its own lattice; there is no data-path collective.  What the ranks do share is (i) a
deterministic assignment of configurations to ranks and (ii) the timing reduction: the job time is
the MAX over ranks of the device time, and the job throughput is all ranks' iterations over that
time.  This module holds exactly that (no CUDA, no method arithmetic), so that it can be exercised
with the `gloo` backend on CPU (tests/test_replicas_gloo.py); bench.py uses it with `nccl`.
"""
from __future__ import annotations

from typing import List, Sequence


def rank_seed(base_seed: int, rank: int) -> int:
    """Seed of the configuration rank `rank` fixes: distinct per rank, reproducible per (base, rank)."""
    return int(base_seed) + 1000 * int(rank)


def assign_configs(n_configs: int, world: int, rank: int) -> List[int]:
    """Indices of an ensemble of `n_configs` configurations fixed by `rank` (round-robin; every
    configuration goes to exactly one rank, loads differ by at most one)."""
    if world < 1 or not (0 <= rank < world) or n_configs < 0:
        raise ValueError("assign_configs: need world >= 1, 0 <= rank < world, n_configs >= 0")
    return list(range(rank, n_configs, world))


def max_over_ranks(value: float, device=None) -> float:
    """MAX over all ranks of a per-rank scalar (device milliseconds); identity when not distributed."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    """SUM over all ranks of a per-rank scalar (e.g. iterations applied by each replica)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def job_throughput(units_all_ranks: float, max_ms: float) -> float:
    """Whole-job throughput: the units all ranks processed / the slowest rank's time (units per s)."""
    if max_ms <= 0:
        raise ValueError("job_throughput: non-positive time")
    return float(units_all_ranks) / (max_ms * 1e-3)


def gather_results(values: Sequence[float], device=None) -> List[List[float]]:
    """All ranks' per-rank result vectors (theta, F, iterations, ...), rank-ordered, on every rank."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [t.tolist()]
    out = [torch.empty_like(t) for _ in range(dist.get_world_size())]
    dist.all_gather(out, t)
    return [o.tolist() for o in out]
