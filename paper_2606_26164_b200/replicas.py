"""Multi-GPU host logic: independent replicas.

The CHISAO cycle has two cross-sample steps (f_max of Eq. 3 and the deduplication of Eq. 4),
so sharding one population over ranks would change the method; BASELINE.json's north_star runs everything on
one GPU.  `bench.py --gpus N` therefore runs N independent replicas of the workload, one process per GPU,
with rank-specific seeds for the initial population and the Philox stream; there is no data-path collective.
The only communication is the reduction of the timing (max over ranks) and of the work counters (sum).
"""
from __future__ import annotations

from . import inputs


def replica_workload(c: int, rank: int, N=None, n_osc=None):
    """Workload of replica `rank`: same objective (parameters are part of the problem), its own initial
    population seed and algorithm seed."""
    wl = inputs.config(c, N=N, n_osc=n_osc)
    if rank:
        wl.hp.seed = wl.hp.seed + 100000 * rank
        wl.x0 = inputs.uniform_population(wl.hp.N, wl.hp.lo, wl.hp.hi, 2000 + c + 100000 * rank)
    return wl


def _reduce(value: float, dist, device, op_name: str) -> float:
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=getattr(dist.ReduceOp, op_name))
    return float(t.item())


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    return _reduce(value, dist, device, "MAX")


def sum_over_ranks(value: float, dist=None, device="cpu") -> float:
    return _reduce(value, dist, device, "SUM")
