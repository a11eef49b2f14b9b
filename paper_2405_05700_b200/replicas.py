"""Multi-GPU bookkeeping for ``bench.py --gpus N``: replicas only.

Photons are independent ("embarrassingly parallel") and BASELINE.json's north_star scopes
the path to one GPU with no sharding or collectives, so N GPUs run N independent replicas of the
workload (different Philox seeds).  The only cross-rank communication is this reduction of the
timing results: max of the times, sum of the work.  Works on any torch.distributed backend (nccl on
GPUs, gloo in the CPU tests).
"""
from __future__ import annotations


def replica_seed(base_seed: int, rank: int) -> int:
    """Every replica draws from its own Philox key so that replicas are independent samples."""
    return int(base_seed) + int(rank)


def reduce_results(dist, device, times: dict, work: dict) -> tuple[dict, dict]:
    """``times`` -> max over ranks, ``work`` -> sum over ranks.  ``dist`` may be None (single process)."""
    import torch

    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return dict(times), dict(work)
    tk, wk = sorted(times), sorted(work)
    t = torch.tensor([float(times[k]) for k in tk], dtype=torch.float64, device=device)
    w = torch.tensor([float(work[k]) for k in wk], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(w, op=dist.ReduceOp.SUM)
    return {k: float(v) for k, v in zip(tk, t.tolist())}, {k: float(v) for k, v in zip(wk, w.tolist())}


def aggregate_throughput(dist, device, units: float, seconds: float) -> float:
    """Whole-job throughput: units summed over ranks / max time over ranks."""
    t, w = reduce_results(dist, device, {"s": seconds}, {"u": units})
    return w["u"] / t["s"]
