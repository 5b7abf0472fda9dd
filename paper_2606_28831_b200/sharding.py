"""Rank sharding of a workload and the cross-rank reduction of a timed run (bench.py, N > 1).

Every (sequence, KV head) unit of the path is independent (the paper's own tensor-parallel deployment
exchanges nothing but a one-time gather of head counts, L555-562), so ranks take disjoint batches of the same shape and
there is NO data-path collective: the only exchange is this reduction of the measurement itself.
torch.distributed is plumbing here; the module holds none of the method's arithmetic and imports neither the CUDA
binding nor the oracle.
"""
from __future__ import annotations

import torch
import torch.distributed as dist

from workloads.synth import Workload, make_workload


def rank_workload(cfg_index: int, rank: int, **over) -> Workload:
    """The batch of rank `rank`: BASELINE.json configs[cfg_index] with its own seed (same shapes on every rank)."""
    wl = make_workload(cfg_index, **over)
    wl.seed += 1000 * rank
    return wl


def reduce_run(ms_device: float, ms_e2e: float, bytes_total: float, device) -> tuple[float, float, float]:
    """(max over ranks of the device-timed ms, max of the end-to-end ms, sum of the algorithmic bytes)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms_device), float(ms_e2e), float(bytes_total)
    red = torch.tensor([ms_device, ms_e2e], dtype=torch.float64, device=device)
    tot = torch.tensor([float(bytes_total)], dtype=torch.float64, device=device)
    dist.all_reduce(red, op=dist.ReduceOp.MAX)
    dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    return float(red[0]), float(red[1]), float(tot[0])


def job_throughput_gbs(ms_device: float, bytes_all_ranks: float) -> float:
    """Whole-job GB/s: bytes of all ranks over the slowest rank's time."""
    return bytes_all_ranks / (ms_device * 1e-3) / 1e9
