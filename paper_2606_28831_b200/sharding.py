"""Rank sharding of a workload and the cross-rank reduction of a timed run (bench.py, N > 1).

Every (sequence, KV head) unit of the path is independent (the paper's own tensor-parallel deployment
exchanges nothing but a one-time gather of head counts, L555-562), so ranks take disjoint batches of the same shape and
there is NO data-path collective: the only exchanges are this reduction of the measurement itself and, in the
tensor-parallel (KV-head) sharding, the gather of the per-head selection counts (L562).
torch.distributed is plumbing here; the module holds none of the method's arithmetic and imports neither the CUDA
binding nor the oracle.
"""
from __future__ import annotations

import torch
import torch.distributed as dist

import dataclasses

import numpy as np

from workloads.synth import Workload, make_workload


def rank_workload(cfg_index: int, rank: int, **over) -> Workload:
    """The batch of rank `rank`: BASELINE.json configs[cfg_index] with its own seed (same shapes on every rank)."""
    wl = make_workload(cfg_index, **over)
    wl.seed += 1000 * rank
    return wl


def head_shard(wl: Workload, rank: int, world: int) -> Workload:
    """Tensor-parallel (width) sharding: rank `rank` of `world` holds KV heads [rank Hkv / world,
    (rank + 1) Hkv / world) of every sequence with their G query heads each, its own block tables and its own selection
    ("each instance doing head-wise eviction on its own heads").  The shard generates exactly the rows the unsharded
    workload holds for those heads, so per-head results are identical to the single-GPU run."""
    assert wl.Hkv % world == 0 and wl.head_offset == 0
    hl = wl.Hkv // world
    sh = dataclasses.replace(wl, Hq=hl * wl.G, Hkv=hl, score_mode=wl.score_mode[rank * hl:(rank + 1) * hl].copy(),
                             temperature=wl.temperature[:, rank * hl:(rank + 1) * hl].copy(), head_offset=rank * hl,
                             Hkv_total=wl.Hkv, name=f"{wl.name}[heads {rank * hl}:{(rank + 1) * hl}]")
    sh.seed = wl.seed
    return sh


def gather_head_counts(sel_count_local, world: int):
    """The one exchange of the tensor-parallel deployment: "a one-time gather of head counts per sequence" (L562).
    sel_count_local: int32 tensor [B][Hkv / world] of this rank (CPU tensor with gloo, CUDA tensor with nccl: the
    all-gather rides NVLink 5 / NVSwitch; <= 1 KB).  Returns [B][Hkv] in global head order on every rank."""
    if not (dist.is_available() and dist.is_initialized()) or world == 1:
        return sel_count_local.clone()
    parts = [torch.empty_like(sel_count_local) for _ in range(world)]
    dist.all_gather(parts, sel_count_local.contiguous())
    return torch.cat(parts, dim=1)


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
