"""Device-state construction for a synthetic Workload (tests, smoke, bench).

Allocation and host->device marshalling only (torch tensors, page scatter); none of the
method's arithmetic lives here.  Layouts are those of include/hardkv.h.
"""
from __future__ import annotations

import dataclasses

import numpy as np
import torch

from . import hardkv
from workloads.synth import PAGE, Workload


def torch_dtype(wl: Workload):
    return torch.bfloat16 if wl.dtype == "bf16" else torch.float32


def make_engine(wl: Workload, device="cuda:0", want_accum=None, reuse_max: int = 0) -> hardkv.HardKV:
    accum = bool(np.any((wl.score_mode == 1) | (wl.score_mode == 3))) if want_accum is None else want_accum
    return hardkv.HardKV(batch=wl.B, num_q_heads=wl.Hq, num_kv_heads=wl.Hkv, head_dim=wl.d, max_ctx=wl.max_ctx,
                         sink=wl.sink, recent=wl.recent, k_cap=wl.k_cap, cond_cap=wl.cond_cap,
                         kv_dtype=hardkv.BF16 if wl.dtype == "bf16" else hardkv.F32,
                         accum_window=wl.accum_window if accum else 0, sm_scale=float(wl.sm_scale),
                         pool_kernel=wl.pool_kernel, cond_merge=wl.cond_merge, reuse_max=reuse_max, device=device)


def to_dev(x: np.ndarray, wl: Workload, device="cuda:0") -> torch.Tensor:
    """float32 host array holding values representable in the workload dtype -> device tensor."""
    return torch.from_numpy(np.ascontiguousarray(x, np.float32)).to(device).to(torch_dtype(wl)).contiguous()


def make_state(wl: Workload, device="cuda:0", prefill=None, want_mask=False, layers: int = 1, retain=None,
               layer_seeds=None):
    """Allocate and fill the device state of `layers` layers (page tables shared by all layers, L207-209).

    prefill: optional dict (b, h) -> (K0, V0) float32; generated from wl when absent.
    retain: optional set of (b, h): only these units' host prefill arrays are kept in the returned dict
    (full-size tests that sample units; the 64k-context configs would otherwise hold GBs of host memory).
    layer_seeds: optional list of `layers` seeds: layer l is filled from the workload re-seeded with layer_seeds[l]
    (independent data per layer; the returned dict is then keyed (l, b, h)).
    Returns (list of DeviceState, prefill dict or None).  Without layer_seeds, layers l > 0 reuse layer 0's prefill
    values rolled by l rows (distinct addresses and data; the same statistics).
    """
    B, Hkv, Hq, d, mc = wl.B, wl.Hkv, wl.Hq, wl.d, wl.max_ctx
    units = B * Hkv
    ppu, spu = wl.pages_per_unit, wl.sel_pages_per_unit
    dt = torch_dtype(wl)
    base_np, sel_np = wl.page_tables()
    base_table = torch.from_numpy(base_np).to(device)
    sel_pages = torch.from_numpy(sel_np).to(device)
    i32 = lambda a: torch.from_numpy(np.ascontiguousarray(a, np.int32)).to(device)
    accum = bool(np.any(wl.score_mode == 1))
    qcache = bool(np.any(wl.score_mode == 3))
    keep = {} if prefill is None else prefill
    states = []
    for layer in range(layers):
        k_pool = torch.zeros(units * ppu, PAGE, d, dtype=dt, device=device)
        v_pool = torch.zeros(units * ppu, PAGE, d, dtype=dt, device=device)
        for b in range(B):
            for h in range(Hkv):
                if layer_seeds is not None:
                    wl_l = dataclasses.replace(wl)
                    wl_l.seed = layer_seeds[layer]
                    K0, V0 = wl_l.prefill_unit(b, h)
                    if retain is None or (b, h) in retain:
                        keep[(layer, b, h)] = (K0, V0)
                    kd, vd = to_dev(K0, wl, device), to_dev(V0, wl, device)
                elif layer == 0:
                    if (b, h) not in keep:
                        K0, V0 = wl.prefill_unit(b, h)
                        if retain is None or (b, h) in retain:
                            keep[(b, h)] = (K0, V0)
                    else:
                        K0, V0 = keep[(b, h)]
                    kd, vd = to_dev(K0, wl, device), to_dev(V0, wl, device)
                else:
                    src = states[0]
                    tab0 = base_table[b, h].long()
                    n0 = int(wl.n0[b])
                    kd = torch.roll(src.k_pool[tab0].reshape(mc, d)[:n0], layer, 0)
                    vd = torch.roll(src.v_pool[tab0].reshape(mc, d)[:n0], layer, 0)
                n0 = kd.shape[0]
                pad = torch.zeros(mc, d, dtype=dt, device=device)
                pad[:n0] = kd
                k_pool[base_table[b, h].long()] = pad.view(ppu, PAGE, d)
                pad = torch.zeros(mc, d, dtype=dt, device=device)
                pad[:n0] = vd
                v_pool[base_table[b, h].long()] = pad.view(ppu, PAGE, d)
        C = max(wl.cond_cap, 1)
        st = hardkv.DeviceState(
            k_pool=k_pool, v_pool=v_pool, base_table=base_table,
            sel_k_pool=torch.zeros(units * spu, PAGE, d, dtype=dt, device=device),
            sel_v_pool=torch.zeros(units * spu, PAGE, d, dtype=dt, device=device), sel_pages=sel_pages,
            cond_k=torch.zeros(units, C, d, dtype=dt, device=device),
            cond_v=torch.zeros(units, C, d, dtype=dt, device=device),
            cond_pos=torch.full((units, C), -1, dtype=torch.int32, device=device),
            cond_votes=torch.zeros(units, C, dtype=torch.int32, device=device),
            cond_count=torch.zeros(units, dtype=torch.int32, device=device),
            ctx_len=i32(wl.n0), c_lo=torch.full((B,), wl.sink, dtype=torch.int32, device=device),
            l_lower=i32(wl.l_lower), l_upper=i32(wl.l_upper),
            votes=torch.zeros(units, mc, dtype=torch.int32, device=device),
            temperature=torch.from_numpy(np.ascontiguousarray(wl.temperature, np.float32)).to(device),
            score_mode=torch.from_numpy(np.ascontiguousarray(wl.score_mode, np.uint8)).to(device),
            acc=torch.zeros(units, mc, dtype=torch.float32, device=device) if accum else None,
            ring=torch.zeros(units, wl.accum_window, mc, dtype=torch.float32, device=device) if accum else None,
            ring_slot=torch.zeros(units, dtype=torch.int32, device=device) if accum else None,
            sel_idx=torch.full((units, wl.k_cap), -1, dtype=torch.int32, device=device),
            sel_count=torch.zeros(units, dtype=torch.int32, device=device),
            sel_table=torch.full((units, spu), -1, dtype=torch.int32, device=device),
            sel_mask=torch.zeros(units, mc // 8, dtype=torch.uint8, device=device) if want_mask else None,
            logits=torch.zeros(B * Hq, mc, dtype=torch.float32, device=device),
            probs=torch.zeros(units, mc, dtype=torch.float32, device=device),
            err_flag=torch.zeros(1, dtype=torch.int32, device=device),
            dense_lo=i32(np.maximum(np.minimum(wl.sink, wl.n0), wl.n0 - wl.recent)),
            qcache=torch.zeros(B, Hq, wl.accum_window, d, dtype=dt, device=device) if qcache else None,
            qc_count=torch.zeros(B, dtype=torch.int32, device=device) if qcache else None,
            qc_slot=torch.zeros(B, dtype=torch.int32, device=device) if qcache else None,
        )
        states.append(st)
    return states, keep


def gather_rows(pool: torch.Tensor, table_unit: torch.Tensor, n: int) -> np.ndarray:
    """Logical rows 0..n-1 of one unit from a paged pool -> float32 host array [n][d]."""
    d = pool.shape[-1]
    return pool[table_unit.long()].reshape(-1, d)[:n].float().cpu().numpy()


_MUTABLE = ["votes", "cond_k", "cond_v", "cond_pos", "cond_votes", "cond_count", "ctx_len", "c_lo", "dense_lo", "sel_idx",
            "sel_count", "sel_table", "acc", "ring", "ring_slot", "qcache", "qc_count", "qc_slot"]


def snapshot(st: hardkv.DeviceState) -> dict:
    """Clone the tensors a decode step mutates (appended KV rows are rewritten identically on a rerun)."""
    return {n: getattr(st, n).clone() for n in _MUTABLE if getattr(st, n) is not None}


def restore(st: hardkv.DeviceState, snap: dict) -> None:
    for n, t in snap.items():
        getattr(st, n).copy_(t)
