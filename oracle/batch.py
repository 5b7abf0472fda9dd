"""TEST INFRASTRUCTURE ONLY -- the CPU oracle over a whole synthetic Workload (all (b, h) units).

TEST INFRASTRUCTURE: imports oracle/ and the input generator only, never the CUDA binding.
"""
from __future__ import annotations

import numpy as np

from oracle.oracle import OracleConfig, Unit, decode_step_batch
from workloads.synth import Workload


class OracleBatch:
    def __init__(self, wl: Workload, prefill: dict):
        self.wl = wl
        self.cfg = OracleConfig(G=wl.G, d=wl.d, max_ctx=wl.max_ctx, sink=wl.sink, recent=wl.recent, k_cap=wl.k_cap,
                                cond_cap=wl.cond_cap, accum_window=wl.accum_window, sm_scale=float(wl.sm_scale),
                                pool_kernel=wl.pool_kernel, cond_merge=wl.cond_merge,
                                kv_bf16=int(wl.dtype == "bf16"))
        self.units = []
        for b in range(wl.B):
            for h in range(wl.Hkv):
                K0, V0 = prefill[(b, h)]
                self.units.append(Unit(self.cfg, K0, V0, l_upper=int(wl.l_upper[b]), l_lower=int(wl.l_lower[b]),
                                       T=float(wl.temperature[b, h]), score_mode=int(wl.score_mode[h])))
        self.threads = 1

    def step(self, q: np.ndarray, k_new: np.ndarray, v_new: np.ndarray, p: float, do_select: bool = True):
        """q [B][Hq][d], k_new / v_new [B][Hkv][d] (float32, already rounded to the workload dtype)."""
        wl = self.wl
        self.threads = decode_step_batch(self.units, q.reshape(wl.B * wl.Hkv, wl.G, wl.d),
                                         k_new.reshape(wl.B * wl.Hkv, wl.d), v_new.reshape(wl.B * wl.Hkv, wl.d),
                                         p, do_select)

    # ---- stacked views ------------------------------------------------------------------------
    def out(self) -> np.ndarray:
        return np.stack([u.out for u in self.units]).reshape(self.wl.B, self.wl.Hq, self.wl.d)

    def lse(self) -> np.ndarray:
        return np.stack([u.lse for u in self.units]).reshape(self.wl.B, self.wl.Hq)

    def sel_count(self) -> np.ndarray:
        return np.array([u.sel_count for u in self.units], np.int32)

    def sel_idx(self) -> np.ndarray:
        return np.stack([u.sel_idx for u in self.units])

    def cond_count(self) -> np.ndarray:
        return np.array([u.cond_count for u in self.units], np.int32)

    def ctx_len(self) -> np.ndarray:
        return np.array([self.units[b * self.wl.Hkv].n for b in range(self.wl.B)], np.int32)

    def c_lo(self) -> np.ndarray:
        return np.array([self.units[b * self.wl.Hkv].c_lo for b in range(self.wl.B)], np.int32)

    def dense_lo(self) -> np.ndarray:
        return np.array([self.units[b * self.wl.Hkv].dense_lo for b in range(self.wl.B)], np.int32)
