"""Seeded synthetic workloads shaped like the paper's long-decoding runs.

This module is shared by the CUDA binding's tests/bench and by the oracle's
tests.  It holds NONE of the method's arithmetic (no scoring, softmax, Top-p or
attention): only counter-based random inputs (numpy Philox), bf16 rounding of
those inputs, and page-id permutations.  numpy only; importing it never loads
the CUDA library.

Stands in for: Qwen3-8B decoding 10k-32k-token answers (
budgets L239; bs 32 / sparsity L468).  The five configurations are
BASELINE.json's `configs`; where it is silent the values are the readings of
DESIGN.md (section "Input recipe").
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

PAGE = 16
_T_KV, _T_LATENT, _T_QEPS, _T_KNEW, _T_VNEW, _T_PLANT, _T_PAGES, _T_LEN, _T_MIX = range(1, 10)


def round_bf16(x: np.ndarray) -> np.ndarray:
    """float32 -> nearest bf16 (ties to even), returned widened to float32."""
    b = np.ascontiguousarray(x, np.float32).view(np.uint32)
    r = ((b >> 16) & 1) + np.uint32(0x7FFF)
    return ((b + r) & np.uint32(0xFFFF0000)).view(np.float32)


def bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 holding bf16-representable values -> uint16 bit patterns."""
    return (np.ascontiguousarray(x, np.float32).view(np.uint32) >> 16).astype(np.uint16)


def _rng(seed: int, *ids: int) -> np.random.Generator:
    """Counter-based stream: Philox keyed by (seed, mixed ids)."""
    k = np.uint64(0x9E3779B97F4A7C15)
    with np.errstate(over="ignore"):
        for i in ids:
            k = (k ^ np.uint64(i + 0x632BE59BD9B4E019)) * np.uint64(0xBF58476D1CE4E5B9)
            k ^= k >> np.uint64(29)
    return np.random.Generator(np.random.Philox(key=[np.uint64(seed), k]))


@dataclass
class Workload:
    name: str
    index: int
    B: int
    Hq: int
    Hkv: int
    d: int
    dtype: str                       # "f32" | "bf16": dtype of q, K, V
    n0: np.ndarray                   # [B] prefill lengths
    steps: int
    sink: int
    recent: int
    p: float
    k_cap: int
    cond_cap: int
    l_upper: np.ndarray              # [B]
    max_ctx: int
    score_mode: np.ndarray           # [Hkv] uint8, 0 RAW / 1 ACCUM / 2 SNAPKV
    tau_lo: float
    tau_hi: float
    planted: float = 0.05            # fraction of planted heavy hitters
    mix_new_keys: bool = False       # config 3: new key = 0.7 g + 0.3 k_j, j in HH_h
    structured: bool = True          # False: config 0 (iid, per-q-head tau, key 0 x8)
    l_lower: np.ndarray = None       # [B]
    accum_window: int = 32
    pool_kernel: int = 0             # SNAPKV max-pool window (odd; 0: no SNAPKV head)
    cond_merge: int = 0              # 1: condensed-tier evictees are merged (Appendix G) instead of dropped
    contiguous_pages: bool = False   # diagnostic: identity page ids instead of the seeded permutations (L460)
    head_offset: int = 0             # KV-head (tensor-parallel) shard: this workload holds KV heads [head_offset,
    Hkv_total: int = 0               # head_offset + Hkv) of a batch with Hkv_total heads (0: not a shard) -- same data
                                     # per (sequence, head) as the unsharded workload
    seed: int = 0
    temperature: np.ndarray = field(default=None)  # [B][Hkv] calibration T (reading C10: 1)

    def __post_init__(self):
        self._memo = {}
        self.seed = 28831000 + self.index
        if self.l_lower is None:
            self.l_lower = np.zeros(self.B, np.int32)
        if self.temperature is None:
            self.temperature = np.ones((self.B, self.Hkv), np.float32)
        assert self.max_ctx % PAGE == 0 and self.k_cap % PAGE == 0

    G = property(lambda s: s.Hq // s.Hkv)
    sm_scale = property(lambda s: np.float32(1.0 / np.sqrt(s.d)))
    pages_per_unit = property(lambda s: s.max_ctx // PAGE)
    sel_pages_per_unit = property(lambda s: s.k_cap // PAGE)

    def _round(self, x):
        return round_bf16(x) if self.dtype == "bf16" else np.ascontiguousarray(x, np.float32)

    # ---- latent structure per (b, KV head) ---------------------------------------------
    def latent(self, b: int, h: int):
        """(q_bar[d], u_hat[d], tau): persistent query direction and logit temperature."""
        key = ("latent", self.seed, b, h, self.d, self.tau_lo, self.tau_hi, self.head_offset)
        if key not in self._memo:
            g = _rng(self.seed, _T_LATENT, b, h + self.head_offset)
            qb = g.standard_normal(self.d).astype(np.float32)
            tau = np.float32(np.exp(g.uniform(np.log(self.tau_lo), np.log(self.tau_hi))))
            self._memo[key] = (qb, qb / np.linalg.norm(qb), tau)
        return self._memo[key]

    def _prefill_heavy_hitters(self, b: int, h: int) -> np.ndarray:
        """Positions of the planted heavy hitters of the prefill (memoised: a pure function of the seed and shape)."""
        key = ("hh", self.seed, b, h, int(self.n0[b]), self.planted, self.head_offset)
        if key not in self._memo:
            self._memo[key] = np.flatnonzero(self.planted_mask(b, h, 0, int(self.n0[b])))
        return self._memo[key]

    def planted_mask(self, b: int, h: int, lo: int, hi: int) -> np.ndarray:
        """Which positions in [lo, hi) carry a planted heavy hitter (data-only rule)."""
        if not self.structured or self.planted <= 0:
            return np.zeros(hi - lo, bool)
        out = np.empty(hi - lo, bool)
        blk = 4096
        for s in range(lo // blk, (hi + blk - 1) // blk):
            m = _rng(self.seed, _T_PLANT, b, h + self.head_offset, s).random(blk) < self.planted
            a, e = max(lo, s * blk), min(hi, (s + 1) * blk)
            out[a - lo:e - lo] = m[a - s * blk:e - s * blk]
        return out

    def _plant(self, rows: np.ndarray, mask: np.ndarray, u_hat: np.ndarray) -> np.ndarray:
        """k = |g| (0.8 u + 0.6 g_perp_hat): cosine 0.8 to the latent direction."""
        if mask.any():
            g = rows[mask].astype(np.float64)
            u = u_hat.astype(np.float64)
            perp = g - np.outer(g @ u, u)
            perp /= np.linalg.norm(perp, axis=1, keepdims=True)
            nrm = np.linalg.norm(g, axis=1, keepdims=True)
            rows[mask] = (nrm * (0.8 * u[None, :] + 0.6 * perp)).astype(np.float32)
        return rows

    # ---- prefill KV of one unit -----------------------------------------------------------
    def prefill_unit(self, b: int, h: int):
        """(K0, V0) float32 [n0[b]][d], already rounded to the workload dtype."""
        n = int(self.n0[b])
        g = _rng(self.seed, _T_KV, b, h + self.head_offset)
        K = g.standard_normal((n, self.d), dtype=np.float32)
        V = g.standard_normal((n, self.d), dtype=np.float32)
        if self.structured:
            _, u_hat, _ = self.latent(b, h)
            K = self._plant(K, self.planted_mask(b, h, 0, n), u_hat)
        else:
            K[0] *= 8.0                                  # config 0: key at pos 0 scaled x8 (sink)
        return self._round(K), self._round(V)

    # ---- per-step inputs ---------------------------------------------------------------------
    def step_q(self, t: int) -> np.ndarray:
        """q [B][Hq][d] of decode step t (float32, rounded to the workload dtype)."""
        ht = self.Hkv_total or self.Hkv          # a head shard draws the whole batch's stream and keeps its heads
        eps = _rng(self.seed, _T_QEPS, t).standard_normal((self.B, ht * self.G, self.d), dtype=np.float32)
        eps = np.ascontiguousarray(eps[:, self.head_offset * self.G:(self.head_offset + self.Hkv) * self.G])
        q = np.empty_like(eps)
        if self.structured:
            for b in range(self.B):
                for h in range(self.Hkv):
                    qb, _, tau = self.latent(b, h)
                    sl = slice(h * self.G, (h + 1) * self.G)
                    q[b, sl] = tau * (np.float32(0.9) * qb[None, :] + np.float32(np.sqrt(0.19)) * eps[b, sl])
        else:
            gq = _rng(self.seed, _T_LATENT, 0)
            tau_g = np.exp(gq.uniform(np.log(self.tau_lo), np.log(self.tau_hi), size=(self.B, self.Hq)))
            q = eps * tau_g[..., None].astype(np.float32)
        return self._round(q)

    def step_kv(self, t: int, prefill_K=None):
        """(k_new, v_new) [B][Hkv][d] appended at decode step t (position n0[b]+t).

        prefill_K: dict (b,h)->K0, needed only when mix_new_keys (config 3)."""
        ht, h0 = self.Hkv_total or self.Hkv, self.head_offset
        k = _rng(self.seed, _T_KNEW, t).standard_normal((self.B, ht, self.d), dtype=np.float32)[:, h0:h0 + self.Hkv].copy()
        v = _rng(self.seed, _T_VNEW, t).standard_normal((self.B, ht, self.d), dtype=np.float32)[:, h0:h0 + self.Hkv].copy()
        if self.structured:
            mixr = _rng(self.seed, _T_MIX, t).random((self.B, ht))[:, h0:h0 + self.Hkv]
            for b in range(self.B):
                pos = int(self.n0[b]) + t
                for h in range(self.Hkv):
                    if self.mix_new_keys:
                        hh = self._prefill_heavy_hitters(b, h)
                        if len(hh):
                            j = hh[int(mixr[b, h] * len(hh)) % len(hh)]
                            k[b, h] = np.float32(0.7) * k[b, h] + np.float32(0.3) * prefill_K[(b, h)][j]
                    elif self.planted_mask(b, h, pos, pos + 1)[0]:
                        _, u_hat, _ = self.latent(b, h)
                        k[b, h] = self._plant(k[b, h][None, :].copy(), np.array([True]), u_hat)[0]
        return self._round(k), self._round(v)

    # ---- physical page ids ("requests are assigned random block indices", L460) ----------------
    def page_tables(self):
        """base_table [B][Hkv][max_ctx/16], sel_pages [B][Hkv][k_cap/16]: seeded permutations."""
        nb = self.B * self.Hkv * self.pages_per_unit
        ns = self.B * self.Hkv * self.sel_pages_per_unit
        if self.contiguous_pages:
            return (np.arange(nb, dtype=np.int32).reshape(self.B, self.Hkv, self.pages_per_unit),
                    np.arange(ns, dtype=np.int32).reshape(self.B, self.Hkv, self.sel_pages_per_unit))
        g = _rng(self.seed, _T_PAGES, self.head_offset) if self.head_offset else _rng(self.seed, _T_PAGES)
        base = g.permutation(nb).astype(np.int32).reshape(self.B, self.Hkv, self.pages_per_unit)
        sel = g.permutation(ns).astype(np.int32).reshape(self.B, self.Hkv, self.sel_pages_per_unit)
        return base, sel


def make_workload(index: int, **over) -> Workload:
    """BASELINE.json configs[index]; keyword overrides shrink a config for tests."""
    i32 = lambda *v: np.array(v, np.int32)
    if index == 0:
        kw = dict(name="c0-tiny-fp32", B=1, Hq=4, Hkv=1, d=64, dtype="f32", n0=i32(512), steps=8, sink=4, recent=64,
                  p=0.9, k_cap=512, cond_cap=16, l_upper=i32(448), max_ctx=528, score_mode=np.zeros(1, np.uint8),
                  tau_lo=0.5, tau_hi=4.0, structured=False)
    elif index == 1:
        kw = dict(name="c1-llama8b-16k", B=1, Hq=32, Hkv=8, d=128, dtype="bf16", n0=i32(16384), steps=64, sink=4,
                  recent=128, p=0.95, k_cap=4096, cond_cap=256, l_upper=i32(16284), max_ctx=16448,
                  score_mode=np.zeros(8, np.uint8), tau_lo=0.25, tau_hi=8.0)
    elif index == 2:
        B = over.get("B", 16)
        n0 = _rng(28831002, _T_LEN).integers(4096, 32768, size=16, endpoint=True).astype(np.int32)[:B]
        kw = dict(name="c2-batched-32k", B=B, Hq=32, Hkv=8, d=128, dtype="bf16", n0=n0, steps=256, sink=4,
                  recent=128, p=0.95, k_cap=8192, cond_cap=256, l_upper=(n0 - 132).astype(np.int32), max_ctx=33024,
                  score_mode=np.zeros(8, np.uint8), tau_lo=0.25, tau_hi=8.0)
    elif index == 3:
        B = over.get("B", 32)
        kw = dict(name="c3-longgen-b32", B=B, Hq=28, Hkv=4, d=128, dtype="bf16", n0=np.full(B, 1024, np.int32),
                  steps=11264, sink=4, recent=256, p=0.9, k_cap=3072, cond_cap=256,
                  l_upper=np.full(B, 8192, np.int32), max_ctx=12288, score_mode=np.zeros(4, np.uint8),
                  tau_lo=0.25, tau_hi=8.0, mix_new_keys=True)
    elif index == 4:
        B = over.get("B", 8)
        kw = dict(name="c4-hetero-64k", B=B, Hq=40, Hkv=8, d=128, dtype="bf16", n0=np.full(B, 65536, np.int32),
                  steps=128, sink=4, recent=128, p=0.95, k_cap=16384, cond_cap=256,
                  l_upper=np.full(B, 65468, np.int32), max_ctx=65664,
                  score_mode=np.array([0, 0, 0, 0, 1, 1, 1, 1], np.uint8), tau_lo=0.25, tau_hi=8.0)
    else:
        raise ValueError(index)
    kw.update(over)
    return Workload(index=index, **kw)
