"""Byte accounting of one layer-step.

numpy only; imports neither the CUDA binding nor the oracle (both legs of bench.py use it to turn a
measured time into GB/s of the same B_min).  It holds none of the method's arithmetic.
"""
from __future__ import annotations

import numpy as np


def algorithmic_bytes(wl, ctx_len, c_lo, sel_count, cond_count) -> dict:
    """B_min of one layer-step: per (b, h), with R = bytes of one K (or V) row,
    R*[N_c (K scan) + 2k (read selected K,V) + 2k (write selected tier) + 2(s + W + cond)] + 4k (indices).
    ctx_len, c_lo: [B] AFTER the step's append/retire; sel_count, cond_count: [B*Hkv]."""
    R = wl.d * (2 if wl.dtype == "bf16" else 4)
    n = np.repeat(np.asarray(ctx_len, np.int64), wl.Hkv)
    lo = np.repeat(np.asarray(c_lo, np.int64), wl.Hkv)
    k = np.asarray(sel_count, np.int64)
    cc = np.asarray(cond_count, np.int64)
    N_c = np.maximum(n - wl.recent - lo, 0)
    s_end = np.minimum(wl.sink, n)
    dense = s_end + (n - np.maximum(n - wl.recent, s_end))
    score = R * N_c
    attend = R * (2 * k + 2 * (dense + cc)) + 4 * k
    rewrite_write = R * 2 * k
    return {"score": int(score.sum()), "attend": int(attend.sum()), "rewrite_write": int(rewrite_write.sum()),
            "total": int((score + attend + rewrite_write).sum()),
            # implementation traffic of the select stage (not part of B_min): logits in, probs out, indices out
            "select_bytes": int(((4 * wl.G + 4) * N_c + 4 * k).sum()),
            "dense_attention_bytes": int((2 * R * n).sum()),
            "mean_k": float(k.mean()), "max_k": int(k.max()), "mean_pool": float(N_c.mean())}
