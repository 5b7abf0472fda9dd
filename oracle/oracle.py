"""TEST INFRASTRUCTURE ONLY -- ctypes view of oracle/hardkv_oracle.c.

This module marshals numpy arrays into the C oracle; it contains none of the
method's arithmetic.  It does not import the CUDA package.
Cites: PAPER.md L78 (pipeline), L108 (Top-p), L735-762 (attention states).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# HARDKV_ORACLE_SANITIZE=1 (tests/test_oracle_sanitized.py): the same source built with AddressSanitizer + UBSan into a
# second library; the process must run with libasan preloaded.
_SANITIZE = os.environ.get("HARDKV_ORACLE_SANITIZE") == "1"
_SO = os.path.join(_HERE, "libhardkv_oracle_asan.so" if _SANITIZE else "libhardkv_oracle.so")
_SRC = os.path.join(_HERE, "hardkv_oracle.c")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (never tuned; it is the plain definition)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < max(
        os.path.getmtime(_SRC), os.path.getmtime(os.path.join(_HERE, "hardkv_oracle.h"))
    ):
        flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"] if _SANITIZE else ["-O2"]
        subprocess.check_call(
            ["gcc", *flags, "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", _SO, _SRC, "-lm"]
        )
    return _SO


class HkoConfig(C.Structure):
    _fields_ = [
        ("G", C.c_int32), ("d", C.c_int32), ("page", C.c_int32), ("max_ctx", C.c_int32),
        ("sink", C.c_int32), ("recent", C.c_int32), ("k_cap", C.c_int32), ("cond_cap", C.c_int32),
        ("accum_window", C.c_int32), ("sm_scale", C.c_float), ("pool_kernel", C.c_int32),
        ("cond_merge", C.c_int32), ("kv_bf16", C.c_int32),
    ]


_F = C.POINTER(C.c_float)
_I = C.POINTER(C.c_int32)


class HkoUnit(C.Structure):
    _fields_ = [
        ("K", _F), ("V", _F),
        ("n", C.c_int32), ("c_lo", C.c_int32), ("dense_lo", C.c_int32), ("l_lower", C.c_int32), ("l_upper", C.c_int32),
        ("votes", _I),
        ("cond_k", _F), ("cond_v", _F), ("cond_pos", _I), ("cond_votes", _I), ("cond_count", C.c_int32),
        ("score_mode", C.c_int32), ("T", C.c_float),
        ("acc", _F), ("ring", _F), ("ring_slot", C.c_int32),
        ("logits", _F), ("probs", _F),
        ("sel_idx", _I), ("sel_count", C.c_int32), ("k_topp", C.c_int32), ("tau_bits", C.c_uint32),
        ("sel_k", _F), ("sel_v", _F), ("out", _F), ("lse", _F),
        ("qcache", _F), ("qc_count", C.c_int32), ("qc_slot", C.c_int32),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        cp, up = C.POINTER(HkoConfig), C.POINTER(HkoUnit)
        _lib.hko_append.argtypes = [cp, up, _F, _F]
        _lib.hko_retire.argtypes = [cp, up]
        _lib.hko_retire.restype = C.c_int
        _lib.hko_retire_q.argtypes = [cp, up, _F]
        _lib.hko_retire_q.restype = C.c_int
        _lib.hko_score.argtypes = [cp, up, _F]
        _lib.hko_qcache_push.argtypes = [cp, up, _F]
        _lib.hko_qcache_push.restype = None
        _lib.hko_calibrate.argtypes = [cp, up]
        _lib.hko_solve_temperature.argtypes = [cp, up, C.c_float, C.c_float, C.c_float, C.c_float, C.c_int,
                                               C.POINTER(C.c_double)]
        _lib.hko_solve_temperature.restype = C.c_int
        _lib.hko_topp_select.argtypes = [cp, up, C.c_float, C.c_int]
        _lib.hko_rewrite.argtypes = [cp, up]
        _lib.hko_attend.argtypes = [cp, up, _F]
        _lib.hko_decode_step.argtypes = [cp, up, _F, _F, _F, C.c_float, C.c_int]
        _lib.hko_decode_step_batch.argtypes = [cp, up, C.c_int32, _F, _F, _F, C.c_float, C.c_int]
        _lib.hko_decode_step_batch.restype = C.c_int
        _D = C.POINTER(C.c_double)
        _lib.hko_state_of_set.argtypes = [cp, _F, _F, _F, _I, C.c_int32, _D, _D, _D]
        _lib.hko_merge.argtypes = [C.c_int32, _D, _D, _D, _D, C.c_double, C.c_double]
        _lib.hko_sel_table.argtypes = [cp, up, _I, _I]
        _lib.hko_sel_mask.argtypes = [cp, up, C.POINTER(C.c_uint8)]
        for f in ("hko_append", "hko_score", "hko_calibrate", "hko_topp_select", "hko_rewrite", "hko_attend",
                  "hko_decode_step", "hko_state_of_set", "hko_merge", "hko_sel_table", "hko_sel_mask"):
            getattr(_lib, f).restype = None
    return _lib


def _fp(a: np.ndarray):
    assert a.dtype == np.float32 and a.flags.c_contiguous
    return a.ctypes.data_as(_F)


def _ip(a: np.ndarray):
    assert a.dtype == np.int32 and a.flags.c_contiguous
    return a.ctypes.data_as(_I)


@dataclass
class OracleConfig:
    G: int
    d: int
    max_ctx: int
    sink: int
    recent: int
    k_cap: int
    cond_cap: int
    page: int = 16
    accum_window: int = 32
    sm_scale: float | None = None
    pool_kernel: int = 0
    cond_merge: int = 0
    kv_bf16: int = 0

    def c(self) -> HkoConfig:
        s = self.sm_scale if self.sm_scale is not None else 1.0 / float(np.sqrt(self.d))
        return HkoConfig(self.G, self.d, self.page, self.max_ctx, self.sink, self.recent, self.k_cap,
                         self.cond_cap, self.accum_window, np.float32(s), self.pool_kernel,
                         self.cond_merge, self.kv_bf16)


class Unit:
    """State of one (b, h) pair: numpy arrays owned here, viewed by the C struct."""

    def __init__(self, cfg: OracleConfig, K0: np.ndarray, V0: np.ndarray, l_upper: int, l_lower: int = 0,
                 T: float = 1.0, score_mode: int = 0):
        self.cfg = cfg
        n0 = K0.shape[0]
        d, mc = cfg.d, cfg.max_ctx
        assert K0.shape == (n0, d) and V0.shape == (n0, d) and n0 <= mc
        self.K = np.zeros((mc, d), np.float32); self.K[:n0] = K0
        self.V = np.zeros((mc, d), np.float32); self.V[:n0] = V0
        self.votes = np.zeros(mc, np.int32)
        self.cond_k = np.zeros((max(cfg.cond_cap, 1), d), np.float32)
        self.cond_v = np.zeros((max(cfg.cond_cap, 1), d), np.float32)
        self.cond_pos = np.full(max(cfg.cond_cap, 1), -1, np.int32)
        self.cond_votes = np.zeros(max(cfg.cond_cap, 1), np.int32)
        self.acc = np.zeros(mc, np.float32) if score_mode == 1 else None
        self.ring = np.zeros((cfg.accum_window, mc), np.float32) if score_mode == 1 else None
        self.logits = np.zeros((cfg.G, mc), np.float32)
        self.probs = np.zeros(mc, np.float32)
        self.sel_idx = np.full(max(cfg.k_cap, 1), -1, np.int32)
        self.sel_k = np.zeros((max(cfg.k_cap, 1), d), np.float32)
        self.sel_v = np.zeros((max(cfg.k_cap, 1), d), np.float32)
        self.out = np.zeros((cfg.G, d), np.float32)
        self.lse = np.zeros(cfg.G, np.float32)
        self.ccfg = cfg.c()
        self.u = HkoUnit()
        u = self.u
        u.K, u.V = _fp(self.K), _fp(self.V)
        u.n, u.c_lo, u.l_lower, u.l_upper = n0, cfg.sink, l_lower, l_upper
        u.dense_lo = max(min(cfg.sink, n0), n0 - cfg.recent)
        u.votes = _ip(self.votes)
        u.cond_k, u.cond_v = _fp(self.cond_k), _fp(self.cond_v)
        u.cond_pos, u.cond_votes, u.cond_count = _ip(self.cond_pos), _ip(self.cond_votes), 0
        u.score_mode, u.T = score_mode, np.float32(T)
        if score_mode == 1:
            u.acc, u.ring = _fp(self.acc), _fp(self.ring)
        u.ring_slot = 0
        u.logits, u.probs = _fp(self.logits), _fp(self.probs)
        u.sel_idx, u.sel_count, u.k_topp, u.tau_bits = _ip(self.sel_idx), 0, 0, 0
        u.sel_k, u.sel_v, u.out, u.lse = _fp(self.sel_k), _fp(self.sel_v), _fp(self.out), _fp(self.lse)
        self.qcache = np.zeros((max(cfg.accum_window, 1), cfg.G, d), np.float32) if score_mode == 3 else None
        if score_mode == 3:
            u.qcache = _fp(self.qcache)
        u.qc_count, u.qc_slot = 0, 0

    # --- scalars -------------------------------------------------------------------
    n = property(lambda s: s.u.n)
    c_lo = property(lambda s: s.u.c_lo)
    dense_lo = property(lambda s: s.u.dense_lo)
    sel_count = property(lambda s: s.u.sel_count)
    k_topp = property(lambda s: s.u.k_topp)
    cond_count = property(lambda s: s.u.cond_count)
    tau_bits = property(lambda s: s.u.tau_bits)

    @property
    def pool(self) -> tuple[int, int]:
        hi = max(self.u.n - self.cfg.recent, self.u.c_lo)
        return self.u.c_lo, hi

    # --- stages ----------------------------------------------------------------------
    def append(self, k_new, v_new):
        lib().hko_append(C.byref(self.ccfg), C.byref(self.u), _fp(_f32(k_new)), _fp(_f32(v_new)))

    def retire(self) -> int:
        return lib().hko_retire(C.byref(self.ccfg), C.byref(self.u))

    def retire_q(self, q) -> int:
        return lib().hko_retire_q(C.byref(self.ccfg), C.byref(self.u), _fp(_f32(q)))

    def qcache_push(self, q):
        lib().hko_qcache_push(C.byref(self.ccfg), C.byref(self.u), _fp(_f32(q)))

    def score(self, q):
        lib().hko_score(C.byref(self.ccfg), C.byref(self.u), _fp(_f32(q)))

    def calibrate(self):
        lib().hko_calibrate(C.byref(self.ccfg), C.byref(self.u))

    def solve_temperature(self, p: float, t_min: float = 0.03125, t_max: float = 32.0, eps: float = 1e-4,
                          max_iter: int = 40) -> tuple[int, float]:
        """Algorithm 2 on the logits of the last score(); sets T. Returns (rounds, residual)."""
        r = C.c_double()
        it = lib().hko_solve_temperature(C.byref(self.ccfg), C.byref(self.u), np.float32(p), np.float32(t_min),
                                         np.float32(t_max), np.float32(eps), int(max_iter), C.byref(r))
        return it, r.value

    T = property(lambda s: float(s.u.T))

    def topp_select(self, p: float, count_votes: bool = True):
        lib().hko_topp_select(C.byref(self.ccfg), C.byref(self.u), np.float32(p), int(count_votes))

    def rewrite(self):
        lib().hko_rewrite(C.byref(self.ccfg), C.byref(self.u))

    def attend(self, q):
        lib().hko_attend(C.byref(self.ccfg), C.byref(self.u), _fp(_f32(q)))

    def decode_step(self, q, k_new, v_new, p: float, do_select: bool = True):
        lib().hko_decode_step(C.byref(self.ccfg), C.byref(self.u), _fp(_f32(q)), _fp(_f32(k_new)),
                              _fp(_f32(v_new)), np.float32(p), int(do_select))

    def sel_table(self, sel_pages: np.ndarray) -> np.ndarray:
        out = np.empty(self.cfg.k_cap // self.cfg.page, np.int32)
        sp = np.ascontiguousarray(sel_pages, np.int32)
        lib().hko_sel_table(C.byref(self.ccfg), C.byref(self.u), _ip(sp), _ip(out))
        return out

    def sel_mask(self) -> np.ndarray:
        out = np.empty(self.cfg.max_ctx // 8, np.uint8)
        lib().hko_sel_mask(C.byref(self.ccfg), C.byref(self.u), out.ctypes.data_as(C.POINTER(C.c_uint8)))
        return out


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def decode_step_batch(units: list[Unit], q: np.ndarray, k_new: np.ndarray, v_new: np.ndarray, p: float,
                      do_select: bool = True) -> int:
    """q [n_units][G][d], k_new/v_new [n_units][d]; OpenMP over units. Returns threads used."""
    arr = (HkoUnit * len(units))(*[u.u for u in units])
    q, k_new, v_new = _f32(q), _f32(k_new), _f32(v_new)
    nt = lib().hko_decode_step_batch(C.byref(units[0].ccfg), arr, len(units), _fp(q), _fp(k_new), _fp(v_new),
                                     np.float32(p), int(do_select))
    for u, cu in zip(units, arr):   # copy the scalar fields back (arrays are shared by pointer)
        for f in ("n", "c_lo", "dense_lo", "cond_count", "ring_slot", "qc_count", "qc_slot", "sel_count", "k_topp", "tau_bits"):
            setattr(u.u, f, getattr(cu, f))
    return nt


def topp_select_row(cfg: OracleConfig, probs: np.ndarray, lo: int, hi: int, l_lower: int, p: float):
    """hko_topp_select on a caller-supplied probability row probs[max_ctx] with pool [lo, hi).
    Returns (sel_idx[:k] ascending, k, k_topp, tau_bits).  Marshalling only: votes are not counted."""
    probs = np.ascontiguousarray(probs, np.float32)
    sel = np.full(max(cfg.k_cap, 1), -1, np.int32)
    u = HkoUnit()
    u.n, u.c_lo, u.l_lower = hi + cfg.recent, lo, l_lower
    u.probs, u.sel_idx = _fp(probs), _ip(sel)
    cc = cfg.c()
    lib().hko_topp_select(C.byref(cc), C.byref(u), np.float32(p), 0)
    return sel[:u.sel_count].copy(), int(u.sel_count), int(u.k_topp), int(u.tau_bits)


def state_of_set(cfg: OracleConfig, q_g, K, V, idx=None):
    """(o[d], m, l) of Eq. 5 for rows idx of K/V (float32 [rows][d])."""
    K, V, q_g = _f32(K), _f32(V), _f32(q_g)
    o = np.zeros(cfg.d, np.float64); m = C.c_double(); l = C.c_double()
    if idx is None:
        ip, n = None, K.shape[0]
    else:
        idx = np.ascontiguousarray(idx, np.int32); ip, n = _ip(idx), len(idx)
    cc = cfg.c()
    lib().hko_state_of_set(C.byref(cc), _fp(q_g), _fp(K), _fp(V), ip, n,
                           o.ctypes.data_as(C.POINTER(C.c_double)), C.byref(m), C.byref(l))
    return o, m.value, l.value


def merge(a, b):
    """Eq. 6 on two (o, m, l) states; returns the merged state."""
    o = np.array(a[0], np.float64); m = C.c_double(a[1]); l = C.c_double(a[2])
    ob = np.ascontiguousarray(b[0], np.float64)
    D = C.POINTER(C.c_double)
    lib().hko_merge(len(o), o.ctypes.data_as(D), C.byref(m), C.byref(l), ob.ctypes.data_as(D), b[1], b[2])
    return o, m.value, l.value
