"""Thin ctypes binding over libhardkv.so (C ABI: include/hardkv.h).

Argument marshalling only: every step of the path runs in the CUDA kernels of csrc/.  torch is
used for device memory and streams.  There is no CPU fallback: importing this module raises if
the shared library is missing, and every call raises on a non-zero status.
Method names mirror the ABI (PAPER.md L78 pipeline: append -> score -> calibrate + Top-p ->
rewrite -> tiered attention L84).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_SO = os.path.join(_HERE, "libhardkv.so")
_INC = os.path.join(os.path.dirname(_HERE), "include")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


def _sources():
    return [os.path.join(_CSRC, f) for f in sorted(os.listdir(_CSRC))] + [os.path.join(_INC, "hardkv.h")]


def build(force: bool = False) -> str:
    """Compile csrc/hardkv.cu for sm_100a into libhardkv.so (in-tree) if it is missing or stale."""
    stale = force or not os.path.exists(_SO) or os.path.getmtime(_SO) < max(os.path.getmtime(s) for s in _sources())
    if stale:
        subprocess.check_call(["nvcc", *NVCC_FLAGS, "-o", _SO, os.path.join(_CSRC, "hardkv.cu")])
    return _SO


class Config(C.Structure):
    _fields_ = [(n, C.c_int32) for n in (
        "batch", "num_q_heads", "num_kv_heads", "head_dim", "page_size", "max_ctx", "sink", "recent", "k_cap",
        "cond_cap", "accum_window", "kv_dtype")] + [("sm_scale", C.c_float), ("pool_kernel", C.c_int32), ("cond_merge", C.c_int32),
                                        ("reuse_max", C.c_int32)]


_STATE_FIELDS = ["k_pool", "v_pool", "base_table", "sel_k_pool", "sel_v_pool", "sel_pages", "cond_k", "cond_v",
                 "cond_pos", "cond_votes", "cond_count", "ctx_len", "c_lo", "l_lower", "l_upper", "votes",
                 "temperature", "score_mode", "acc", "ring", "ring_slot", "sel_idx", "sel_count", "sel_table",
                 "sel_mask", "logits", "probs", "err_flag", "qcache", "qc_count", "qc_slot", "dense_lo"]


class StateStruct(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in _STATE_FIELDS]


F32, BF16 = 0, 1
STEP_REUSE_TIER, STEP_SELECT_REWRITE, STEP_SELECT_SPARSE, STEP_REUSE_SPARSE = 0, 1, 2, 3   # do_select of decode_step
EXPORTS = ["hardkv_workspace_bytes", "hardkv_create", "hardkv_destroy", "hardkv_status_string",
           "hardkv_set_variant", "hardkv_set_select_geometry", "hardkv_set_overlap", "hardkv_set_timing", "hardkv_set_pdl", "hardkv_append_kv", "hardkv_append_kv_merge", "hardkv_score", "hardkv_score_select", "hardkv_qcache_push", "hardkv_calibrate_topp", "hardkv_solve_temperature",
           "hardkv_topp_select", "hardkv_rewrite", "hardkv_decode_attn", "hardkv_rewrite_attend", "hardkv_sparse_attend",
           "hardkv_decode_step", "hardkv_decode_step_host", "hardkv_launch_count", "hardkv_probe_read_stream",
           "hardkv_decode_attn_noalloc"]


def _load():
    if not os.path.exists(_SO):
        raise ImportError(f"{_SO} is not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(_SO)
    vp, cp, sp = C.c_void_p, C.POINTER(Config), C.POINTER(StateStruct)
    lib.hardkv_workspace_bytes.argtypes = [cp, C.POINTER(C.c_size_t)]
    lib.hardkv_create.argtypes = [cp, vp, C.c_size_t, C.POINTER(vp)]
    lib.hardkv_destroy.argtypes = [vp]
    lib.hardkv_destroy.restype = None
    lib.hardkv_status_string.argtypes = [C.c_int]
    lib.hardkv_status_string.restype = C.c_char_p
    lib.hardkv_set_variant.argtypes = [vp, C.c_int32]
    lib.hardkv_set_select_geometry.argtypes = [vp, C.c_int32, C.c_int32]
    lib.hardkv_set_pdl.argtypes = [vp, C.c_int32]
    lib.hardkv_set_overlap.argtypes = [vp, C.c_int32]
    lib.hardkv_set_timing.argtypes = [vp, vp, C.c_int32]
    lib.hardkv_append_kv.argtypes = [vp, sp, vp, vp, vp]
    lib.hardkv_append_kv_merge.argtypes = [vp, sp, vp, vp, vp, vp]
    lib.hardkv_score.argtypes = [vp, sp, vp, vp]
    lib.hardkv_calibrate_topp.argtypes = [vp, sp, C.c_float, vp]
    lib.hardkv_score_select.argtypes = [vp, sp, vp, C.c_float, vp]
    lib.hardkv_qcache_push.argtypes = [vp, sp, vp, vp]
    lib.hardkv_solve_temperature.argtypes = [vp, sp, C.c_float, C.c_float, C.c_float, C.c_float, C.c_int32, vp]
    lib.hardkv_topp_select.argtypes = [vp, sp, C.c_float, vp]
    lib.hardkv_rewrite.argtypes = [vp, sp, vp]
    lib.hardkv_decode_attn.argtypes = [vp, sp, vp, vp, vp, vp]
    lib.hardkv_rewrite_attend.argtypes = [vp, sp, vp, vp, vp, vp]
    lib.hardkv_sparse_attend.argtypes = [vp, sp, vp, vp, vp, vp]
    lib.hardkv_decode_step.argtypes = [vp, sp, vp, vp, vp, C.c_float, C.c_int32, vp, vp, vp]
    lib.hardkv_decode_step_host.argtypes = [vp, sp, vp, vp, vp, C.c_float, C.c_int32, vp, vp]
    lib.hardkv_probe_read_stream.argtypes = [vp, C.c_size_t, vp]
    lib.hardkv_decode_attn_noalloc.argtypes = [cp, sp, vp, vp, vp, vp]
    lib.hardkv_launch_count.argtypes = [vp]
    lib.hardkv_launch_count.restype = C.c_int64
    for n in EXPORTS:
        if n not in ("hardkv_destroy", "hardkv_status_string", "hardkv_launch_count"):
            getattr(lib, n).restype = C.c_int
    return lib


lib = _load()


class HardKVError(RuntimeError):
    pass


def _check(status: int):
    if status != 0:
        raise HardKVError(f"libhardkv: {lib.hardkv_status_string(status).decode()} (status {status})")


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def probe_read_stream(buf: torch.Tensor):
    """One read-only streaming pass over a CUDA tensor on the current stream (hardkv_probe_read_stream)."""
    assert buf.is_cuda and buf.is_contiguous()
    _check(lib.hardkv_probe_read_stream(_ptr(buf), buf.numel() * buf.element_size(), _stream()))


NOALLOC_SCRATCH_BYTES = 4 << 20   # HARDKV_NOALLOC_SCRATCH_BYTES


def decode_attn_noalloc(cfg: "Config", st: "DeviceState", q, out, lse=None):
    """hardkv_decode_attn_noalloc: decode attention over the tiers of `st` with no ctx and no workspace -- the kernel's
    scratch is the library's static device array (4 MiB; calls that overlap on the GPU race on it, see hardkv.h)."""
    _check(lib.hardkv_decode_attn_noalloc(C.byref(cfg), C.byref(st.struct()), _ptr(q), _ptr(out), _ptr(lse), _stream()))


class DeviceState:
    """Caller-owned device state of one layer: torch tensors named like hardkv_state's fields."""

    def __init__(self, **tensors):
        for n in _STATE_FIELDS:
            setattr(self, n, tensors.get(n))
        self._struct = None

    def __setattr__(self, name, value):
        object.__setattr__(self, name, value)
        if name != "_struct":
            object.__setattr__(self, "_struct", None)   # a field was rebound: the marshalled struct is stale

    def struct(self) -> StateStruct:
        """The marshalled hardkv_state (pointers only), built once and kept until a field is rebound: the per-call
        cost of the binding is then a few ctypes conversions, not 32 attribute walks."""
        s = self._struct
        if s is None:
            s = StateStruct()
            for n in _STATE_FIELDS:
                t = getattr(self, n)
                if t is not None:
                    assert t.is_cuda and t.is_contiguous(), n
                setattr(s, n, None if t is None else t.data_ptr())
            object.__setattr__(self, "_struct", s)
        return s


class HardKV:
    """One hardkv_ctx.  Every method enqueues kernels on torch's current stream and returns at once."""

    def __init__(self, *, batch, num_q_heads, num_kv_heads, head_dim, max_ctx, sink, recent, k_cap, cond_cap,
                 kv_dtype, accum_window=0, page_size=16, sm_scale=0.0, pool_kernel=0, cond_merge=0, reuse_max=0,
                 device="cuda:0"):
        self.cfg = Config(batch, num_q_heads, num_kv_heads, head_dim, page_size, max_ctx, sink, recent, k_cap,
                          cond_cap, accum_window, kv_dtype, sm_scale, pool_kernel, cond_merge, reuse_max)
        nbytes = C.c_size_t()
        _check(lib.hardkv_workspace_bytes(C.byref(self.cfg), C.byref(nbytes)))
        self.workspace = torch.zeros(nbytes.value + 256, dtype=torch.uint8, device=device)
        base = (self.workspace.data_ptr() + 255) & ~255
        self._ctx = C.c_void_p()
        _check(lib.hardkv_create(C.byref(self.cfg), C.c_void_p(base), nbytes.value, C.byref(self._ctx)))

    def __del__(self):
        ctx = getattr(self, "_ctx", None)
        if ctx:
            lib.hardkv_destroy(ctx)
            self._ctx = None

    def set_variant(self, v: int):
        _check(lib.hardkv_set_variant(self._ctx, v))

    def set_select_geometry(self, cluster: int = 0, threads: int = 0):
        _check(lib.hardkv_set_select_geometry(self._ctx, cluster, threads))

    def set_timing(self, slots=None):
        """slots: int64 CUDA tensor [capacity][2] preset to (max, 0) per row, or None to turn the hook off."""
        if slots is None:
            _check(lib.hardkv_set_timing(self._ctx, None, 0))
        else:
            assert slots.is_cuda and slots.is_contiguous() and slots.dtype == torch.int64 and slots.shape[1] == 2
            _check(lib.hardkv_set_timing(self._ctx, _ptr(slots), slots.shape[0]))

    def set_overlap(self, on: bool):
        _check(lib.hardkv_set_overlap(self._ctx, int(on)))

    def set_pdl(self, on: bool):
        _check(lib.hardkv_set_pdl(self._ctx, int(on)))

    def append_kv(self, st: DeviceState, k_new, v_new):
        _check(lib.hardkv_append_kv(self._ctx, C.byref(st.struct()), _ptr(k_new), _ptr(v_new), _stream()))

    def append_kv_merge(self, st: DeviceState, k_new, v_new, q):
        _check(lib.hardkv_append_kv_merge(self._ctx, C.byref(st.struct()), _ptr(k_new), _ptr(v_new), _ptr(q), _stream()))

    def score(self, st: DeviceState, q):
        _check(lib.hardkv_score(self._ctx, C.byref(st.struct()), _ptr(q), _stream()))

    def score_select(self, st: DeviceState, q, p: float):
        _check(lib.hardkv_score_select(self._ctx, C.byref(st.struct()), _ptr(q), np.float32(p), _stream()))

    def qcache_push(self, st: DeviceState, q):
        _check(lib.hardkv_qcache_push(self._ctx, C.byref(st.struct()), _ptr(q), _stream()))

    def calibrate_topp(self, st: DeviceState, p: float):
        _check(lib.hardkv_calibrate_topp(self._ctx, C.byref(st.struct()), np.float32(p), _stream()))

    def solve_temperature(self, st: DeviceState, p: float, t_min: float = 0.03125, t_max: float = 32.0,
                          eps: float = 1e-4, max_iter: int = 40):
        """Algorithm 2 (L625-648) on the logits of the last score(); writes st.temperature."""
        _check(lib.hardkv_solve_temperature(self._ctx, C.byref(st.struct()), np.float32(p), np.float32(t_min),
                                            np.float32(t_max), np.float32(eps), int(max_iter), _stream()))

    def topp_select(self, st: DeviceState, p: float):
        _check(lib.hardkv_topp_select(self._ctx, C.byref(st.struct()), np.float32(p), _stream()))

    def rewrite(self, st: DeviceState):
        _check(lib.hardkv_rewrite(self._ctx, C.byref(st.struct()), _stream()))

    def decode_attn(self, st: DeviceState, q, out, lse=None):
        _check(lib.hardkv_decode_attn(self._ctx, C.byref(st.struct()), _ptr(q), _ptr(out), _ptr(lse), _stream()))

    def rewrite_attend(self, st: DeviceState, q, out, lse=None):
        _check(lib.hardkv_rewrite_attend(self._ctx, C.byref(st.struct()), _ptr(q), _ptr(out), _ptr(lse), _stream()))

    def sparse_attend(self, st: DeviceState, q, out, lse=None):
        _check(lib.hardkv_sparse_attend(self._ctx, C.byref(st.struct()), _ptr(q), _ptr(out), _ptr(lse), _stream()))

    def launch_count(self) -> int:
        return int(lib.hardkv_launch_count(self._ctx))

    def decode_step_host(self, st: DeviceState, q_host, k_new_host, v_new_host, p: float, out_host,
                         do_select: bool = True, stream: int | None = None):
        """q_host / k_new_host / v_new_host / out_host: HOST (ideally pinned) torch tensors; see hardkv.h.
        stream: raw cudaStream_t handle (torch.cuda.current_stream().cuda_stream) of a caller that holds on to its
        stream -- saves the per-call lookup in a per-token loop; None = torch's current stream."""
        for t in (q_host, k_new_host, v_new_host, out_host):
            assert not t.is_cuda and t.is_contiguous()
        _check(lib.hardkv_decode_step_host(self._ctx, C.byref(st.struct()), q_host.data_ptr(), k_new_host.data_ptr(),
                                           v_new_host.data_ptr(), p, int(do_select), out_host.data_ptr(),
                                           _stream() if stream is None else stream))

    def decode_step(self, st: DeviceState, q, k_new, v_new, p: float, out, lse=None, do_select: bool = True):
        _check(lib.hardkv_decode_step(self._ctx, C.byref(st.struct()), _ptr(q), _ptr(k_new), _ptr(v_new),
                                      np.float32(p), int(do_select), _ptr(out), _ptr(lse), _stream()))
