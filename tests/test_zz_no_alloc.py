"""hardkv_decode_attn_noalloc: the allocation-free variant of the split-K decode attention (no ctx, no workspace: its
scratch is the library's file-scope static device array) against the existing hardkv_decode_attn on the same state,
two calls in a row, at the tolerances of the other GPU tests.  Named so that pytest collects it last."""
import numpy as np
import pytest
import torch

from gpu_common import DEV, OUT_MAX_ABS, OUT_MEAN_ABS, Pair
from workloads.synth import make_workload

pytestmark = pytest.mark.gpu
i32 = lambda *v: np.array(v, np.int32)
LSE_TOL = 2e-3


def _workloads():
    return {
        "bf16_g4": make_workload(1, n0=i32(2100), max_ctx=2176, k_cap=512, l_upper=i32(1960), cond_cap=32, steps=6),
        "bf16_b3": make_workload(2, B=3, n0=i32(900, 2300, 1500), max_ctx=2400, k_cap=256,
                                 l_upper=i32(900 - 132, 2300 - 132, 1500 - 132), cond_cap=24, steps=6),
        "f32": make_workload(0),
    }


@pytest.mark.parametrize("name", ["bf16_g4", "bf16_b3", "f32"])
def test_noalloc_attention_matches_the_workspace_path_twice(name):
    from paper_2606_28831_b200 import hardkv
    wl = _workloads()[name]
    pr = Pair(wl, want_mask=False)
    # three fused steps through the existing path fill the selected and condensed tiers
    for t in range(3):
        _, _, _, (qd, knd, vnd) = pr.inputs(t)
        pr.eng.decode_step(pr.st, qd, knd, vnd, wl.p, pr.out, pr.lse)
    torch.cuda.synchronize()
    for call, t in enumerate((3, 4)):          # two calls in a row on the shared static scratch, different queries
        _, _, _, (qd, _, _) = pr.inputs(t)
        ref_out, ref_lse = torch.zeros_like(pr.out), torch.zeros_like(pr.lse)
        out, lse = torch.full_like(pr.out, float("nan")), torch.full_like(pr.lse, float("nan"))
        pr.eng.decode_attn(pr.st, qd, ref_out, ref_lse)
        hardkv.decode_attn_noalloc(pr.eng.cfg, pr.st, qd, out, lse)
        torch.cuda.synchronize()
        assert int(pr.st.err_flag.item()) == 0
        assert bool(torch.isfinite(out).all()) and bool(torch.isfinite(lse).all()), (name, call)
        err = (out - ref_out).abs()
        assert float(err.max()) <= OUT_MAX_ABS and float(err.mean()) <= OUT_MEAN_ABS, (name, call, float(err.max()))
        assert float((lse - ref_lse).abs().max()) <= LSE_TOL, (name, call)
        # same kernel, same launch shape, same merge order: in fact the two paths agree bit for bit
        assert torch.equal(out, ref_out) and torch.equal(lse, ref_lse), (name, call)


def test_noalloc_rejects_a_problem_beyond_the_static_scratch():
    """BASELINE configs[2] needs 18 MB of split-K partial states: refused with a clear error before anything is launched
    (the state handed in is never touched)."""
    from paper_2606_28831_b200 import hardkv
    small = _workloads()["bf16_g4"]
    pr = Pair(small, want_mask=False)
    big = hardkv.Config(16, 32, 8, 128, 16, 33024, 4, 128, 8192, 256, 0, hardkv.BF16, 0.0, 0, 0, 0)
    _, _, _, (qd, _, _) = pr.inputs(0)
    with pytest.raises(hardkv.HardKVError, match="static scratch"):
        hardkv.decode_attn_noalloc(big, pr.st, qd, pr.out, pr.lse)
    torch.cuda.synchronize()
