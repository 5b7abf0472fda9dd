"""-m gpu parity tests: the CUDA path (called through the C ABI) against the CPU oracle, element by
element on the same seeded inputs.  Sizes span several tiles and ragged tails of every kernel
(score: 512-token CTA tiles; select: 512 threads / 16 warp segments; rewrite: 64 rows; attention:
128-row chunks) and the degenerate cases (empty pool, single token, ties, k_cap clamp, p = 1).

Bars (BASELINE.json north_star): selection, counts, tables, votes, rewritten rows, condensed-tier
bookkeeping bit-exact given identical probabilities; end to end only tokens within 1e-6 of the
threshold may differ; outputs max-abs <= 2e-2, mean-abs <= 2e-3.
"""
import numpy as np
import pytest
import torch

from workloads.synth import make_workload

pytestmark = pytest.mark.gpu

i32 = lambda *v: np.array(v, np.int32)


def small_workloads():
    """Shrunk versions of BASELINE.json's five configs (same dtype, G, d, structure, parameters)."""
    return {
        "c0": make_workload(0),
        "c1s": make_workload(1, n0=i32(2100), max_ctx=2176, k_cap=512, l_upper=i32(1960), cond_cap=32, steps=6),
        "c2s": make_workload(2, B=3, n0=i32(900, 2300, 1500), max_ctx=2400, k_cap=256,
                             l_upper=i32(900 - 132, 2300 - 132, 1500 - 132), cond_cap=24, steps=6),
        "c3s": make_workload(3, B=2, n0=i32(300, 300), max_ctx=512, k_cap=64, l_upper=i32(48, 48), cond_cap=8,
                             steps=40),
        "c4s": make_workload(4, B=2, n0=i32(1500, 1500), max_ctx=1600, k_cap=384, l_upper=i32(1390, 1390),
                             cond_cap=16, accum_window=4, steps=8),
        "g1d64": make_workload(1, Hq=2, Hkv=2, d=64, n0=i32(700), max_ctx=720, k_cap=128, l_upper=i32(560),
                               cond_cap=4, steps=4),
        "g2": make_workload(1, Hq=4, Hkv=2, n0=i32(640), max_ctx=656, k_cap=160, l_upper=i32(500), cond_cap=4,
                            steps=4),
        # SNAPKV heads (logits max-pooled along the sequence, L278) mixed with RAW heads: G = 4 and G = 7
        "snap4": make_workload(1, n0=i32(2100), max_ctx=2176, k_cap=512, l_upper=i32(1960), cond_cap=32, steps=6,
                               score_mode=np.array([0, 2, 2, 0, 2, 0, 2, 2], np.uint8), pool_kernel=7),
        "snap7": make_workload(3, B=2, n0=i32(1300, 1300), max_ctx=1536, k_cap=256, l_upper=i32(1100, 1100),
                               cond_cap=8, steps=6, score_mode=np.array([2, 2, 0, 2], np.uint8), pool_kernel=5),
        # accumulated attention recomputed from the query cache (L448; score_mode 3), alone and next to ring-sum ACCUM heads
        "qc4": make_workload(1, n0=i32(2100), max_ctx=2176, k_cap=512, l_upper=i32(1960), cond_cap=32, steps=8,
                             score_mode=np.array([0, 3, 3, 0, 3, 0, 3, 3], np.uint8), accum_window=4),
        "qc5": make_workload(4, B=2, n0=i32(1500, 1500), max_ctx=1600, k_cap=384, l_upper=i32(1390, 1390),
                             cond_cap=16, accum_window=6, steps=9, score_mode=np.array([0, 3, 0, 1, 3, 1, 3, 3], np.uint8)),
        # the tensor-core (tcgen05) form of the same metric at its other shapes: more than 128 query rows (20 cached steps
        # x G = 8 = 160 -> the 256-row block) over a pool of several 128-token tiles and both chunk slots of a CTA; d = 64
        "qc8w": make_workload(1, Hq=16, Hkv=2, n0=i32(3300), max_ctx=3408, k_cap=512, l_upper=i32(3100), cond_cap=16,
                              steps=24, score_mode=np.array([3, 3], np.uint8), accum_window=20),
        "qc64": make_workload(1, Hq=8, Hkv=2, d=64, n0=i32(1900), max_ctx=1936, k_cap=256, l_upper=i32(1700), cond_cap=8,
                              steps=10, score_mode=np.array([3, 0], np.uint8), accum_window=8),
        "g8": make_workload(1, Hq=8, Hkv=1, n0=i32(1100), max_ctx=1120, k_cap=1120, l_upper=i32(5000), cond_cap=0,
                            steps=3),
    }


WL = small_workloads()


@pytest.fixture(scope="module")
def P():
    from gpu_common import Pair
    return Pair


@pytest.mark.parametrize("name", list(WL))
def test_stages_teacher_forced(name, P):
    """Each ABI stage against the matching oracle stage, every step; selection fed identical probabilities."""
    wl = WL[name]
    pr = P(wl)
    eng, st, ob = pr.eng, pr.st, pr.ob
    for t in range(min(wl.steps, 6)):
        q, kn, vn, (qd, knd, vnd) = pr.inputs(t)
        G, d = wl.G, wl.d
        # step 0: append + retire
        eng.append_kv(st, knd, vnd)
        for i, u in enumerate(ob.units):
            u.append(kn.reshape(-1, d)[i], vn.reshape(-1, d)[i])
            u.retire()
        pr.check_bookkeeping()
        # step 1: score (and, for heads on the query-cache metric, the window slides: L448)
        eng.score(st, qd)
        if st.qcache is not None:
            eng.qcache_push(st, qd)
        qu = q.reshape(-1, G, d)
        for i, u in enumerate(ob.units):
            u.score(qu[i])
            u.qcache_push(qu[i])
        pr.check_logits()
        # step 2a-2c end to end from the CUDA logits (votes restored afterwards)
        votes0 = st.votes.clone()
        eng.calibrate_topp(st, wl.p)
        for u in ob.units:
            u.calibrate()
            u.topp_select(wl.p, True)
        pr.check_probs()
        pr.check_selection_band()
        # step 2b-2c bit exact from identical probabilities
        st.votes.copy_(votes0)
        pr.upload_oracle_probs()
        eng.topp_select(st, wl.p)
        pr.check_selection_exact()
        # step 3: rewrite
        eng.rewrite(st)
        for u in ob.units:
            u.rewrite()
        pr.check_rewrite_exact()
        # step 4: attention over the three tiers
        eng.decode_attn(st, qd, pr.out, pr.lse)
        for i, u in enumerate(ob.units):
            u.attend(qu[i])
        pr.check_out(f"{name} step {t}")
        # HA-Sparse (L178): the same attention gathered through sel_idx; the selected tier is not touched
        tier0 = (st.sel_k_pool.clone(), st.sel_v_pool.clone())
        out2, lse2 = torch.zeros_like(pr.out), torch.zeros_like(pr.lse)
        eng.sparse_attend(st, qd, out2, lse2)
        assert torch.equal(out2, pr.out) and torch.equal(lse2, pr.lse)
        assert torch.equal(tier0[0], st.sel_k_pool) and torch.equal(tier0[1], st.sel_v_pool)


@pytest.mark.parametrize("name", ["c0", "c2s", "c3s", "c4s", "snap4"])
def test_sparse_regime_steps(name, P):
    """HA-Sparse decode steps (do_select 2 / 3: select every 3rd step, attend through sel_idx in between, no
    rewrite ever) against the oracle run with the same compression interval (L178, L191, L274)."""
    from paper_2606_28831_b200 import hardkv
    wl = WL[name]
    pr = P(wl, want_mask=False, reuse_max=2)
    tier0 = (pr.st.sel_k_pool.clone(), pr.st.sel_v_pool.clone())
    for t in range(min(wl.steps, 9)):
        q, kn, vn, (qd, knd, vnd) = pr.inputs(t)
        sel = t % 3 == 0
        pr.eng.decode_step(pr.st, qd, knd, vnd, wl.p, pr.out, pr.lse,
                           do_select=hardkv.STEP_SELECT_SPARSE if sel else hardkv.STEP_REUSE_SPARSE)
        pr.ob.step(q, kn, vn, wl.p, do_select=sel)
        pr.check_out(f"{name} sparse step {t}")
        if sel:
            pr.check_selection_band()
        pr.force_discrete_state()
    assert torch.equal(tier0[0], pr.st.sel_k_pool) and torch.equal(tier0[1], pr.st.sel_v_pool)


@pytest.mark.parametrize("name", list(WL))
@pytest.mark.parametrize("teacher", [True, False])
def test_fused_decode_step(name, teacher, P):
    """hardkv_decode_step (one call per step) over a trajectory, teacher-forced and free-running."""
    wl = WL[name]
    pr = P(wl, want_mask=False)
    first_div, emax = None, 0.0
    for t in range(min(wl.steps, 12)):
        q, kn, vn, (qd, knd, vnd) = pr.inputs(t)
        pr.eng.decode_step(pr.st, qd, knd, vnd, wl.p, pr.out, pr.lse)
        pr.ob.step(q, kn, vn, wl.p)
        emax = max(emax, pr.check_out(f"{name} step {t}")[0])
        f = pr.check_selection_band()
        if f == 0:
            pr.check_bookkeeping()
            pr.check_rewrite_exact()
            pr.check_votes()
        if teacher:
            pr.force_discrete_state()
        elif f:
            # free running: report the first divergence, then let the ORACLE adopt the CUDA path's
            # discrete state so that the rest of the trajectory is still compared step by step
            first_div = t if first_div is None else first_div
            pr.adopt_cuda_discrete_state()
    print(f"[{name} {'teacher-forced' if teacher else 'free-running'}] near-threshold flips {pr.flips_total}, "
          f"first divergence step {first_div}, max-abs output error over the run {emax:.2e}")


@pytest.mark.parametrize("variant", [0, 2, 3, 4])
@pytest.mark.parametrize("name", ["c1s", "c2s", "c3s", "c4s", "g1d64", "snap4", "qc4"])
def test_kernel_variants(name, variant, P):
    """Variant 0 (generic fp32-FMA kernels), 2 (TMA-staged persistent score), 3 (score and selection fused into one
    persistent kernel: CTAs stream K pages and the CTA that retires a unit's last chunk runs its selection) and 4 (the
    publishing persistent score kernel with the select kernel co-resident behind it, longest unit first) against the
    oracle; the default is variant 1.  Variants 3 and 4 do not apply to configs with SNAPKV heads (the pooling pass sits
    between score and select).  qc4 (query-cache heads): variant 0 runs the mma.sync form of the query-cache passes, the
    others the tcgen05 form; with a query cache in the state variants 3 / 4 run their stages back to back."""
    from paper_2606_28831_b200 import hardkv
    wl = WL[name]
    pr = P(wl, want_mask=False)
    if variant in (3, 4) and wl.pool_kernel > 1:
        with pytest.raises(hardkv.HardKVError):
            pr.eng.set_variant(variant)
        return
    pr.eng.set_variant(variant)
    for t in range(min(wl.steps, 8)):
        q, kn, vn, (qd, knd, vnd) = pr.inputs(t)
        pr.eng.decode_step(pr.st, qd, knd, vnd, wl.p, pr.out, pr.lse)
        pr.ob.step(q, kn, vn, wl.p)
        pr.check_out(f"{name} v{variant} step {t}")
        pr.check_selection_band()
        pr.force_discrete_state()
    pr.check_logits()


@pytest.mark.parametrize("cluster,threads", [(1, 512), (2, 512), (4, 512), (8, 512), (1, 1024), (2, 1024)])
@pytest.mark.parametrize("name", ["c2s", "c4s", "g8"])
def test_select_every_cluster_size(name, cluster, threads, P):
    """The select kernel at every cluster size (1 = single CTA, no DSMEM) and both CTA sizes (512 threads, two CTAs per
    SM; 1024 threads, one per SM): bit exact from identical probabilities."""
    wl = WL[name]
    pr = P(wl)
    pr.eng.set_select_geometry(cluster, threads)
    for t in range(3):
        q, kn, vn, (qd, knd, vnd) = pr.inputs(t)
        pr.eng.decode_step(pr.st, qd, knd, vnd, wl.p, pr.out, pr.lse)
        pr.ob.step(q, kn, vn, wl.p)
        pr.check_out(f"{name} C{cluster} step {t}")
        assert pr.check_selection_band() == 0
        votes0 = pr.st.votes.clone()
        pr.upload_oracle_probs()
        pr.eng.topp_select(pr.st, wl.p)
        pr.st.votes.copy_(votes0)
        np.testing.assert_array_equal(pr.st.sel_idx.cpu().numpy(), pr.ob.sel_idx())
        np.testing.assert_array_equal(pr.st.sel_count.cpu().numpy(), pr.ob.sel_count())


@pytest.mark.parametrize("variant", [1, 3])
@pytest.mark.parametrize("name", ["c2s", "c3s", "c4s", "g8"])
def test_score_select_entry(name, variant, P):
    """hardkv_score_select (stages 1 + 2a-2c in one call) against the oracle stages: logits, probabilities and the
    selection -- as separate kernels (variant 1) and as the fused persistent kernel (variant 3), over several steps so
    that units of different lengths finish their scan at different times; also a batch of more chunks than SMs."""
    import dataclasses
    wl = WL[name]
    if name == "c2s":    # more (unit, chunk) work items than CTAs: CTAs take several items and switch role mid-kernel
        wl = make_workload(2, B=12, n0=np.linspace(1400, 5200, 12).astype(np.int32), max_ctx=5376, k_cap=512,
                           l_upper=np.linspace(1400, 5200, 12).astype(np.int32) - 132, cond_cap=16, steps=4)
    pr = P(wl)
    pr.eng.set_variant(variant)
    for t in range(min(wl.steps, 4)):
        q, kn, vn, (qd, knd, vnd) = pr.inputs(t)
        pr.eng.append_kv(pr.st, knd, vnd)
        pr.eng.score_select(pr.st, qd, wl.p)
        qu = q.reshape(-1, wl.G, wl.d)
        for i, u in enumerate(pr.ob.units):
            u.append(kn.reshape(-1, wl.d)[i], vn.reshape(-1, wl.d)[i])
            u.retire()
            u.score(qu[i]); u.calibrate(); u.topp_select(wl.p, True)
        pr.check_bookkeeping()
        pr.check_logits()
        pr.check_probs()
        if pr.check_selection_band() == 0:
            pr.check_selection_exact()
        pr.force_discrete_state()
    assert int(pr.st.err_flag.item()) == 0


def test_select_interval_reuses_selected_tier(P):
    """do_select = 0 between compressions (L274): append + attend over the previous selected tier."""
    wl = WL["c1s"]
    pr = P(wl, want_mask=False, reuse_max=2)
    for t in range(6):
        q, kn, vn, (qd, knd, vnd) = pr.inputs(t)
        sel = (t % 3 == 0)
        pr.eng.decode_step(pr.st, qd, knd, vnd, wl.p, pr.out, pr.lse, do_select=sel)
        pr.ob.step(q, kn, vn, wl.p, do_select=sel)
        pr.check_out(f"step {t}")
        assert pr.check_selection_band(own_probs=sel) == 0
        pr.check_bookkeeping()


@pytest.mark.parametrize("case", ["ties", "one_dominant", "p1", "l_lower", "clamp", "zeros", "n1"])
def test_select_degenerate(case, P):
    """Top-p edge cases on hand-made probability rows, bit exact."""
    wl = make_workload(1, Hq=4, Hkv=1, n0=i32(1200), max_ctx=1216, k_cap=1216 if case != "clamp" else 64,
                       l_upper=i32(5000), cond_cap=0, l_lower=i32(2000 if case == "l_lower" else 0))
    if case == "n1":
        wl = make_workload(1, Hq=4, Hkv=1, n0=i32(4 + 128 + 1), max_ctx=160, k_cap=16, l_upper=i32(5000), cond_cap=0)
    pr = P(wl)
    u = pr.ob.units[0]
    lo, hi = u.pool
    N = hi - lo
    rng = np.random.default_rng(5)
    p = 0.9
    if case == "ties":
        row = np.full(N, 1.0 / N, np.float32)
    elif case == "one_dominant":
        row = np.full(N, 1e-12, np.float32); row[N // 3] = 1.0
    elif case == "p1":
        row = rng.random(N).astype(np.float32); row /= row.sum(); p = 1.0
    elif case == "zeros":
        row = np.zeros(N, np.float32); row[5:40] = 1.0 / 35
    elif case == "n1":
        row = np.ones(N, np.float32)
    else:
        row = rng.random(N).astype(np.float32) ** 4; row /= row.sum()
        row[100:140] = row[100]   # a run of exact ties inside the row
    u.probs[lo:hi] = row
    u.topp_select(p, True)
    pr.upload_oracle_probs()
    pr.eng.topp_select(pr.st, p)
    pr.check_selection_exact()
    assert u.sel_count > 0


def test_topp_select_flags_a_row_that_is_not_a_probability_row(P):
    """hardkv_topp_select takes the caller's probabilities as given; its integer-mass histogram is exact for rows that
    sum to far less than 4096, so a row that sums to more than 4 in any warp's share is flagged (err_flag 3) instead of
    being selected from silently; a normalised row leaves the flag alone."""
    wl = make_workload(1, Hq=4, Hkv=1, n0=i32(1200), max_ctx=1216, k_cap=1216, l_upper=i32(5000), cond_cap=0)
    pr = P(wl)
    u = pr.ob.units[0]
    lo, hi = u.pool
    u.probs[lo:hi] = np.float32(1.0 / (hi - lo))
    pr.upload_oracle_probs()
    pr.eng.topp_select(pr.st, 0.9)
    assert int(pr.st.err_flag.item()) == 0
    u.probs[lo:hi] = np.float32(0.5)
    pr.upload_oracle_probs()
    pr.eng.topp_select(pr.st, 0.9)
    assert int(pr.st.err_flag.item()) == 3
    pr.st.err_flag.zero_()


def test_empty_pool_and_growth(P):
    """Context shorter than sink + recent: empty pool, dense tier only; then the pool opens."""
    wl = make_workload(1, Hq=8, Hkv=2, n0=i32(3), max_ctx=256, k_cap=64, l_upper=i32(30), cond_cap=4, recent=16)
    pr = P(wl, want_mask=False)
    for t in range(70):
        q, kn, vn, (qd, knd, vnd) = pr.inputs(t)
        pr.eng.decode_step(pr.st, qd, knd, vnd, wl.p, pr.out, pr.lse)
        pr.ob.step(q, kn, vn, wl.p)
        pr.check_out(f"step {t}")
        assert pr.check_selection_band() == 0
        pr.check_bookkeeping()
        pr.check_votes()


def test_cuda_graph_replay(P):
    """The fused step captured once and replayed: shapes static, counts on the device (L53, L63)."""
    wl = WL["c2s"]
    pr = P(wl, want_mask=False)
    q, kn, vn, (qd, knd, vnd) = pr.inputs(0)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        pr.eng.decode_step(pr.st, qd, knd, vnd, wl.p, pr.out, pr.lse)   # warm-up outside capture (step 0)
    torch.cuda.current_stream().wait_stream(s)
    pr.ob.step(q, kn, vn, wl.p)
    pr.check_out("warm-up step")
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        pr.eng.decode_step(pr.st, qd, knd, vnd, wl.p, pr.out, pr.lse)
    # capture does not execute: the first replay is step 1
    for t in range(1, 5):
        q, kn, vn, (q2, k2, v2) = pr.inputs(t)
        qd.copy_(q2); knd.copy_(k2); vnd.copy_(v2)
        g.replay()
        pr.ob.step(q, kn, vn, wl.p)
        pr.check_out(f"replay {t}")
        assert pr.check_selection_band() == 0
        pr.check_bookkeeping()


def test_error_paths(P):
    """Host-detectable errors come back as status codes; a full context sets err_flag on the device."""
    from paper_2606_28831_b200 import hardkv
    with pytest.raises(hardkv.HardKVError):
        hardkv.HardKV(batch=1, num_q_heads=6, num_kv_heads=2, head_dim=128, max_ctx=64, sink=4, recent=8, k_cap=16,
                      cond_cap=0, kv_dtype=hardkv.BF16)          # G = 3 is not built
    with pytest.raises(hardkv.HardKVError):
        hardkv.HardKV(batch=1, num_q_heads=4, num_kv_heads=1, head_dim=128, max_ctx=70, sink=4, recent=8, k_cap=16,
                      cond_cap=0, kv_dtype=hardkv.BF16)          # max_ctx not a multiple of the page
    wl = make_workload(1, Hq=4, Hkv=1, n0=i32(64), max_ctx=64, k_cap=16, l_upper=i32(100), cond_cap=0, recent=16)
    pr = P(wl, want_mask=False)
    q, kn, vn, (qd, knd, vnd) = pr.inputs(0)
    pr.eng.append_kv(pr.st, knd, vnd)                             # ctx_len == max_ctx: no room
    torch.cuda.synchronize()
    assert int(pr.st.err_flag.item()) == 1 and int(pr.st.ctx_len.item()) == 64
    # the same through the fused step, whose append kernel runs on a forked branch beside the score kernel and leaves the
    # per-sequence scalars to the attention kernel to write back: a full context stays exactly as it was
    pr.st.err_flag.zero_()
    before = (int(pr.st.ctx_len.item()), int(pr.st.c_lo.item()), int(pr.st.dense_lo.item()))
    pr.eng.decode_step(pr.st, qd, knd, vnd, wl.p, pr.out, pr.lse)
    torch.cuda.synchronize()
    assert int(pr.st.err_flag.item()) == 1
    assert (int(pr.st.ctx_len.item()), int(pr.st.c_lo.item()), int(pr.st.dense_lo.item())) == before
    with pytest.raises(hardkv.HardKVError):
        pr.eng.score(pr.st, None)


@pytest.mark.parametrize("name", ["c1s", "c4s", "snap4", "snap7", "c0"])
def test_solve_temperature(name, P):
    """hardkv_solve_temperature (Algorithm 2) against the oracle's bisection on the same logits.
    Floating point decides every branch of the search, so the unique thing compared is the root: T agrees to
    1e-3 relative (both sides stop within eps = 1e-5 of mass error, which bounds T to ~1e-4 of the root);
    ACCUM heads keep their T bit for bit.  The solved T then drives one calibrated selection step."""
    wl = WL[name]
    pr = P(wl, want_mask=False)
    eng, st, ob = pr.eng, pr.st, pr.ob
    q, kn, vn, (qd, knd, vnd) = pr.inputs(0)
    eng.append_kv(st, knd, vnd)
    eng.score(st, qd)
    eng.solve_temperature(st, wl.p, t_min=0.0625, t_max=16.0, eps=1e-5, max_iter=40)
    T_gpu = st.temperature.cpu().numpy().reshape(-1)
    qu = q.reshape(-1, wl.G, wl.d)
    for i, u in enumerate(ob.units):
        u.append(kn.reshape(-1, wl.d)[i], vn.reshape(-1, wl.d)[i])
        u.retire()
        u.score(qu[i])
        T0 = u.T
        it, resid = u.solve_temperature(wl.p, t_min=0.0625, t_max=16.0, eps=1e-5, max_iter=40)
        mode = int(wl.score_mode[i % wl.Hkv])
        if mode == 1:
            assert it == 0 and T_gpu[i] == np.float32(T0)
        else:
            assert resid <= 1e-5 and it >= 1
            assert abs(T_gpu[i] - u.T) <= 1e-3 * u.T, (i, mode, T_gpu[i], u.T)
            if mode == 0:
                assert abs(T_gpu[i] - 1.0) < 5e-3          # g = id: T* = 1 (pin P13)
        u.u.T = np.float32(T_gpu[i])                        # teacher-force T, then one calibrated selection
    eng.calibrate_topp(st, wl.p)
    for u in ob.units:
        u.calibrate()
        u.topp_select(wl.p, True)
    pr.check_probs()
    pr.check_selection_band()


MERGE_WL = {
    # fp32, G = 4: the first step retires 45 tokens at once into 4 slots (loop of merges inside one call)
    "merge0": make_workload(0, l_upper=i32(400), cond_cap=4, cond_merge=1),
    # bf16, G = 4, three sequences of different lengths, one retirement per step, tier full after 6 steps
    "merge4": make_workload(2, B=3, n0=i32(900, 2300, 1500), max_ctx=2400, k_cap=256,
                            l_upper=i32(900 - 132, 2300 - 132, 1500 - 132), cond_cap=6, steps=14, cond_merge=1),
    # bf16, G = 7 with mixed new keys: the first step retires 11 tokens into 8 slots, then one per step
    "merge7": make_workload(3, B=2, n0=i32(300, 300), max_ctx=512, k_cap=64, l_upper=i32(30, 30), cond_cap=8,
                            steps=14, cond_merge=1),
}


@pytest.mark.parametrize("name", list(MERGE_WL))
def test_condensed_tier_weighted_merging(name, P):
    """cfg.cond_merge: evictees of the full condensed tier are folded into the best-scoring resident with the
    LSE-preserving weights of Appendix G (Eq. 9) -- stand-alone entry and fused step against the oracle.  Slots,
    positions and votes are exact; merged rows agree to one ulp of kv_dtype (fp32 vs fp64 before the store
    rounding); the state is teacher-forced after every step."""
    wl = MERGE_WL[name]
    pr = P(wl, want_mask=False)
    merged_any = False
    for t in range(min(wl.steps, 14)):
        q, kn, vn, (qd, knd, vnd) = pr.inputs(t)
        full_before = [u.cond_count == wl.cond_cap for u in pr.ob.units]
        if t % 2 == 0:     # the stand-alone entry, then the rest of the step from its stages
            pr.eng.append_kv_merge(pr.st, knd, vnd, qd)
            qu = q.reshape(-1, wl.G, wl.d)
            for i, u in enumerate(pr.ob.units):
                u.append(kn.reshape(-1, wl.d)[i], vn.reshape(-1, wl.d)[i])
                merged_any |= bool(u.retire_q(qu[i]) and full_before[i])
            pr.check_bookkeeping()
            pr.force_discrete_state()
            pr.eng.score(pr.st, qd)
            pr.eng.calibrate_topp(pr.st, wl.p)
            pr.eng.rewrite_attend(pr.st, qd, pr.out, pr.lse)
            for i, u in enumerate(pr.ob.units):
                u.score(qu[i]); u.calibrate(); u.topp_select(wl.p, True); u.rewrite(); u.attend(qu[i])
        else:
            pr.eng.decode_step(pr.st, qd, knd, vnd, wl.p, pr.out, pr.lse)
            pr.ob.step(q, kn, vn, wl.p)
            pr.check_bookkeeping()
        pr.check_out(f"{name} step {t}")
        pr.check_selection_band()
        pr.force_discrete_state()
    assert merged_any


@pytest.mark.parametrize("name,steps", [("c2s", 64), ("c4s", 48), ("snap7", 40)])
def test_long_teacher_forced_trajectory(name, steps, P):
    """Many fused steps in a row (votes accumulate, the condensed tier fills and turns over, the ACCUM ring wraps
    several times, the context grows across page and chunk boundaries): every step judged against the oracle."""
    import dataclasses
    wl = dataclasses.replace(WL[name], steps=steps, max_ctx=WL[name].max_ctx + 64)
    pr = P(wl, want_mask=False)
    for t in range(steps):
        q, kn, vn, (qd, knd, vnd) = pr.inputs(t)
        pr.eng.decode_step(pr.st, qd, knd, vnd, wl.p, pr.out, pr.lse)
        pr.ob.step(q, kn, vn, wl.p)
        pr.check_out(f"{name} step {t}")
        if pr.check_selection_band() == 0:
            pr.check_bookkeeping()
            pr.check_votes()
        pr.force_discrete_state()
    if name != "snap7":
        assert all(u.cond_count == wl.cond_cap for u in pr.ob.units)      # the condensed tier did fill


def test_paper_regime_hysteresis_and_interval(P):
    """The paper's periodic regime on one trajectory (L197, L270, L274): compression every 4th step, L_lower =
    L_upper - 20.  The pool starts below L_lower (everything is selected: no sparsity yet), grows past it (Top-p
    selection), then past L_upper (the oldest tokens retire into the condensed tier); the steps in between reuse the
    rewritten tier (HA-Max, do_select = 0)."""
    wl = make_workload(1, Hq=8, Hkv=2, n0=i32(700), max_ctx=800, k_cap=640, l_upper=i32(620), cond_cap=8, steps=72)
    wl.l_lower = i32(600)
    pr = P(wl, want_mask=False, reuse_max=3)
    phases = set()
    for t in range(72):
        q, kn, vn, (qd, knd, vnd) = pr.inputs(t)
        sel = t % 4 == 0
        pr.eng.decode_step(pr.st, qd, knd, vnd, wl.p, pr.out, pr.lse, do_select=sel)
        pr.ob.step(q, kn, vn, wl.p, do_select=sel)
        pr.check_out(f"paper regime step {t}")
        u = pr.ob.units[0]
        lo, hi = u.pool
        if sel:
            pr.check_selection_band()
            if hi - lo <= 600:
                assert u.sel_count == hi - lo
                phases.add("all")
            else:
                assert u.sel_count < hi - lo
                phases.add("topp")
        if u.cond_count > 0:
            phases.add("retire")
        pr.check_bookkeeping()
        pr.force_discrete_state()
    assert phases == {"all", "topp", "retire"}


def test_cuda_graph_replay_widened_entries(P):
    """The widened entry points are capturable too (no allocation, no synchronisation, no host read-back): one graph
    holding append + merge, score, the Algorithm 2 solve, calibrate + Top-p and the HA-Sparse attention is replayed
    and compared with the same calls made eagerly on a second, identical engine."""
    import dataclasses
    wl = dataclasses.replace(WL["snap4"], cond_merge=1)
    a, b = P(wl, want_mask=False), P(wl, want_mask=False)

    def calls(pr, qd, knd, vnd):
        pr.eng.append_kv_merge(pr.st, knd, vnd, qd)
        pr.eng.score(pr.st, qd)
        pr.eng.solve_temperature(pr.st, wl.p, t_min=0.0625, t_max=16.0, eps=1e-5, max_iter=30)
        pr.eng.calibrate_topp(pr.st, wl.p)
        pr.eng.sparse_attend(pr.st, qd, pr.out, pr.lse)

    q, kn, vn, (qd, knd, vnd) = a.inputs(0)
    qb, kb, vb = qd.clone(), knd.clone(), vnd.clone()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        calls(a, qd, knd, vnd)                              # warm-up outside capture (step 0)
    torch.cuda.current_stream().wait_stream(s)
    calls(b, qb, kb, vb)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        calls(a, qd, knd, vnd)
    for t in range(1, 4):
        _, _, _, (q2, k2, v2) = a.inputs(t)
        qd.copy_(q2); knd.copy_(k2); vnd.copy_(v2)
        g.replay()
        calls(b, q2, k2, v2)
        torch.cuda.synchronize()
        for f in ("temperature", "sel_count", "sel_idx", "cond_k", "cond_pos", "votes", "ctx_len", "c_lo"):
            assert torch.equal(getattr(a.st, f), getattr(b.st, f)), (t, f)
        assert torch.equal(a.out, b.out) and torch.equal(a.lse, b.lse)


def test_depth_one_graph_over_layers_with_shared_block_ids():
    """Depth (Fig. 6: "head-independent indices ... regularized for all layers", so one block id
    addresses the same block in every layer and kernel executions can be captured "throughout the model's depth"): four
    layers of INDEPENDENTLY seeded KV data and inputs share one base_table / sel_pages, the four layer-steps of a decode
    step are captured into ONE CUDA graph, and every layer is compared with its own oracle after every replay."""
    import dataclasses
    from gpu_common import DEV, Pair
    from oracle.batch import OracleBatch
    from paper_2606_28831_b200 import harness
    Lyr = 4
    wl = make_workload(2, B=3, n0=i32(900, 2300, 1500), max_ctx=2400, k_cap=256, l_upper=i32(900 - 132, 2300 - 132, 1500 - 132),
                       cond_cap=24, steps=8)
    seeds = [wl.seed + 7919 * (l + 1) for l in range(Lyr)]
    wls = []
    for sd in seeds:
        w = dataclasses.replace(wl)
        w.seed = sd
        w.page_tables = wl.page_tables      # the block ids are the model's, not the layer's (L207-209)
        wls.append(w)
    eng = harness.make_engine(wl, DEV)
    states, prefill = harness.make_state(wl, DEV, layers=Lyr, layer_seeds=seeds)
    assert all(s.base_table.data_ptr() == states[0].base_table.data_ptr() and
               s.sel_pages.data_ptr() == states[0].sel_pages.data_ptr() for s in states)      # block ids shared by all layers
    assert len({s.k_pool.data_ptr() for s in states}) == Lyr                                  # distinct KV data per layer
    pairs = []
    for l in range(Lyr):      # a Pair-shaped view per layer: the shared engine, that layer's state and oracle
        pr = Pair.__new__(Pair)
        pr.wl, pr.eng, pr.st = wls[l], eng, states[l]
        pr.prefill = {(b, h): prefill[(l, b, h)] for b in range(wl.B) for h in range(wl.Hkv)}
        pr.ob = OracleBatch(wls[l], pr.prefill)
        pr.out = torch.zeros(wl.B, wl.Hq, wl.d, dtype=torch.float32, device=DEV)
        pr.lse = torch.zeros(wl.B, wl.Hq, dtype=torch.float32, device=DEV)
        pr.last_p, pr.flips_total = wl.p, 0
        pairs.append(pr)
    assert not np.array_equal(pairs[0].prefill[(0, 0)][0], pairs[1].prefill[(0, 0)][0])
    bufs = [tuple(x.clone() for x in pr.inputs(0)[3]) for pr in pairs]

    def all_layers():
        for pr, (qd, kd, vd) in zip(pairs, bufs):
            eng.decode_step(pr.st, qd, kd, vd, wl.p, pr.out, pr.lse)

    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    snaps = [harness.snapshot(st) for st in states]
    with torch.cuda.stream(s):
        all_layers()                                      # warm-up outside capture
    torch.cuda.current_stream().wait_stream(s)
    torch.cuda.synchronize()
    for st, sn in zip(states, snaps):
        harness.restore(st, sn)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        all_layers()                                      # ONE graph over the depth of the model
    for t in range(6):
        hosts = []
        for pr, (qd, kd, vd) in zip(pairs, bufs):
            q, kn, vn, (q2, k2, v2) = pr.inputs(t)
            qd.copy_(q2); kd.copy_(k2); vd.copy_(v2)
            hosts.append((q, kn, vn))
        g.replay()
        for l, (pr, (q, kn, vn)) in enumerate(zip(pairs, hosts)):
            pr.ob.step(q, kn, vn, wl.p)
            pr.check_out(f"layer {l} step {t}")
            if pr.check_selection_band() == 0:
                pr.check_bookkeeping()
                pr.check_rewrite_exact()
                pr.check_votes()
            pr.force_discrete_state()
    assert not torch.equal(pairs[0].out, pairs[1].out)


@pytest.mark.parametrize("name", ["c1s", "c2s", "c3s", "c4s", "g1d64", "g8", "c2m", "qc4"])
def test_select_attention_overlap(name, P):
    """hardkv_decode_step launches the attention kernel programmatically behind the select kernel (it starts on the SMs
    that finished selections leave, takes the units in the order their selections finish and waits per unit on a flag).
    Bit for bit the same as plain stream order (hardkv_set_overlap(0)) on a second engine, step after step; c2m has more
    units than one wave of select CTAs leaves SMs for."""
    if name == "c2m":
        n0 = np.linspace(500, 2600, 12).astype(np.int32)
        wl = make_workload(2, B=12, n0=n0, max_ctx=2816, k_cap=384, l_upper=(n0 - 132).astype(np.int32), cond_cap=16, steps=6)
    else:
        wl = WL[name]
    a, b = P(wl, want_mask=False), P(wl, want_mask=False)
    b.eng.set_overlap(0)
    for t in range(min(wl.steps, 6)):
        q, kn, vn, (qd, knd, vnd) = a.inputs(t)
        a.eng.decode_step(a.st, qd, knd, vnd, wl.p, a.out, a.lse)
        b.eng.decode_step(b.st, qd, knd, vnd, wl.p, b.out, b.lse)
        a.ob.step(q, kn, vn, wl.p)
        a.check_out(f"{name} step {t}")
        for f in ("sel_count", "sel_idx", "sel_table", "votes", "probs", "sel_k_pool", "sel_v_pool", "cond_pos", "cond_k"):
            assert torch.equal(getattr(a.st, f), getattr(b.st, f)), (t, f)
        assert torch.equal(a.out, b.out) and torch.equal(a.lse, b.lse)
    assert int(a.st.err_flag.item()) == 0 and int(b.st.err_flag.item()) == 0
