"""-m gpu parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (the fused
hardkv_decode_step over the whole batch, replayed from a captured CUDA graph where the config says so), judged on
SAMPLED units the oracle computes one by one -- or on every unit where the oracle can follow (config 3 at B = 4).

Per sampled (sequence, KV head) and step: selection (contract band 1e-6 absolute, plus the relative band and flip bound
of gpu_common.band_check; and, band-free, the CUDA selection equals the oracle's Top-p rule applied to the CUDA path's
own stored probabilities bit for bit), sel_count, sel_table, the rewritten K AND V rows with the zero tail, votes, the
condensed tier (positions, votes, K / V rows), ctx_len / c_lo / dense_lo, and attention outputs (max-abs 2e-2,
mean-abs 2e-3).  After a near-threshold flip the sampled units are teacher-forced so later steps stay comparable.
"""
import numpy as np
import pytest
import torch

from gpu_common import OUT_MAX_ABS, OUT_MEAN_ABS, Pair, band_check
from oracle.oracle import OracleConfig, Unit, decode_step_batch, topp_select_row
from paper_2606_28831_b200 import harness
from workloads.synth import PAGE, make_workload

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


class Sampled:
    """The fused CUDA step over a whole full-size batch + oracle units for a sample of its (b, h) pairs."""

    def __init__(self, wl, sample, prefill=None, graph=False):
        self.wl, self.sample = wl, sample
        self.eng = harness.make_engine(wl, DEV)
        (self.st,), self.prefill = harness.make_state(wl, DEV, prefill=prefill, retain=set(sample))
        self.cfg = OracleConfig(G=wl.G, d=wl.d, max_ctx=wl.max_ctx, sink=wl.sink, recent=wl.recent, k_cap=wl.k_cap,
                                cond_cap=wl.cond_cap, accum_window=wl.accum_window, sm_scale=float(wl.sm_scale),
                                pool_kernel=wl.pool_kernel)
        self.snap = harness.snapshot(self.st)
        self.pk = {u: kv[0] for u, kv in self.prefill.items()} if wl.mix_new_keys else None
        self.out = torch.zeros(wl.B, wl.Hq, wl.d, dtype=torch.float32, device=DEV)
        _, self.sel_pages = wl.page_tables()
        tdt = harness.torch_dtype(wl)
        self.qd = torch.zeros(wl.B, wl.Hq, wl.d, dtype=tdt, device=DEV)
        self.kd = torch.zeros(wl.B, wl.Hkv, wl.d, dtype=tdt, device=DEV)
        self.vd = torch.zeros(wl.B, wl.Hkv, wl.d, dtype=tdt, device=DEV)
        self.graph, self.use_graph = None, graph
        self.reset()

    def reset(self):
        wl = self.wl
        harness.restore(self.st, self.snap)
        self.units = [Unit(self.cfg, *self.prefill[(b, h)], l_upper=int(wl.l_upper[b]), l_lower=int(wl.l_lower[b]),
                           T=float(wl.temperature[b, h]), score_mode=int(wl.score_mode[h])) for b, h in self.sample]
        self.flips = self.in_band = 0
        self.emax = 0.0
        self.graph = None

    def step(self, t, p, full_check=True):
        wl, st, sample, units = self.wl, self.st, self.sample, self.units
        q = wl.step_q(t)
        kn, vn = wl.step_kv(t, self.pk)
        self.qd.copy_(harness.to_dev(q, wl, DEV)); self.kd.copy_(harness.to_dev(kn, wl, DEV))
        self.vd.copy_(harness.to_dev(vn, wl, DEV))
        if self.use_graph:
            if self.graph is None:      # captured ONCE (static shapes, counts on the device: L53, L63), replayed every step
                s = torch.cuda.Stream()
                s.wait_stream(torch.cuda.current_stream())
                snap = harness.snapshot(st)
                with torch.cuda.stream(s):
                    self.eng.decode_step(st, self.qd, self.kd, self.vd, p, self.out)   # warm-up outside capture
                torch.cuda.current_stream().wait_stream(s)
                torch.cuda.synchronize()
                harness.restore(st, snap)
                self.graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(self.graph):
                    self.eng.decode_step(st, self.qd, self.kd, self.vd, p, self.out)
            self.graph.replay()
        else:
            self.eng.decode_step(st, self.qd, self.kd, self.vd, p, self.out)
        qs = np.stack([q[b, h * wl.G:(h + 1) * wl.G] for b, h in sample])
        decode_step_batch(units, qs, np.stack([kn[b, h] for b, h in sample]), np.stack([vn[b, h] for b, h in sample]), p)
        torch.cuda.synchronize()
        assert int(st.err_flag.item()) == 0
        o = self.out.cpu().numpy()
        rows = torch.tensor([b * wl.Hkv + h for b, h in sample], device=DEV)
        cnt = st.sel_count[rows].cpu().numpy()
        idx = st.sel_idx[rows].cpu().numpy()
        ctx, clo, dlo = st.ctx_len.cpu().numpy(), st.c_lo.cpu().numpy(), st.dense_lo.cpu().numpy()
        errs, flipped = [], False
        for j, ((b, h), u) in enumerate(zip(sample, units)):
            assert (ctx[b], clo[b], dlo[b]) == (u.n, u.c_lo, u.dense_lo), (t, b, h)
            a, r = idx[j, :cnt[j]], u.sel_idx[:u.sel_count]
            assert np.all(np.diff(a) > 0), "sel_idx must be ascending"
            tau = float(np.array([u.tau_bits], np.uint32).view(np.float32)[0])
            f, nb = band_check(sorted(set(a.tolist()) ^ set(r.tolist())), u.probs, tau, where=f"step {t} unit {(b, h)}")
            self.flips += f
            self.in_band += nb
            flipped |= f > 0
            errs.append(np.abs(o[b, h * wl.G:(h + 1) * wl.G] - u.out))
        e = np.stack(errs)
        assert np.isfinite(o).all() and e.max() <= OUT_MAX_ABS and e.mean() <= OUT_MEAN_ABS, (t, e.max(), e.mean())
        self.emax = max(self.emax, float(e.max()))
        if full_check or flipped:
            self.full_check(t, p, cnt, idx)
        if flipped:
            self.teacher_force()

    def full_check(self, t, p, cnt, idx):
        """Everything the step writes for the sampled units, against the oracle (exact unless a flip excuses it)."""
        wl, st = self.wl, self.st
        rows = torch.tensor([b * wl.Hkv + h for b, h in self.sample], device=DEV)
        probs = st.probs[rows].cpu().numpy()
        votes = st.votes[rows].cpu().numpy()
        tab = st.sel_table[rows].cpu().numpy()
        ccnt = st.cond_count[rows].cpu().numpy()
        cpos, cvot = st.cond_pos[rows].cpu().numpy(), st.cond_votes[rows].cpu().numpy()
        ck, cv = st.cond_k[rows].float().cpu().numpy(), st.cond_v[rows].float().cpu().numpy()
        for j, ((b, h), u) in enumerate(zip(self.sample, self.units)):
            where = f"step {t} unit {(b, h)}"
            # band-free: the CUDA selection is the oracle's Top-p rule on the CUDA path's own probabilities, bit for bit
            lo, hi = u.pool
            sel, k, _, _ = topp_select_row(self.cfg, probs[j], lo, hi, int(wl.l_lower[b]), p)
            assert k == cnt[j], where
            np.testing.assert_array_equal(idx[j, :k], sel, err_msg=where)
            np.testing.assert_allclose(probs[j, lo:hi], u.probs[lo:hi], atol=2e-7, rtol=2e-4, err_msg=where)
            used = (k + PAGE - 1) // PAGE
            sp = self.sel_pages[b, h]
            np.testing.assert_array_equal(tab[j], np.where(np.arange(len(sp)) < used, sp, -1), err_msg=where)
            # rewritten rows (K and V) + zero tail: byte-exact copies of the base rows the CUDA path selected
            if used:
                pages = torch.from_numpy(sp[:used].astype(np.int64)).to(DEV)
                rk = st.sel_k_pool[pages].reshape(used * PAGE, wl.d).float().cpu().numpy()
                rv = st.sel_v_pool[pages].reshape(used * PAGE, wl.d).float().cpu().numpy()
                np.testing.assert_array_equal(rk[:k], u.K[idx[j, :k]], err_msg=where)
                np.testing.assert_array_equal(rv[:k], u.V[idx[j, :k]], err_msg=where)
                assert not rk[k:].any() and not rv[k:].any(), where
            if np.array_equal(idx[j, :k], u.sel_idx[:u.sel_count]):
                np.testing.assert_array_equal(votes[j], u.votes, err_msg=where)
            c = u.cond_count
            assert ccnt[j] == c, where
            np.testing.assert_array_equal(cpos[j, :c], u.cond_pos[:c], err_msg=where)
            np.testing.assert_array_equal(cvot[j, :c], u.cond_votes[:c], err_msg=where)
            np.testing.assert_array_equal(ck[j, :c], u.cond_k[:c], err_msg=where)
            np.testing.assert_array_equal(cv[j, :c], u.cond_v[:c], err_msg=where)

    def teacher_force(self):
        wl, st = self.wl, self.st
        for (b, h), u in zip(self.sample, self.units):
            i = b * wl.Hkv + h
            st.votes[i].copy_(torch.from_numpy(u.votes))

    def report(self, what):
        print(f"[{what}] near-threshold flips {self.flips} (tokens of the sampled units inside the relative band, summed "
              f"over flipped unit-steps: {self.in_band}), max-abs output error {self.emax:.2e}")


def run_sampled(wl, sample, steps, p=None, graph=False):
    s = Sampled(wl, sample, graph=graph)
    for t in range(steps):
        s.step(t, wl.p if p is None else p)
    s.report(f"{wl.name} {steps} steps")
    return s


def test_config2_full_size_sampled():
    """The bench workload in the bench's launch configuration: one captured graph of the fused step, replayed."""
    wl = make_workload(2)
    order = np.argsort(wl.n0)
    sample = [(int(order[0]), 0), (int(order[-1]), 7), (int(order[len(order) // 2]), 3), (int(order[-2]), 1),
              (int(order[1]), 5), (int(order[-1]), 2)]
    run_sampled(wl, sample, steps=6, graph=True)


def test_config1_full_size_sampled():
    wl = make_workload(1)
    run_sampled(wl, [(0, h) for h in (0, 3, 7)], steps=4)


def _condensed_tier_invariants(pr, where):
    """The CUDA path's discrete state judged WITHOUT the oracle's trajectory (pins P10 / P11 restated on device data):
    votes freeze when a token retires, so for every unit the condensed residents must be exactly the top-C_cap of the
    retired positions [sink, c_lo) by (votes, position), cond_votes must equal the votes of those positions, and the
    rows must be byte copies of the base rows (generator data held in the oracle units' K / V arrays)."""
    wl, st, ob = pr.wl, pr.st, pr.ob
    votes, cpos, cvot = (x.cpu().numpy() for x in (st.votes, st.cond_pos, st.cond_votes))
    ccnt, clo = st.cond_count.cpu().numpy(), st.c_lo.cpu().numpy()
    ck, cv = st.cond_k.float().cpu().numpy(), st.cond_v.float().cpu().numpy()
    for i, u in enumerate(ob.units):
        b = i // wl.Hkv
        retired = np.arange(wl.sink, clo[b])
        c = min(len(retired), wl.cond_cap)
        assert ccnt[i] == c, (where, i)
        if c == 0:
            continue
        order = np.lexsort((retired, votes[i, retired]))[::-1][:c]          # largest (votes, pos) first
        assert set(cpos[i, :c].tolist()) == set(retired[order].tolist()), (where, i, "residents != top-C of the retired")
        np.testing.assert_array_equal(cvot[i, :c], votes[i, cpos[i, :c]], err_msg=f"{where} unit {i}")
        np.testing.assert_array_equal(ck[i, :c], u.K[cpos[i, :c]], err_msg=f"{where} unit {i}")
        np.testing.assert_array_equal(cv[i, :c], u.V[cpos[i, :c]], err_msg=f"{where} unit {i}")


def test_config3_full_trajectory_one_graph_b4():
    """BASELINE configs[3] as it is defined, at B = 4: 1024-token prefill, then the context is grown to
    12288 by 11264 appended tokens, every shape padded to the static capacity and the WHOLE run replayed from ONE
    captured single-step graph (L53, L63, L168).  The plain oracle needs ~0.1-0.2 s per step for the 16 (sequence, KV
    head) units at the full pool, so it follows the run in WINDOWS (the first 192 steps, then around n = 2048, 4096, the
    start of retirement at n = 8453, and the last 64 steps up to 12288), all 16 units, every step of a window compared
    (selection bands + flip bound + own-probability selection, outputs, bookkeeping, votes, rewritten rows), teacher
    forced on flips.  Between windows the CUDA path runs alone; at the start of the next window its discrete state is
    first judged on its own (condensed tier == top-C of the retired tokens by votes, vote totals == sum of the per-step
    budgets, arithmetic ctx_len / c_lo / dense_lo) and then adopted by the oracle."""
    wl = make_workload(3, B=4)
    pr = Pair(wl, want_mask=False)
    eng, st, ob = pr.eng, pr.st, pr.ob
    q, kn, vn, (qd, knd, vnd) = pr.inputs(0)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    snap = harness.snapshot(st)
    with torch.cuda.stream(s):
        eng.decode_step(st, qd, knd, vnd, wl.p, pr.out, pr.lse)      # warm-up outside capture
    torch.cuda.current_stream().wait_stream(s)
    torch.cuda.synchronize()
    harness.restore(st, snap)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        eng.decode_step(st, qd, knd, vnd, wl.p, pr.out, pr.lse)
    n0 = int(wl.n0[0])
    steps = wl.max_ctx - n0
    assert steps == 11264
    t_of = lambda n: n - n0 - 1                                       # the step after which ctx_len == n
    windows = [(0, 192), (t_of(2048) - 40, t_of(2048) + 24), (t_of(4096) - 40, t_of(4096) + 24),
               (t_of(8453) - 30, t_of(8453) + 70), (steps - 64, steps)]
    in_window = np.zeros(steps, bool)
    for a_, b_ in windows:
        in_window[a_:b_] = True
    flips, emax, first_flip, kmax, votes_total, compared = 0, 0.0, None, 0, 0, 0
    synced = True                                                     # oracle state == CUDA state (modulo checks)
    for t in range(steps):
        q, kn, vn, (q2, k2, v2) = pr.inputs(t)
        qd.copy_(q2); knd.copy_(k2); vnd.copy_(v2)
        if in_window[t] and not synced:
            # ---- judge the CUDA path's state on its own, then let the oracle adopt it -------------------------------
            where = f"adoption before step {t}"
            n = n0 + t
            assert (st.ctx_len.cpu().numpy() == n).all() and int(st.err_flag.item()) == 0
            clo = max(wl.sink, n - wl.recent - int(wl.l_upper[0]))
            assert (st.c_lo.cpu().numpy() == clo).all() and (st.dense_lo.cpu().numpy() == n - wl.recent).all()
            assert int(st.votes.sum().item()) == votes_total, where           # P11: sum of votes == sum of budgets
            _condensed_tier_invariants(pr, where)
            for u in ob.units:
                u.u.n, u.u.c_lo, u.u.dense_lo = n, clo, n - wl.recent
            pr.adopt_cuda_discrete_state()
            synced = True
        g.replay()
        kvf = (kn.reshape(-1, wl.d), vn.reshape(-1, wl.d))
        if in_window[t]:
            ob.step(q, kn, vn, wl.p)
            e, _ = pr.check_out(f"c3 step {t}")
            emax = max(emax, e)
            f = pr.check_selection_band(own_probs=True)
            pr.check_probs()
            if f == 0:
                pr.check_bookkeeping()
                pr.check_votes()
                pr.check_rewrite_exact()
            else:
                flips += f
                first_flip = t if first_flip is None else first_flip
                pr.force_discrete_state()
            compared += 1
        else:
            for i, u in enumerate(ob.units):                          # the oracle's base rows follow the generator
                u.K[n0 + t], u.V[n0 + t] = kvf[0][i], kvf[1][i]
            synced = False
        cnt = st.sel_count.cpu().numpy()
        assert (cnt <= wl.k_cap).all()
        kmax = max(kmax, int(cnt.max()))
        votes_total += int(cnt.sum())
    assert int(st.ctx_len.max()) == wl.max_ctx and int(st.err_flag.item()) == 0
    assert int(st.votes.sum().item()) == votes_total
    _condensed_tier_invariants(pr, "end of the trajectory")
    assert all(u.cond_count == wl.cond_cap for u in ob.units)       # the pool passed l_upper: the condensed tier filled
    assert kmax == wl.k_cap                                         # the static capacity clamp was reached (L233)
    print(f"[c3 B=4 full trajectory, one graph, {steps} steps, {compared} of them beside the oracle] flips {flips} "
          f"(first at step {first_flip}), max-abs output error {emax:.2e}")


@pytest.fixture(scope="module")
def c3_prefill():
    """Prefill rows of config 3 at B = 32 for the longest checkpoint; shorter checkpoints take a prefix (any seeded rows
    serve: both sides consume the same arrays)."""
    wl = make_workload(3, n0=np.full(32, 12280, np.int32))
    return {(b, h): wl.prefill_unit(b, h) for b in range(wl.B) for h in range(wl.Hkv)}


@pytest.mark.parametrize("n_end", [2048, 4096, 8192, 12288])
def test_config3_b32_checkpoints(n_end, c3_prefill):
    """Config 3 at its full batch (B = 32) at the checkpoints of SURVEY 8(d): 8 fused steps ending at n_end, replayed
    from one graph, on sampled units.  The state is built directly at n_end - 8 (fresh votes; the carried state is what
    the B = 4 trajectory covers): below l_upper = 8192 nothing retires; above it the first step retires the whole
    excess at once (thousands of tokens through the 256 slots) and the pool stays pinned at l_upper."""
    n0 = n_end - 8
    wl = make_workload(3, n0=np.full(32, n0, np.int32))
    sample = [(0, 0), (13, 2), (31, 3), (20, 1)]
    pre = {u: (kv[0][:n0], kv[1][:n0]) for u, kv in c3_prefill.items()}
    s = Sampled(wl, sample, prefill=pre, graph=True)
    for t in range(8):
        s.step(t, wl.p)
    assert int(s.st.ctx_len.max()) == n_end
    s.report(f"c3 B=32 checkpoint n={n_end}")


@pytest.fixture(scope="module")
def c4_state():
    wl = make_workload(4)
    # RAW heads 1 and 3, ACCUM heads 4, 6 and 7 (the 32-deep ring; the select kernel runs as a cluster of 4 CTAs here)
    sample = [(0, 1), (3, 6), (7, 4), (5, 7), (2, 3)]
    return Sampled(wl, sample, graph=True)


@pytest.mark.parametrize("p", [0.8, 0.9, 0.95, 0.99])
def test_config4_full_size_sweep_ring_wraps(p, c4_state):
    """BASELINE configs[4] at full size (B 8, 40 q / 8 KV heads, 64k context, half the heads on accumulated attention):
    40 fused steps per p so the 32-deep ACCUM ring fills AND wraps at 64k under the cluster select path, at all four p
    of the sweep, each from one captured graph.  Full checks on the first steps, around the wrap, and at the end."""
    s = c4_state
    s.reset()
    steps = 40
    for t in range(steps):
        s.step(t, p, full_check=(t < 2 or t in (31, 32, 33) or t == steps - 1))
    for (b, h), u in zip(s.sample, s.units):
        if s.wl.score_mode[h] == 1:
            assert u.u.ring_slot == steps % s.wl.accum_window     # the ring wrapped
    s.report(f"c4 p={p} {steps} steps")


def test_config4_full_size_query_cache_recompute():
    """SURVEY 8(f)-1 / PAPER.md L448: BASELINE configs[4] with its accumulated-attention heads (4-7) on the query-cache
    form -- the last 32 queries score the CURRENT 64k pool (M = 160 query rows per unit, a real contraction) instead of
    summing a ring of per-step rows.  40 steps so the query window fills and wraps; sampled units against the oracle."""
    wl = make_workload(4, score_mode=np.array([0, 0, 0, 0, 3, 3, 3, 3], np.uint8))
    s = Sampled(wl, [(0, 1), (3, 6), (7, 4), (5, 7)], graph=True)
    steps = 36
    for t in range(steps):
        s.step(t, 0.9, full_check=(t < 2 or t in (31, 32, 33) or t == steps - 1))
    assert all(u.u.qc_count == wl.accum_window for (b, h), u in zip(s.sample, s.units) if wl.score_mode[h] == 3)
    s.report(f"c4 query-cache ACCUM p=0.9 {steps} steps")


def test_config2_full_size_snapkv_solve_then_step():
    """Full-size config 2 with half the KV heads on the SNAPKV metric (window 7): Algorithm 2 solves T on the first
    step's logits (sampled units against the oracle's bisection, 1e-3 relative), then fused steps run with the
    solved temperatures (L607: solve at the first compression, reuse afterwards)."""
    wl = make_workload(2, score_mode=np.array([0, 2, 0, 2, 0, 2, 0, 2], np.uint8), pool_kernel=7)
    order = np.argsort(wl.n0)
    sample = [(int(order[0]), 1), (int(order[-1]), 7), (int(order[len(order) // 2]), 2), (int(order[-1]), 3)]
    s = Sampled(wl, sample)
    eng, st, units = s.eng, s.st, s.units
    q = wl.step_q(0)
    kn, vn = wl.step_kv(0, None)
    qd, knd, vnd = (harness.to_dev(x, wl, DEV) for x in (q, kn, vn))
    eng.append_kv(st, knd, vnd)
    eng.score(st, qd)
    eng.solve_temperature(st, wl.p, t_min=0.0625, t_max=16.0, eps=1e-5, max_iter=40)
    T = st.temperature.cpu().numpy()
    # sharp heads select fewer tokens than one pooling window holds copies of the top logit: no T matches the mass
    # (the paper's "failure cases ... illness of the problem", L605) and the bisection runs into T_min
    assert np.isfinite(T).all() and (T >= 0.0625).all() and (T <= 16.0).all()
    raw = T[:, 0::2]
    assert np.abs(raw - 1.0).max() < 5e-3                       # g = id heads: T* = 1 (pin P13)
    for (b, h), u in zip(sample, units):
        u.append(kn[b, h], vn[b, h]); u.retire()
        u.score(q[b, h * wl.G:(h + 1) * wl.G])
        it, resid = u.solve_temperature(wl.p, t_min=0.0625, t_max=16.0, eps=1e-5, max_iter=40)
        assert abs(T[b, h] - u.T) <= 1e-3 * u.T, (b, h, T[b, h], u.T)
        assert resid <= 1e-5 or u.T < 0.0626 or it == 40, (b, h, resid, u.T, it)
        u.u.T = np.float32(T[b, h])
    # the rest of step 0 (select + rewrite + attend with the solved T), then fused steps
    eng.calibrate_topp(st, wl.p)
    eng.rewrite_attend(st, qd, s.out)
    for (b, h), u in zip(sample, units):
        u.calibrate(); u.topp_select(wl.p, True); u.rewrite(); u.attend(q[b, h * wl.G:(h + 1) * wl.G])
    torch.cuda.synchronize()
    o = s.out.cpu().numpy()
    rows = torch.tensor([b * wl.Hkv + h for b, h in sample], device=DEV)
    cnt, idx = st.sel_count[rows].cpu().numpy(), st.sel_idx[rows].cpu().numpy()
    flipped = False
    for j, ((b, h), u) in enumerate(zip(sample, units)):
        tau = float(np.array([u.tau_bits], np.uint32).view(np.float32)[0])
        f, _ = band_check(sorted(set(idx[j, :cnt[j]].tolist()) ^ set(u.sel_idx[:u.sel_count].tolist())), u.probs, tau,
                          where=f"solve step unit {(b, h)}")
        flipped |= f > 0
        e = np.abs(o[b, h * wl.G:(h + 1) * wl.G] - u.out)
        assert e.max() <= OUT_MAX_ABS and e.mean() <= OUT_MEAN_ABS, (b, h, e.max())
    s.full_check(0, wl.p, cnt, idx)
    s.teacher_force()
    for t in (1, 2):
        s.step(t, wl.p)
    s.report("c2 snapkv + solved T")
