"""Shared helpers of the -m gpu parity tests: run the CUDA path (through the C ABI binding) and the
CPU oracle on the same seeded inputs and compare.  Tolerances are BASELINE.json's north_star:
bit-exact selection / counts / tables given identical probabilities; end to end only tokens
within 1e-6 of the Top-p threshold may differ; attention max-abs 2e-2 and mean-abs 2e-3.
"""
from __future__ import annotations

import numpy as np
import torch

from oracle.batch import OracleBatch
from oracle.oracle import topp_select_row
from paper_2606_28831_b200 import harness
from workloads.synth import PAGE, Workload

OUT_MAX_ABS, OUT_MEAN_ABS, TAU_BAND = 2e-2, 2e-3, 1e-6
# The contract's band is absolute (north_star: "tokens within 1e-6 of the Top-p threshold may differ").  On flat heads
# tau itself is a few 1e-6, so the tests also hold a RELATIVE band: the two sides' fp32 probabilities agree to 2e-4
# relative (check_probs), so a token can only change sides if it sits within ~4e-4 of tau relatively; and the number
# of flips per (unit, step) is bounded.
TAU_REL_BAND, MAX_FLIPS_PER_UNIT = 1e-3, 16
DEV = "cuda:0"


def band_check(diff, P_oracle, tau, where=""):
    """Flipped tokens `diff` of one unit against the oracle's probabilities and threshold: contract band, relative band,
    flip bound.  Returns (#flips, #tokens of the unit inside the relative band)."""
    if not len(diff):
        return 0, 0
    Pd = P_oracle[diff].astype(np.float64)
    assert np.all(np.abs(Pd - tau) <= TAU_BAND), (where, "outside the contract band", diff[:8], Pd[:8], tau)
    assert np.all(np.abs(Pd - tau) <= TAU_REL_BAND * tau + 1e-12), (where, "outside the relative band", diff[:8], Pd[:8], tau)
    in_band = int(np.count_nonzero(np.abs(P_oracle.astype(np.float64) - tau) <= TAU_REL_BAND * tau + 1e-12))
    assert len(diff) <= min(in_band, MAX_FLIPS_PER_UNIT), (where, "too many flips", len(diff), in_band)
    return len(diff), in_band


def np_of(t: torch.Tensor) -> np.ndarray:
    return t.detach().float().cpu().numpy() if t.dtype == torch.bfloat16 else t.detach().cpu().numpy()


class Pair:
    """CUDA engine + device state and the oracle, built from one workload and one prefill."""

    def __init__(self, wl: Workload, want_mask=True, reuse_max=0):
        self.wl = wl
        self.eng = harness.make_engine(wl, DEV, reuse_max=reuse_max)
        (self.st,), self.prefill = harness.make_state(wl, DEV, want_mask=want_mask)
        self.ob = OracleBatch(wl, self.prefill)
        self.out = torch.zeros(wl.B, wl.Hq, wl.d, dtype=torch.float32, device=DEV)
        self.lse = torch.zeros(wl.B, wl.Hq, dtype=torch.float32, device=DEV)
        self.last_p = wl.p          # nucleus mass of the last select call (tests that sweep p set it)
        self.flips_total = 0

    def inputs(self, t: int):
        wl = self.wl
        q = wl.step_q(t)
        k_new, v_new = wl.step_kv(t, {u: kv[0] for u, kv in self.prefill.items()} if wl.mix_new_keys else None)
        return q, k_new, v_new, (harness.to_dev(q, wl, DEV), harness.to_dev(k_new, wl, DEV),
                                 harness.to_dev(v_new, wl, DEV))

    # ---- comparisons ---------------------------------------------------------------------------
    def check_bookkeeping(self):
        wl, st, ob = self.wl, self.st, self.ob
        assert int(np_of(st.err_flag)[0]) == 0
        np.testing.assert_array_equal(np_of(st.ctx_len), ob.ctx_len())
        np.testing.assert_array_equal(np_of(st.c_lo), ob.c_lo())
        np.testing.assert_array_equal(np_of(st.dense_lo), ob.dense_lo())
        np.testing.assert_array_equal(np_of(st.cond_count), ob.cond_count())
        cpos, cvot = np_of(st.cond_pos), np_of(st.cond_votes)
        ck, cv = np_of(st.cond_k), np_of(st.cond_v)
        for i, u in enumerate(ob.units):
            c = u.cond_count
            np.testing.assert_array_equal(cpos[i, :c], u.cond_pos[:c])
            np.testing.assert_array_equal(cvot[i, :c], u.cond_votes[:c])
            if wl.cond_merge:    # merged rows: fp32 vs fp64 arithmetic before the store rounding, one ulp of kv_dtype
                tol = dict(rtol=2.0 ** -7, atol=1e-6) if wl.dtype == "bf16" else dict(rtol=1e-5, atol=1e-6)
                np.testing.assert_allclose(ck[i, :c], u.cond_k[:c], **tol)
                np.testing.assert_allclose(cv[i, :c], u.cond_v[:c], **tol)
            else:
                np.testing.assert_array_equal(ck[i, :c], u.cond_k[:c])   # row copies: bit exact
                np.testing.assert_array_equal(cv[i, :c], u.cond_v[:c])

    def check_votes(self):
        votes = np_of(self.st.votes)
        for i, u in enumerate(self.ob.units):
            np.testing.assert_array_equal(votes[i], u.votes)

    def check_selection_exact(self):
        wl, st, ob = self.wl, self.st, self.ob
        np.testing.assert_array_equal(np_of(st.sel_count), ob.sel_count())
        np.testing.assert_array_equal(np_of(st.sel_idx), ob.sel_idx())
        _, sel_pages = wl.page_tables()
        sel_pages = sel_pages.reshape(wl.B * wl.Hkv, -1)
        tab = np_of(st.sel_table)
        mask = np_of(st.sel_mask) if st.sel_mask is not None else None
        for i, u in enumerate(ob.units):
            np.testing.assert_array_equal(tab[i], u.sel_table(sel_pages[i]))
            if mask is not None:
                np.testing.assert_array_equal(mask[i], u.sel_mask())
        self.check_votes()

    def check_selection_band(self, own_probs=True):
        """End to end.  (1) The contract: the symmetric difference to the oracle's selection holds only tokens within
        TAU_BAND (absolute) of the oracle threshold -- and, stricter, within a relative band of it, and only a bounded
        number of them.  (2) Band-free evidence: the CUDA selection is bit for bit what the oracle's Top-p rule selects
        from the CUDA path's own stored fp32 probabilities (which check_probs ties to the oracle's to 2e-4 relative)."""
        st, ob, wl = self.st, self.ob, self.wl
        cnt, idx = np_of(st.sel_count), np_of(st.sel_idx)
        probs = np_of(st.probs) if own_probs else None
        flips = 0
        for i, u in enumerate(ob.units):
            a = set(idx[i, :cnt[i]].tolist())
            b = set(u.sel_idx[:u.sel_count].tolist())
            assert sorted(a) == idx[i, :cnt[i]].tolist(), "sel_idx must be ascending"
            tau = float(np.array([u.tau_bits], np.uint32).view(np.float32)[0])
            f, _ = band_check(sorted(a ^ b), u.probs, tau, where=f"unit {i}")
            flips += f
            if own_probs:
                lo, hi = u.pool
                sel, k, _, _ = topp_select_row(ob.cfg, probs[i], lo, hi, int(wl.l_lower[i // wl.Hkv]), self.last_p)
                assert k == cnt[i], (i, k, cnt[i])
                np.testing.assert_array_equal(idx[i, :k], sel)
        self.flips_total += flips
        return flips

    def check_rewrite_exact(self):
        wl, st, ob = self.wl, self.st, self.ob
        sk, sv = np_of(st.sel_k_pool), np_of(st.sel_v_pool)
        _, sel_pages = wl.page_tables()
        sel_pages = sel_pages.reshape(wl.B * wl.Hkv, -1)
        for i, u in enumerate(ob.units):
            k = u.sel_count
            kend = (k + PAGE - 1) // PAGE * PAGE
            if kend == 0:
                continue
            rows_k = sk[sel_pages[i, :kend // PAGE]].reshape(kend, wl.d)
            rows_v = sv[sel_pages[i, :kend // PAGE]].reshape(kend, wl.d)
            np.testing.assert_array_equal(rows_k, u.sel_k[:kend])   # includes the zero tail
            np.testing.assert_array_equal(rows_v, u.sel_v[:kend])

    def check_out(self, what=""):
        o, ref = np_of(self.out), self.ob.out()
        err = np.abs(o - ref)
        assert np.isfinite(o).all(), what
        assert err.max() <= OUT_MAX_ABS and err.mean() <= OUT_MEAN_ABS, (what, err.max(), err.mean())
        np.testing.assert_allclose(np_of(self.lse), self.ob.lse(), atol=2e-3, rtol=1e-4)
        return float(err.max()), float(err.mean())

    def check_logits(self):
        wl = self.wl
        lg = np_of(self.st.logits).reshape(wl.B * wl.Hkv, wl.G, wl.max_ctx)
        for i, u in enumerate(self.ob.units):
            lo, hi = u.pool
            np.testing.assert_allclose(lg[i][:, lo:hi], u.logits[:, lo:hi], atol=3e-4, rtol=2e-5)

    def check_probs(self):
        pr = np_of(self.st.probs)
        for i, u in enumerate(self.ob.units):
            lo, hi = u.pool
            np.testing.assert_allclose(pr[i, lo:hi], u.probs[lo:hi], atol=2e-7, rtol=2e-4)

    # ---- teacher forcing: overwrite the CUDA path's discrete state with the oracle's --------------
    def force_discrete_state(self):
        st, ob, wl = self.st, self.ob, self.wl
        st.votes.copy_(torch.from_numpy(np.stack([u.votes for u in ob.units])))
        st.cond_pos.copy_(torch.from_numpy(np.stack([u.cond_pos for u in ob.units])))
        st.cond_votes.copy_(torch.from_numpy(np.stack([u.cond_votes for u in ob.units])))
        st.cond_count.copy_(torch.from_numpy(ob.cond_count()))
        st.cond_k.copy_(harness.to_dev(np.stack([u.cond_k for u in ob.units]), wl, DEV))
        st.cond_v.copy_(harness.to_dev(np.stack([u.cond_v for u in ob.units]), wl, DEV))

    def adopt_cuda_discrete_state(self):
        """Free-running runs: after a near-threshold flip the ORACLE adopts the CUDA path's discrete state (selection,
        votes, condensed tier), so that every later step is still compared like for like instead of being skipped."""
        st, ob, wl = self.st, self.ob, self.wl
        votes, cpos, cvot = np_of(st.votes), np_of(st.cond_pos), np_of(st.cond_votes)
        ck, cv, ccnt = np_of(st.cond_k), np_of(st.cond_v), np_of(st.cond_count)
        cnt, idx = np_of(st.sel_count), np_of(st.sel_idx)
        for i, u in enumerate(ob.units):
            u.votes[:] = votes[i]
            u.cond_pos[:], u.cond_votes[:] = cpos[i], cvot[i]
            u.cond_k[:], u.cond_v[:] = ck[i], cv[i]
            u.u.cond_count = int(ccnt[i])
            u.sel_idx[:] = idx[i]
            u.u.sel_count = int(cnt[i])
            u.rewrite()

    def upload_oracle_probs(self):
        self.st.probs.copy_(torch.from_numpy(np.stack([u.probs for u in self.ob.units])))
