"""Pins P1-P12 of the CPU oracle: the oracle is checked
against what the paper and the mathematics fix, never against itself or the CUDA path.

Citations are PAPER.md lines: Top-p/M_k L108, order invariance L116 + Thm D.3,
budget vs temperature L72-74/L100, exact tiered attention L84, Eq. 4-6,
votes L86, Tier 3 L76.
"""
import itertools
import math

import numpy as np
import pytest
import scipy.special
import scipy.stats
import torch

from oracle.oracle import OracleConfig, Unit, merge, state_of_set


def _unit(G=4, d=64, n0=200, max_ctx=256, s=4, W=16, k_cap=256, C=8, l_upper=10**6, seed=0, T=1.0, mode=0,
          l_lower=0, sm_scale=None):
    rng = np.random.default_rng(seed)
    cfg = OracleConfig(G=G, d=d, max_ctx=max_ctx, sink=s, recent=W, k_cap=k_cap, cond_cap=C, sm_scale=sm_scale)
    K0 = rng.standard_normal((n0, d)).astype(np.float32)
    V0 = rng.standard_normal((n0, d)).astype(np.float32)
    return cfg, Unit(cfg, K0, V0, l_upper=l_upper, l_lower=l_lower, T=T, score_mode=mode), rng


def _set_logits(u: Unit, z):
    """Write a [G][N] logit block onto the pool of u."""
    lo, hi = u.pool
    z = np.atleast_2d(np.asarray(z, np.float32))
    assert z.shape[1] == hi - lo
    u.logits[:, lo:hi] = z


def _w(P):
    return np.rint(P.astype(np.float64) * 4294967296.0).astype(np.uint64)


# ---- P1: p = 1 => selected = whole pool and the tiered output is dense attention (L84) ---------
@pytest.mark.parametrize("G,d", [(4, 64), (7, 128)])
def test_p1_dense_equivalence(G, d):
    cfg, u, rng = _unit(G=G, d=d, n0=200, max_ctx=256, W=16, k_cap=256)
    for t in range(5):
        q = (rng.standard_normal((G, d)) * 1.7).astype(np.float32)
        kn, vn = rng.standard_normal(d).astype(np.float32), rng.standard_normal(d).astype(np.float32)
        u.decode_step(q, kn, vn, p=1.0)
        n = u.n
        lo, hi = u.pool
        assert u.sel_count == hi - lo and list(u.sel_idx[:u.sel_count]) == list(range(lo, hi))
        Kt = torch.tensor(u.K[:n], dtype=torch.float64)[None]
        Vt = torch.tensor(u.V[:n], dtype=torch.float64)[None]
        qt = torch.tensor(q, dtype=torch.float64)[:, None, :]
        ref = torch.nn.functional.scaled_dot_product_attention(qt, Kt.expand(G, -1, -1), Vt.expand(G, -1, -1))
        np.testing.assert_allclose(u.out, ref[:, 0].numpy(), rtol=0, atol=1e-5)
        x = (qt[:, 0] @ Kt[0].T) / math.sqrt(d)
        np.testing.assert_allclose(u.lse, torch.logsumexp(x, -1).numpy(), rtol=0, atol=1e-5)


def test_p1_with_condensed_and_retired_is_not_dense_but_subset_exact():
    """With retirement on, the output is exact attention over D u I u C (L84), checked by SDPA on that set."""
    cfg, u, rng = _unit(G=2, d=64, n0=120, max_ctx=160, W=8, k_cap=160, C=4, l_upper=60)
    for t in range(6):
        q = rng.standard_normal((2, 64)).astype(np.float32)
        u.decode_step(q, rng.standard_normal(64).astype(np.float32), rng.standard_normal(64).astype(np.float32), p=1.0)
    live = list(range(cfg.sink)) + list(range(u.c_lo, u.n)) + list(u.cond_pos[:u.cond_count])
    assert len(set(live)) == len(live)
    Kt = torch.tensor(u.K[live], dtype=torch.float64)[None].expand(2, -1, -1)
    Vt = torch.tensor(u.V[live], dtype=torch.float64)[None].expand(2, -1, -1)
    ref = torch.nn.functional.scaled_dot_product_attention(torch.tensor(q, dtype=torch.float64)[:, None], Kt, Vt)
    np.testing.assert_allclose(u.out, ref[:, 0].numpy(), atol=1e-5, rtol=0)


# ---- score: closed forms (unit-vector queries; LSE identity with the pinned attention state) ---
def test_score_closed_forms():
    cfg, u, rng = _unit(G=4, d=64, n0=100, max_ctx=128, W=10, sm_scale=0.25)
    lo, hi = u.pool
    q = np.zeros((4, 64), np.float32)
    for g, (j, a) in enumerate([(0, 1.0), (5, -2.0), (63, 0.5), (17, 3.0)]):
        q[g, j] = a
    u.score(q)
    for g, (j, a) in enumerate([(0, 1.0), (5, -2.0), (63, 0.5), (17, 3.0)]):
        np.testing.assert_array_equal(u.logits[g, lo:hi], (np.float64(0.25) * a * u.K[lo:hi, j].astype(np.float64)).astype(np.float32))
    q = rng.standard_normal((4, 64)).astype(np.float32)
    u.score(q)
    for g in range(4):   # log-sum-exp of the scores == LSE of the attention state over the same rows
        _, m, l = state_of_set(cfg, q[g], u.K, u.V, np.arange(lo, hi))
        assert abs(scipy.special.logsumexp(u.logits[g, lo:hi].astype(np.float64)) - (m + math.log(l))) < 1e-5


# ---- calibrate: reduces to a library softmax; group mean; temperature; ACCUM window -------------
@pytest.mark.parametrize("G,T", [(1, 1.0), (4, 1.0), (5, 0.5), (3, 2.5)])
def test_calibrate_is_mean_of_library_softmax(G, T):
    cfg, u, rng = _unit(G=G, d=64, n0=300, max_ctx=320, W=20, T=T)
    lo, hi = u.pool
    z = rng.standard_normal((G, hi - lo)) * 3
    _set_logits(u, z)
    u.calibrate()
    ref = scipy.special.softmax(u.logits[:, lo:hi].astype(np.float64) / T, axis=1).mean(0)
    np.testing.assert_allclose(u.probs[lo:hi], ref, rtol=2e-7, atol=0)
    assert abs(u.probs[lo:hi].astype(np.float64).sum() - 1) < 1e-5


def test_accum_is_sliding_window_sum():
    """ACCUM == 'accumulated attention over the last w steps' (BASELINE config 4, reading C4), renormalised."""
    w = 4
    rng = np.random.default_rng(3)
    cfg = OracleConfig(G=2, d=64, max_ctx=128, sink=2, recent=8, k_cap=128, cond_cap=4, accum_window=w)
    u = Unit(cfg, rng.standard_normal((60, 64)).astype(np.float32), rng.standard_normal((60, 64)).astype(np.float32),
             l_upper=55, score_mode=1)
    rows = []
    for t in range(11):
        u.append(rng.standard_normal(64).astype(np.float32), rng.standard_normal(64).astype(np.float32))
        u.retire()
        lo, hi = u.pool
        z = rng.standard_normal((2, hi - lo)) * 2
        _set_logits(u, z)
        u.calibrate()
        row = np.zeros(cfg.max_ctx)
        row[lo:hi] = scipy.special.softmax(u.logits[:, lo:hi].astype(np.float64), axis=1).mean(0)
        rows.append(row)
        ref = np.sum(rows[-w:], axis=0)[lo:hi]
        np.testing.assert_allclose(u.probs[lo:hi], ref / ref.sum(), rtol=5e-6, atol=1e-9)


# ---- P2: brute force minimality on tiny pools (L108) --------------------------------------------
@pytest.mark.parametrize("seed", range(12))
def test_p2_bruteforce_minimal_nucleus(seed):
    rng = np.random.default_rng(100 + seed)
    N = int(rng.integers(3, 13))
    W = 4
    cfg, u, _ = _unit(G=1, d=64, n0=4 + N + W, max_ctx=64, s=4, W=W, k_cap=64)
    P = rng.dirichlet(np.ones(N) * rng.choice([0.2, 1.0, 5.0])).astype(np.float32)
    if seed % 3 == 0:
        P[rng.integers(0, N, 3)] = P[0]      # force ties
    lo, hi = u.pool
    assert hi - lo == N
    u.probs[lo:hi] = P
    p = np.float32(rng.choice([0.5, 0.8, 0.9, 0.95]))
    u.topp_select(float(p), count_votes=False)
    w = _w(P)
    theta = max(1, math.ceil(float(np.float64(p) * np.float64(int(w.sum())))))
    sel = np.array(u.sel_idx[:u.sel_count]) - lo
    k = len(sel)
    assert int(w[sel].sum()) >= theta                                             # mass >= p
    for r in range(k):                                                            # no smaller subset reaches it
        for sub in itertools.combinations(range(N), r):
            assert int(w[list(sub)].sum()) < theta
    unsel = np.setdiff1d(np.arange(N), sel)
    if len(unsel):
        assert P[sel].min() >= P[unsel].max()                                     # a prefix of the sorted order
        ties = unsel[P[unsel] == P[sel].min()]
        sel_ties = sel[P[sel] == P[sel].min()]
        if len(ties):
            assert sel_ties.max() < ties.min()                                    # ties: position ascending
    assert int(w[sel].sum()) - int(w[sel].min()) < theta                          # dropping the last falls below
    assert list(sel) == sorted(sel)


# ---- P3 ties, P4 degenerate, P5 closed form -----------------------------------------------------
def test_p3_all_equal():
    cfg, u, _ = _unit(G=1, d=64, n0=4 + 1000 + 16, max_ctx=1024, W=16, k_cap=1024)
    _set_logits(u, np.zeros((1, 1000)))
    u.calibrate()
    u.topp_select(0.9)
    lo, _ = u.pool
    assert u.sel_count == 900 and list(u.sel_idx[:900]) == list(range(lo, lo + 900))
    assert (u.votes[lo:lo + 900] == 1).all() and u.votes.sum() == 900


def test_p4_one_dominant():
    cfg, u, rng = _unit(G=1, d=64, n0=4 + 500 + 16, max_ctx=528, W=16, k_cap=528)
    z = rng.standard_normal((1, 500)); z[0, 123] += 40
    _set_logits(u, z)
    u.calibrate(); u.topp_select(0.9)
    assert u.sel_count == 1 and u.sel_idx[0] == u.pool[0] + 123


@pytest.mark.parametrize("p,expect", [(0.9, 231), (0.95, 300)])
def test_p5_geometric_closed_form(p, expect):
    lam, N = 0.01, 2000
    r = math.exp(-lam)
    assert math.ceil(math.log(1 - p * (1 - r ** N)) / math.log(r)) == expect
    cfg, u, _ = _unit(G=1, d=64, n0=4 + N + 16, max_ctx=2048, W=16, k_cap=2048)
    _set_logits(u, -lam * np.arange(N)[None, :])
    u.calibrate(); u.topp_select(p)
    assert u.sel_count == expect and list(u.sel_idx[:expect]) == list(range(4, 4 + expect))


# ---- P6: order invariance under T > 0 (Constraint 1 L116, Thm D.3) and nesting in p -------------
def test_p6_temperature_and_p_nesting():
    rng = np.random.default_rng(6)
    N = 3000
    z = rng.standard_normal((1, N)) * 2
    sets, ks = [], []
    for T in (0.5, 1.0, 2.0, 4.0):
        cfg, u, _ = _unit(G=1, d=64, n0=4 + N + 16, max_ctx=3072, W=16, k_cap=3072, T=T)
        _set_logits(u, z)
        u.calibrate(); u.topp_select(0.9)
        sets.append(set(u.sel_idx[:u.sel_count])); ks.append(u.sel_count)
        order = np.argsort(-u.probs[4:4 + N], kind="stable")       # Top-k set == k largest raw logits
        assert sets[-1] == set(4 + np.argsort(-u.logits[0, 4:4 + N], kind="stable")[:ks[-1]]) == set(4 + order[:ks[-1]])
    assert all(a <= b + 1 for a, b in zip(ks, ks[1:])) and ks[0] < ks[-1]          # k(T) non-decreasing
    assert all(a <= b for a, b in zip(sets, sets[1:]))                             # nested prefixes of one order
    cfg, u, _ = _unit(G=4, d=64, n0=4 + N + 16, max_ctx=3072, W=16, k_cap=3072)
    _set_logits(u, rng.standard_normal((4, N)) * 2)
    u.calibrate()
    prev = set()
    for p in (0.5, 0.8, 0.9, 0.95, 0.99, 1.0):
        u.topp_select(p, count_votes=False)
        cur = set(u.sel_idx[:u.sel_count])
        assert prev <= cur
        prev = cur
    assert len(prev) == N


# ---- P7: per-head budgets follow the logit temperature (L72-74, L100) ---------------------------
@pytest.mark.parametrize("p,sigma", [(0.95, 1.0), (0.95, 2.0), (0.9, 0.5), (0.9, 1.5)])
def test_p7_gaussian_budget_law(p, sigma):
    """iid N(0,sigma^2) logits: k/N -> Phi(Phi^-1(p) - sigma) (lognormal weights, size-biased tail)."""
    N = 16384
    rng = np.random.default_rng(int(sigma * 10) + int(p * 100))
    cfg, u, _ = _unit(G=1, d=64, n0=4 + N + 16, max_ctx=16416, W=16, k_cap=16416)
    _set_logits(u, rng.standard_normal((1, N)) * sigma)
    u.calibrate(); u.topp_select(p)
    expect = scipy.stats.norm.cdf(scipy.stats.norm.ppf(p) - sigma)
    assert abs(u.sel_count / N - expect) < 0.03          # 3 % of N (heavy lognormal tail at sigma=2)


# ---- P8: merge operator algebra (Eq. 6) -----------------------------------------------------------
def test_p8_merge_algebra():
    rng = np.random.default_rng(8)
    d, n = 64, 90
    cfg = OracleConfig(G=1, d=d, max_ctx=128, sink=0, recent=0, k_cap=16, cond_cap=0)
    K = (rng.standard_normal((n, d)) * 2).astype(np.float32); V = rng.standard_normal((n, d)).astype(np.float32)
    q = rng.standard_normal(d).astype(np.float32)
    full = state_of_set(cfg, q, K, V, np.arange(n))
    ref = torch.nn.functional.scaled_dot_product_attention(
        torch.tensor(q, dtype=torch.float64)[None, None], torch.tensor(K, dtype=torch.float64)[None],
        torch.tensor(V, dtype=torch.float64)[None])[0, 0].numpy()
    np.testing.assert_allclose(full[0], ref, atol=1e-12)
    for trial in range(5):
        lab = rng.integers(0, 3, n)
        parts = [state_of_set(cfg, q, K, V, np.flatnonzero(lab == j)) for j in range(3)]
        for order in itertools.permutations(range(3)):                     # commutative + associative
            left = merge(merge(parts[order[0]], parts[order[1]]), parts[order[2]])
            right = merge(parts[order[0]], merge(parts[order[1]], parts[order[2]]))
            for st in (left, right):
                np.testing.assert_allclose(st[0], full[0], rtol=1e-9, atol=1e-12)
                assert abs(st[1] + math.log(st[2]) - (full[1] + math.log(full[2]))) < 1e-9
    empty = state_of_set(cfg, q, K, V, np.zeros(0, np.int32))
    assert empty[2] == 0.0
    for st in (merge(full, empty), merge(empty, full)):                    # identity
        np.testing.assert_array_equal(st[0], full[0]); assert st[1:] == full[1:]


# ---- P9: rewrite copies, pads and table (L172, reading C9) ---------------------------------------
def test_p9_rewrite_and_table():
    cfg, u, rng = _unit(G=2, d=64, n0=300, max_ctx=320, W=16, k_cap=128)
    u.score(rng.standard_normal((2, 64)).astype(np.float32) * 3); u.calibrate(); u.topp_select(0.7)
    u.sel_k[:] = 7.0; u.sel_v[:] = 7.0
    u.rewrite()
    k = u.sel_count
    assert 0 < k < 128 and k % 16 != 0
    idx = u.sel_idx[:k]
    assert (np.diff(idx) > 0).all() and (u.sel_idx[k:] == -1).all()
    assert u.sel_k[:k].tobytes() == u.K[idx].tobytes() and u.sel_v[:k].tobytes() == u.V[idx].tobytes()
    end = -(-k // 16) * 16
    assert (u.sel_k[k:end] == 0).all() and (u.sel_v[k:end] == 0).all() and (u.sel_k[end:] == 7.0).all()
    pages = np.arange(100, 108, dtype=np.int32)
    tab = u.sel_table(pages)
    assert list(tab[:end // 16]) == list(pages[:end // 16]) and (tab[end // 16:] == -1).all()
    mask = u.sel_mask()
    bits = np.unpackbits(mask, bitorder="little")
    assert set(np.flatnonzero(bits)) == set(idx)


# ---- P10 / P11: condensed tier == top-C_cap of the retirement log; bookkeeping invariants ---------
def test_p10_p11_condensed_and_bookkeeping():
    C = 6
    cfg, u, rng = _unit(G=2, d=64, n0=150, max_ctx=256, s=4, W=12, k_cap=48, C=C, l_upper=100)
    log = []                                     # (votes at retirement, pos)
    total_sel = 0
    for t in range(70):
        q = rng.standard_normal((2, 64)).astype(np.float32) * 4
        c_before, votes_before = u.c_lo, u.votes.copy()
        u.decode_step(q, rng.standard_normal(64).astype(np.float32), rng.standard_normal(64).astype(np.float32), p=0.6)
        for pos in range(c_before, u.c_lo):
            log.append((int(votes_before[pos]), pos))
        total_sel += u.sel_count
        lo, hi = u.pool
        # P11
        assert hi - lo <= 100 and u.sel_count <= cfg.k_cap and u.cond_count <= C
        sel = u.sel_idx[:u.sel_count]
        assert ((sel >= lo) & (sel < hi)).all() and u.votes.sum() == total_sel
        dense = set(range(cfg.sink)) | set(range(hi, u.n))
        assert dense | set(range(lo, hi)) | {p for _, p in log} == set(range(u.n))
        assert len(dense) + (hi - lo) + len(log) == u.n
        # P10
        want = sorted(log, reverse=True)[:C]
        have = sorted(zip(u.cond_votes[:u.cond_count].tolist(), u.cond_pos[:u.cond_count].tolist()), reverse=True)
        assert have == want
        for j in range(u.cond_count):
            assert u.cond_k[j].tobytes() == u.K[u.cond_pos[j]].tobytes()
            assert u.cond_v[j].tobytes() == u.V[u.cond_pos[j]].tobytes()
    assert len(log) > 3 * C and u.sel_count == cfg.k_cap or u.k_topp <= cfg.k_cap


def test_k_cap_clamp_keeps_best_of_same_order():
    cfg, u, rng = _unit(G=1, d=64, n0=4 + 400 + 16, max_ctx=432, W=16, k_cap=32)
    _set_logits(u, rng.standard_normal((1, 400)) * 0.3)
    u.calibrate(); u.topp_select(0.95)
    assert u.k_topp > 32 and u.sel_count == 32
    best = 4 + np.argsort(-u.probs[4:404], kind="stable")[:32]
    assert set(u.sel_idx[:32]) == set(best)


def test_l_lower_selects_everything():
    cfg, u, rng = _unit(G=1, d=64, n0=4 + 100 + 16, max_ctx=128, W=16, k_cap=128, l_lower=100)
    _set_logits(u, rng.standard_normal((1, 100)) * 3)
    u.calibrate(); u.topp_select(0.5)
    assert u.sel_count == 100


# ---- P12: integer mass vs fp64 sorted cumsum ----------------------------------------------------
@pytest.mark.parametrize("seed", range(4))
def test_p12_integer_mass_vs_real(seed):
    rng = np.random.default_rng(1200 + seed)
    N = 5000
    cfg, u, _ = _unit(G=2, d=64, n0=4 + N + 16, max_ctx=5024, W=16, k_cap=5024)
    _set_logits(u, rng.standard_normal((2, N)) * rng.choice([0.5, 1.5, 3.0]))
    u.calibrate(); u.topp_select(0.9, count_votes=False)
    P = np.sort(u.probs[4:4 + N].astype(np.float64))[::-1]
    cum = np.cumsum(P) / P.sum()
    k_real = int(np.searchsorted(cum, 0.9) + 1)
    k_int = u.sel_count
    a, b = sorted((k_real, k_int))
    assert all(abs(cum[j - 1] - 0.9) <= N * 2.0 ** -33 + 1e-7 for j in range(a, b + 1)) or a == b


def test_empty_pool_and_short_context():
    cfg = OracleConfig(G=2, d=64, max_ctx=64, sink=4, recent=16, k_cap=32, cond_cap=4)
    rng = np.random.default_rng(0)
    u = Unit(cfg, rng.standard_normal((3, 64)).astype(np.float32), rng.standard_normal((3, 64)).astype(np.float32), l_upper=8)
    for t in range(30):
        q = rng.standard_normal((2, 64)).astype(np.float32)
        u.decode_step(q, rng.standard_normal(64).astype(np.float32), rng.standard_normal(64).astype(np.float32), p=0.9)
        lo, hi = u.pool
        assert hi - lo == max(0, min(u.n - 16 - 4, 8))
        if u.n <= 20:
            assert u.sel_count == 0
            n = u.n
            Kt = torch.tensor(u.K[:n], dtype=torch.float64)[None].expand(2, -1, -1)
            Vt = torch.tensor(u.V[:n], dtype=torch.float64)[None].expand(2, -1, -1)
            ref = torch.nn.functional.scaled_dot_product_attention(torch.tensor(q, dtype=torch.float64)[:, None], Kt, Vt)
            np.testing.assert_allclose(u.out, ref[:, 0].numpy(), atol=1e-5, rtol=0)


# ---- golden fixtures: closed-form nucleus sizes (tests/golden/closed_forms.txt, with derivations) ----
def _golden_rows():
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "closed_forms.txt")
    rows = []
    for line in open(path):
        line = line.strip()
        if line and not line.startswith("#"):
            case, N, p, param, k = line.split()
            rows.append((case, int(N), float(p), float(param), int(k)))
    return rows


@pytest.mark.parametrize("case,N,p,param,expect", _golden_rows())
def test_golden_closed_forms(case, N, p, param, expect):
    mc = (4 + N + 16 + 15) // 16 * 16
    cfg, u, rng = _unit(G=1, d=64, n0=4 + N + 16, max_ctx=mc, W=16, k_cap=mc)
    if case == "equal":
        z = np.zeros((1, N))
    elif case == "geometric":
        z = -param * np.arange(N)[None, :]
    else:
        z = rng.standard_normal((1, N)); z[0, N // 2] += param
    _set_logits(u, z)
    u.calibrate(); u.topp_select(p)
    assert u.sel_count == expect
    if case != "dominant":
        assert list(u.sel_idx[:expect]) == list(range(4, 4 + expect))


# ---- P14: SNAPKV metric = max-pool of the raw logits along the sequence (L150, L278) ------------
@pytest.mark.parametrize("G,kernel,T", [(1, 7, 1.0), (4, 5, 0.7), (3, 1, 2.0)])
def test_p14_snapkv_maxpool_is_library_maxpool(G, kernel, T):
    """calibrate() of a SNAPKV head == mean_g softmax(max_pool1d(z_g) / T), the pooling done by
    torch.nn.functional.max_pool1d (stride 1, -inf padding = window clipped to the pool)."""
    rng = np.random.default_rng(14)
    cfg = OracleConfig(G=G, d=64, max_ctx=256, sink=4, recent=16, k_cap=256, cond_cap=8, pool_kernel=kernel)
    K0 = rng.standard_normal((200, 64)).astype(np.float32)
    u = Unit(cfg, K0, K0.copy(), l_upper=10**6, T=T, score_mode=2)
    lo, hi = u.pool
    z = (rng.standard_normal((G, hi - lo)) * 3).astype(np.float32)
    _set_logits(u, z)
    u.calibrate()
    zt = torch.tensor(z, dtype=torch.float64)[None]
    pooled = torch.nn.functional.max_pool1d(zt, kernel, stride=1, padding=kernel // 2)[0]
    ref = torch.softmax(pooled / T, -1).mean(0).numpy()
    np.testing.assert_allclose(u.probs[lo:hi], ref, rtol=1e-6, atol=1e-12)
    if kernel == 1:   # identity window: the SNAPKV head is a RAW head
        cfg0, u0, _ = _unit(G=G, T=T)
        _set_logits(u0, z); u0.calibrate()
        np.testing.assert_array_equal(u0.probs[lo:hi], u.probs[lo:hi])


# ---- P13: temperature solve, Algorithm 2 (L625-648) for Problem 1 (L108-110) --------------------
def _topk_mass_np(P, k):
    w = _w(np.asarray(P, np.float32))
    return float(np.sort(w)[::-1][:k].sum() / w.sum())


@pytest.mark.parametrize("G,sigma", [(1, 1.0), (4, 2.5)])
def test_p13_identity_metric_solves_to_one(G, sigma):
    """g = id: S_hat(T = 1) == S, so Problem 1's minimiser is T* = 1 (mass error 0 there)."""
    cfg, u, rng = _unit(G=G, n0=1200, max_ctx=1280, W=16, k_cap=1280, seed=13)
    lo, hi = u.pool
    _set_logits(u, rng.standard_normal((G, hi - lo)) * sigma)
    it, resid = u.solve_temperature(0.9, t_min=0.25, t_max=3.0, eps=1e-7, max_iter=60)
    assert abs(u.T - 1.0) < 2e-3 and resid < 1e-4 and 1 <= it <= 60


def test_p13_snapkv_geometric_closed_form():
    """z_i = -lam * i with a max-pool of radius r: g(z) has r + 1 copies of the top logit, then the
    same geometric tail, so M_k(S) and M_k(S_hat(T)) are geometric sums and T* is the root of a
    scalar equation, solved here by scipy.optimize.brentq (independent of the oracle)."""
    import scipy.optimize
    lam, N, r, p = 0.1, 400, 5, 0.9
    cfg = OracleConfig(G=1, d=64, max_ctx=N + 32, sink=4, recent=16, k_cap=N + 32, cond_cap=8, pool_kernel=2 * r + 1)
    K0 = np.zeros((N + 20, 64), np.float32)
    u = Unit(cfg, K0, K0.copy(), l_upper=10**6, score_mode=2)
    _set_logits(u, -lam * np.arange(N)[None, :])
    rho = math.exp(-lam)
    k = math.ceil(math.log(1 - p * (1 - rho ** N)) / math.log(rho))          # pin P5's closed form
    MkS = (1 - rho ** k) / (1 - rho ** N)

    def f(T):
        q = math.exp(-lam / T)
        geo = lambda m: (1 - q ** m) / (1 - q)       # 1 + q + ... + q^(m-1)
        return MkS - (r + geo(k - r)) / (r + geo(N - r))

    Tstar = scipy.optimize.brentq(f, 0.25, 4.0, xtol=1e-10)
    it, resid = u.solve_temperature(p, t_min=0.25, t_max=4.0, eps=1e-7, max_iter=60)
    assert u.k_topp == k
    assert abs(u.T - Tstar) < 2e-3 * Tstar, (u.T, Tstar)
    assert abs(Tstar - 1.0) > 0.03          # the case is not the trivial T* = 1


@pytest.mark.parametrize("mode,kernel", [(0, 0), (2, 7)])
def test_p13_root_bracket_and_monotonicity(mode, kernel):
    """Independent numpy evaluation at the returned T: the mass error is within eps, M_k(S_hat(T)) decreases in T
    (why bisection applies, L599 'sharpened for lower T and flattened for higher T') and the root is bracketed."""
    rng = np.random.default_rng(131)
    G, p, eps = 4, 0.9, 1e-5
    cfg = OracleConfig(G=G, d=64, max_ctx=2048, sink=4, recent=32, k_cap=2048, cond_cap=8, pool_kernel=kernel)
    K0 = np.zeros((2000, 64), np.float32)
    u = Unit(cfg, K0, K0.copy(), l_upper=10**6, score_mode=mode, T=5.0)
    lo, hi = u.pool
    z = (rng.standard_normal((G, hi - lo)) * 2.0).astype(np.float32)
    _set_logits(u, z)
    zt = torch.tensor(z, dtype=torch.float64)
    gz = torch.nn.functional.max_pool1d(zt[None], kernel, stride=1, padding=kernel // 2)[0] if mode == 2 else zt
    S = torch.softmax(zt, -1).mean(0).numpy().astype(np.float32)
    w = _w(S); order = np.argsort(-S, kind="stable")
    k = int(np.searchsorted(np.cumsum(w[order]), math.ceil(p * float(w.sum()))) + 1)
    MkS = _topk_mass_np(S, k)
    Mk = lambda T: _topk_mass_np(torch.softmax(gz / T, -1).mean(0).numpy().astype(np.float32), k)
    it, resid = u.solve_temperature(p, t_min=0.125, t_max=8.0, eps=eps, max_iter=50)
    assert u.k_topp == k
    assert abs(Mk(u.T) - MkS) <= eps + 1e-6 and resid <= eps
    grid = [0.125, 0.25, 0.5, 1.0, 2.0, 4.0, 8.0]
    vals = [Mk(T) for T in grid]
    assert all(a > b for a, b in zip(vals, vals[1:]))
    assert vals[0] > MkS > vals[-1]
    if mode == 0:
        assert abs(u.T - 1.0) < 1e-2
    else:
        assert u.T < 1.0    # maxima of 7 iid logits spread less (std ~0.6 sigma): flatter at T = 1, so T* < 1


def test_p13_accum_heads_are_left_alone():
    cfg, u, rng = _unit(G=2, mode=1, T=1.5)
    lo, hi = u.pool
    _set_logits(u, rng.standard_normal((2, hi - lo)))
    assert u.solve_temperature(0.9) == (0, 0.0) and u.T == 1.5


# ---- P15: LSE-preserving weighted merging of the condensed tier (Appendix G, Eq. 9, Thm G.1) -----
def _merge_case(gap, G=1, seed=15, bf16=0):
    """A full 4-slot tier, l_upper tiny so the next step retires one token that loses on votes (votes 0 < residents' 5):
    the newcomer is the evictee and must be folded into the best-scoring resident."""
    rng = np.random.default_rng(seed)
    d = 64
    cfg = OracleConfig(G=G, d=d, max_ctx=128, sink=4, recent=8, k_cap=128, cond_cap=4, cond_merge=1, kv_bf16=bf16,
                       sm_scale=1.0)
    K0 = rng.standard_normal((60, d)).astype(np.float32) * 0.3
    V0 = rng.standard_normal((60, d)).astype(np.float32)
    u = Unit(cfg, K0, V0, l_upper=60 - 8 - 4 - 1)       # pool 48 > 47: exactly one retirement
    q = rng.standard_normal((G, d)).astype(np.float32) * 0.3
    qbar = q.mean(0)
    # residents: slot 2 is aligned with the queries (the anchor), the others are weak
    u.u.cond_count = 4
    for j in range(4):
        u.cond_k[j] = rng.standard_normal(d).astype(np.float32) * 0.05
        u.cond_v[j] = rng.standard_normal(d).astype(np.float32)
        u.cond_pos[j] = 100 + j; u.cond_votes[j] = 5
    u.cond_k[2] = (qbar / np.dot(qbar, qbar) * 2.0).astype(np.float32)            # x_anchor = 2
    u.K[4] = (qbar / np.dot(qbar, qbar) * (2.0 - gap)).astype(np.float32)         # evictee t = c_lo = 4: x_e = 2 - gap
    return cfg, u, q


@pytest.mark.parametrize("G,gap", [(1, 0.5), (4, 1.5), (1, 0.0)])
def test_p15_merge_weights_are_the_pair_softmax(G, gap):
    cfg, u, q = _merge_case(gap, G=G)
    Ka, Va, Ke, Ve = u.cond_k[2].copy(), u.cond_v[2].copy(), u.K[4].copy(), u.V[4].copy()
    others = (u.cond_k[[0, 1, 3]].copy(), u.cond_v[[0, 1, 3]].copy(), u.cond_pos.copy(), u.cond_votes.copy())
    assert u.retire_q(q) == 1 and u.c_lo == 5 and u.cond_count == 4
    xa = float(np.mean(q.astype(np.float64) @ Ka.astype(np.float64)))
    xe = float(np.mean(q.astype(np.float64) @ Ke.astype(np.float64)))
    w = torch.softmax(torch.tensor([xa, xe], dtype=torch.float64), 0).numpy()       # Eq. 9's weights, library softmax
    np.testing.assert_allclose(u.cond_k[2], w[0] * Ka + w[1] * Ke, rtol=0, atol=1e-6)
    np.testing.assert_allclose(u.cond_v[2], w[0] * Va + w[1] * Ve, rtol=0, atol=1e-6)
    np.testing.assert_array_equal(u.cond_k[[0, 1, 3]], others[0])                     # only the anchor changes
    np.testing.assert_array_equal(u.cond_v[[0, 1, 3]], others[1])
    np.testing.assert_array_equal(u.cond_pos, others[2]); np.testing.assert_array_equal(u.cond_votes, others[3])
    if gap == 0.0:
        assert abs(w[0] - 0.5) < 1e-6                                                  # equal scores: the midpoint


def test_p15_se_between_eviction_and_keeping_and_theorem_g1_limit():
    """G = 1: the merged key scores the weighted mean of the pair's scores (Eq. 9.a is linear in K), so its
    exponential lies between the pair's and below keeping both (h(t) > 0, Eq. 13-14), and the SE error of Eq. 10
    relative to keeping both vanishes as x_a - x_e grows (Thm G.1, Eq. 11 / 15)."""
    errs = []
    for gap in (0.5, 2.0, 6.0, 12.0):
        cfg, u, q = _merge_case(gap, G=1)
        Ka, Ke = u.cond_k[2].astype(np.float64), u.K[4].astype(np.float64)
        u.retire_q(q)
        x = lambda K: float(q[0].astype(np.float64) @ K)
        se_merge, se_keep, se_evict = math.exp(x(u.cond_k[2].astype(np.float64))), math.exp(x(Ka)) + math.exp(x(Ke)), math.exp(x(Ka))
        w = torch.softmax(torch.tensor([x(Ka), x(Ke)], dtype=torch.float64), 0).numpy()
        assert abs(math.log(se_merge) - (w[0] * x(Ka) + w[1] * x(Ke))) < 1e-5           # Eq. 9.a
        assert math.exp(x(Ke)) * (1 - 1e-6) <= se_merge <= se_evict * (1 + 1e-6) <= se_keep
        errs.append((se_keep - se_merge) / se_keep)
    assert all(a > b for a, b in zip(errs, errs[1:])) and errs[-1] < 1e-4


def test_p15_displaced_resident_is_merged_and_bf16_store():
    """The newcomer wins on votes: it takes the weakest slot and the displaced resident is the evictee; the merged
    anchor row of a bf16 tier is bf16-representable and within half an ulp (at most 2^-8 relative) of the exact combination."""
    cfg, u, q = _merge_case(1.0, G=2, bf16=1)
    u.votes[4] = 9                                       # newcomer outranks every resident (votes 5)
    u.cond_votes[1] = 3                                  # slot 1 is the weakest: displaced
    Ka, Ke = u.cond_k[2].copy(), u.cond_k[1].copy()
    Kt = u.K[4].copy()
    u.retire_q(q)
    assert u.cond_pos[1] == 4 and u.cond_votes[1] == 9
    np.testing.assert_array_equal(u.cond_k[1], Kt)
    xs = [float(np.mean(q.astype(np.float64) @ u.cond_k[j].astype(np.float64))) for j in range(4)]
    # the anchor is the best-scoring resident after the replacement (the aligned newcomer, slot 1, or slot 2)
    a = 1 if float(np.mean(q.astype(np.float64) @ Kt.astype(np.float64))) > 2.0 else 2
    base = Kt if a == 1 else Ka
    xa = float(np.mean(q.astype(np.float64) @ base.astype(np.float64)))
    xe = float(np.mean(q.astype(np.float64) @ Ke.astype(np.float64)))
    wa = 1.0 / (1.0 + math.exp(xe - xa))
    exact = wa * base.astype(np.float64) + (1 - wa) * Ke.astype(np.float64)
    got = u.cond_k[a]
    assert np.all((got.view(np.uint32) & 0xffff) == 0)                                # bf16-representable
    np.testing.assert_allclose(got, exact, rtol=2.0 ** -8, atol=1e-30)


# ---- golden fixtures: closed-form roots T* of Problem 1 (tests/golden/temperature_roots.txt; written by
#      tests/golden/make_temperature_roots.py from the geometric sums, scipy only) -------------------------------
def _root_rows():
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "temperature_roots.txt")
    rows = []
    for line in open(path):
        line = line.strip()
        if line and not line.startswith("#"):
            lam, N, r, p, k, T = line.split()
            rows.append((float(lam), int(N), int(r), float(p), int(k), float(T)))
    return rows


@pytest.mark.parametrize("lam,N,r,p,k,Tstar", _root_rows())
def test_golden_temperature_roots(lam, N, r, p, k, Tstar):
    cfg = OracleConfig(G=1, d=64, max_ctx=(N + 20 + 15) // 16 * 16, sink=4, recent=16, k_cap=(N + 20 + 15) // 16 * 16,
                       cond_cap=8, pool_kernel=2 * r + 1)
    K0 = np.zeros((N + 20, 64), np.float32)
    u = Unit(cfg, K0, K0.copy(), l_upper=10**6, score_mode=2)
    _set_logits(u, -lam * np.arange(N)[None, :])
    it, resid = u.solve_temperature(p, t_min=0.25, t_max=4.0, eps=1e-7, max_iter=60)
    assert u.k_topp == k
    assert abs(u.T - Tstar) < 2e-3 * Tstar, (u.T, Tstar)


# ---- P16: the steps between two compressions (do_select = 0, L274) attend every live token exactly once ----------
@pytest.mark.parametrize("interval,p", [(4, 1.0), (5, 0.9), (3, 0.6)])
def test_p16_reuse_steps_partition_the_live_tokens(interval, p):
    """Between compressions only Step 1 of L78 runs: the new token joins the dense tier, which grows from the anchor
    of the last compression; nothing retires.  So the attended positions are sinks + [dense_lo, n) + the selection of
    the last compression + the condensed residents: no position twice, none of them dropped.  Checked against a
    library log-sum-exp / SDPA over that explicit position list (a duplicate or a dropped token changes both), and at
    p = 1 with large caps against dense attention over all n tokens."""
    G, d = 3, 64
    cfg, u, rng = _unit(G=G, d=d, n0=150, max_ctx=256, s=4, W=12, k_cap=256, C=6,
                        l_upper=10**6 if p == 1.0 else 110)
    sel_at = None
    for t in range(22):
        q = (rng.standard_normal((G, d)) * 1.5).astype(np.float32)
        kn, vn = rng.standard_normal(d).astype(np.float32), rng.standard_normal(d).astype(np.float32)
        do_sel = t % interval == 0
        n_before, clo_before, cc_before = u.n, u.c_lo, u.cond_count
        u.decode_step(q, kn, vn, p=p, do_select=do_sel)
        assert u.n == n_before + 1
        if do_sel:
            sel_at = u.n
            assert u.dense_lo == max(cfg.sink, u.n - cfg.recent)
        else:   # no retirement, no re-anchoring between compressions
            assert (u.c_lo, u.cond_count) == (clo_before, cc_before) and u.dense_lo == max(cfg.sink, sel_at - cfg.recent)
        pos = list(range(min(cfg.sink, u.n))) + list(range(u.dense_lo, u.n)) + list(u.sel_idx[:u.sel_count]) + \
            list(u.cond_pos[:u.cond_count])
        assert len(set(pos)) == len(pos), "a position is attended twice"
        if p == 1.0:
            assert sorted(pos) == list(range(u.n)), "a live token is dropped"
        Kt = torch.tensor(u.K[pos], dtype=torch.float64)[None].expand(G, -1, -1)
        Vt = torch.tensor(u.V[pos], dtype=torch.float64)[None].expand(G, -1, -1)
        qt = torch.tensor(q, dtype=torch.float64)
        ref = torch.nn.functional.scaled_dot_product_attention(qt[:, None], Kt, Vt)
        np.testing.assert_allclose(u.out, ref[:, 0].numpy(), atol=1e-5, rtol=0)
        x = (qt @ Kt[0].T) / math.sqrt(d)
        np.testing.assert_allclose(u.lse, torch.logsumexp(x, -1).numpy(), atol=1e-5, rtol=0)
    assert p == 1.0 or u.cond_count > 0     # the deferred retirements did happen at the compression steps


# ---- P17: accumulated attention recomputed from the query cache (L448, L122-124; reading C18) ---------------------
def test_p17_qcache_accum_equals_ring_sum_on_a_static_pool_and_library_softmax():
    """score_mode 3 scores the CURRENT pool with every query of the sliding window.  (a) While the pool does not change,
    that is the sum of the window's per-step rows -- the ring-sum ACCUM form already pinned by
    test_accum_is_sliding_window_sum -- so both modes must give the same normalised row, before and after the window
    wraps.  (b) Independently: the row equals the mean over (cached step, head) of scipy softmax rows of numpy logits.
    (c) When the pool does change the two forms differ (old rows were normalised over old pools): the recomputed one is
    still the library softmax mean over the NEW pool."""
    w, G, d = 4, 3, 64
    rng = np.random.default_rng(11)
    cfg = OracleConfig(G=G, d=d, max_ctx=160, sink=2, recent=8, k_cap=160, cond_cap=4, accum_window=w)
    K0, V0 = rng.standard_normal((90, d)).astype(np.float32), rng.standard_normal((90, d)).astype(np.float32)
    ring, qc = Unit(cfg, K0, V0, l_upper=10**6, T=0.7, score_mode=1), Unit(cfg, K0, V0, l_upper=10**6, T=0.7, score_mode=3)
    lo, hi = qc.pool
    qs = []
    for t in range(7):                                    # static pool: no append; the window wraps at t = 4
        q = (rng.standard_normal((G, d)) * 1.3).astype(np.float32)
        qs.append(q)
        ring.score(q); ring.calibrate()
        qc.qcache_push(q); qc.calibrate()
        np.testing.assert_allclose(qc.probs[lo:hi], ring.probs[lo:hi], rtol=3e-6, atol=1e-12)
        win = qs[-w:]
        z = np.stack([(np.float64(cfg.c().sm_scale) * (qq.astype(np.float64) @ K0[lo:hi].astype(np.float64).T)) / np.float64(np.float32(0.7))
                      for qq in win])                     # [steps][G][N]
        ref = scipy.special.softmax(z, axis=2).mean(axis=(0, 1))
        np.testing.assert_allclose(qc.probs[lo:hi], ref / ref.sum(), rtol=2e-7, atol=0)
        assert abs(qc.probs[lo:hi].astype(np.float64).sum() - 1) < 1e-5
    # (c) the pool moves: decode steps append tokens; the recomputed metric follows the library form on the new pool
    for t in range(3):
        q = (rng.standard_normal((G, d)) * 1.3).astype(np.float32)
        qs.append(q)
        kn, vn = rng.standard_normal(d).astype(np.float32), rng.standard_normal(d).astype(np.float32)
        qc.decode_step(q, kn, vn, p=0.9)
        ring.decode_step(q, kn, vn, p=0.9)
        lo, hi = qc.pool
        z = np.stack([(np.float64(cfg.c().sm_scale) * (qq.astype(np.float64) @ qc.K[lo:hi].astype(np.float64).T)) / np.float64(np.float32(0.7))
                      for qq in qs[-w:]])
        ref = scipy.special.softmax(z, axis=2).mean(axis=(0, 1))
        np.testing.assert_allclose(qc.probs[lo:hi], ref / ref.sum(), rtol=2e-7, atol=0)
    assert not np.allclose(qc.probs[lo:hi], ring.probs[lo:hi], rtol=1e-4)
    assert qc.u.qc_count == w and qc.u.qc_slot == (7 + 3) % w
