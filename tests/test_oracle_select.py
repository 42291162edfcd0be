"""Pins for oracle O3-O10 (Eq.1-5, A.2-A.9, Eq.15) -- brute force, invariants, hand-worked."""
import math
import os

import numpy as np
import pytest

import oracle
from paper_2607_07724_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden", "margin_examples.txt")


def _f(x):
    return synth.bf16_to_f32(x).astype(np.float64)


def _brute_tile_scores(inp, meta, policy):
    """numpy restatement of Eq.1/Eq.2 + Eq.3 with an independent formula for Quest
    (max(q a, q b) = q+ a + q- b for a >= b)."""
    cfg = inp.cfg
    H, N, d, Bn, G = cfg.n_q_heads, cfg.seqlen, cfg.head_dim, cfg.block, cfg.group
    T = N // Bn
    Q = _f(inp.Q).reshape(H, T, Bn, d)
    kmean, kmin, kmax = meta
    out = np.full((T, H, T), -np.inf)
    for h in range(H):
        g = h // G
        if policy in ("topk", "router"):
            s = np.einsum("trc,bc->trb", Q[h], kmean[g].astype(np.float64))
            s = s.astype(np.float32) * np.float32(1.0 / math.sqrt(d))
        else:
            qp, qn = np.maximum(Q[h], 0), np.minimum(Q[h], 0)
            s = np.einsum("trc,bc->trb", qp, _f(kmax[g])) + np.einsum("trc,bc->trb", qn, _f(kmin[g]))
            s = s.astype(np.float32)
        ts = s.max(axis=1).astype(np.float64)          # [T, T(b)]
        ts[np.triu_indices(T, 1)] = -np.inf            # causal: b <= t only
        out[:, h, :] = ts
    return out


@pytest.mark.parametrize("policy", ["topk", "quest"])
def test_tile_scores_brute_force(c1_inputs, c1_meta, policy):
    cfg = c1_inputs.cfg
    r = oracle.select(c1_inputs.Q, c1_meta, cfg.block, policy, cfg.k_budget, 0.25, want_scores=True)
    want = _brute_tile_scores(c1_inputs, c1_meta, policy)
    got = r["tile_score"].astype(np.float64)
    vis = np.isfinite(want)
    assert np.array_equal(np.isfinite(got), vis)
    # same value up to the summation order of the double accumulation (1 fp32 ulp)
    assert np.allclose(got[vis], want[vis], rtol=2.5e-7, atol=1e-7)


@pytest.mark.parametrize("policy", ["topk", "router", "quest", "router_quest"])
def test_selection_vs_stable_sort(c1_inputs, c1_meta, policy):
    """O5-O7, O10 against numpy lexsort on the oracle's own tile scores."""
    cfg = c1_inputs.cfg
    k, NB = cfg.k_budget, cfg.n_blocks
    r = oracle.select(c1_inputs.Q, c1_meta, cfg.block, policy, k, 0.25, want_scores=True)
    W = r["W"]
    assert W == (2 * k if "router" in policy else k)
    T, H = NB, cfg.n_q_heads
    for t in range(T):
        for h in range(H):
            ts = r["tile_score"][t, h, : t + 1]
            free = np.arange(1, t)
            order = free[np.lexsort((free, -ts[1:t].astype(np.float64)))] if t > 1 else free
            full = [0] + ([t] if t > 0 else []) + list(order)
            cnt = min(2 * k if r["trigger"][t] else k, t + 1, W)
            assert r["kv_count"][h, t] == cnt
            row = r["kv_idx"][h, t]
            assert list(row[:cnt]) == full[:cnt]
            assert np.all(row[cnt:] == NB)
            # sigma (Eq.4 with reading G1/G5)
            f = 1 if t == 0 else 2
            if t + 1 <= k:
                want = 1.0
            else:
                u = ts[order]
                num = np.float32(u[k - 1 - f]) - np.float32(u[k - f])
                den = np.float32(u[0]) - np.float32(u[k - f])
                want = 0.0 if den == 0 else float(np.float32(num) / np.float32(den))
            assert r["sigma"][h, t] == np.float32(want)
    assert np.all((r["sigma"] >= 0) & (r["sigma"] <= 1))          # L21, L102


def _parse_gold():
    sel, routes = [], []
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        p = [x.strip() for x in line.split("|")]
        if p[1] == "route":
            routes.append((p[0], np.array(p[2].split(), np.float32), float(p[3]), float(p[4]),
                           [int(x) for x in p[5].split()]))
        else:
            sel.append(dict(name=p[0], t=int(p[1]), nb=int(p[2]), k=int(p[3]),
                            ts=np.array(p[4].split(), np.float32), sigma=float(p[5]),
                            row0=[int(x) for x in p[6].split()], cnt0=int(p[7]),
                            row1=[int(x) for x in p[8].split()], cnt1=int(p[9])))
    return sel, routes


def test_hand_worked_margin_examples():
    sel, routes = _parse_gold()
    assert len(sel) == 6 and len(routes) == 1
    for e in sel:
        sig, idx_sorted, _ = oracle.select_from_scores(e["ts"], e["t"], e["nb"], e["k"])
        assert abs(sig - e["sigma"]) < 1e-6, e["name"]
        for trig, row, cnt in ((0, e["row0"], e["cnt0"]), (1, e["row1"], e["cnt1"])):
            # orc_fill (Eq.14) takes the tile index from the position: put the example at tile t of a
            # (t+1)-tile sequence and assert on what fill() itself returns for that tile
            t, nb, k = e["t"], e["nb"], e["k"]
            idx_all = np.full((t + 1, 1, 2 * k), nb, np.int32)
            idx_all[t, 0] = idx_sorted
            trigger = np.zeros(t + 1, np.uint8)
            trigger[t] = trig
            kv_idx, kv_count = oracle.fill(idx_all, trigger, nb, k, 2 * k)
            assert int(kv_count[0, t]) == cnt, e["name"]
            assert kv_idx[0, t].tolist() == row, e["name"]
            # non-router width W = k: the untriggered prefix, same count rule
            if not trig:
                kv_k, cnt_k = oracle.fill(idx_all, trigger, nb, k, k)
                assert int(cnt_k[0, t]) == cnt and kv_k[0, t].tolist() == row[:k], e["name"]
    for name, sb, q, tau, tiles in routes:
        sigma = np.repeat(sb[:, None], 3, axis=1)           # 3 identical heads -> mean = sb
        sbar, got_tau, trig = oracle.route(sigma, "router", q)
        assert np.allclose(sbar, sb, atol=1e-7)
        assert abs(got_tau - tau) < 1e-7
        assert list(np.nonzero(trig)[0]) == tiles


def test_sigma_affine_invariance():
    """sigma(a*s + c) == sigma(s) exactly for power-of-two a and representable c (Eq.4 is a ratio
    of differences)."""
    rng = np.random.default_rng(0)
    for _ in range(50):
        t = int(rng.integers(8, 40))
        ts = (rng.integers(-2**10, 2**10, t + 1) / 64.0).astype(np.float32)
        s0, i0, _ = oracle.select_from_scores(ts, t, 64, 5)
        s1, i1, _ = oracle.select_from_scores(ts * np.float32(4.0) + np.float32(3.0), t, 64, 5)
        assert s0 == s1 and np.array_equal(i0, i1)
        assert 0.0 <= s0 <= 1.0


def test_forced_first_and_duplicate_block_ties():
    """Duplicated K blocks give exactly tied scores -> lower block index first (G6)."""
    cfg = synth.CONFIGS["C1"].scaled(1024)
    inp = synth.make_inputs(cfg)
    K = inp.K.copy()
    for b in (3, 5, 9):                       # copies of block 2
        K[:, b * 64:(b + 1) * 64] = K[:, 2 * 64:3 * 64]
    meta = oracle.pool(K, 64)
    for policy in ("topk", "quest"):
        r = oracle.select(inp.Q, meta, 64, policy, 6, 0.0, want_scores=True)
        for t in range(12, 16):
            for h in range(cfg.n_q_heads):
                row = list(r["kv_idx"][h, t][: r["kv_count"][h, t]])
                assert row[0] == 0 and row[1] == t
                ts = r["tile_score"][t, h]
                assert ts[2] == ts[3] == ts[5] == ts[9]
                pos = [row.index(b) for b in (2, 3, 5, 9) if b in row]
                assert pos == sorted(pos)
                present = [b in row for b in (2, 3, 5, 9)]
                assert present == sorted(present, reverse=True)   # never keep 5 without 3, etc.


def test_quest_upper_bound(c1_inputs, c1_meta):
    """Quest score upper-bounds every token-level q.k in its block (L54, L82)."""
    cfg = c1_inputs.cfg
    Q, K = _f(c1_inputs.Q), _f(c1_inputs.K)
    _, kmin, kmax = c1_meta
    rng = np.random.default_rng(1)
    for _ in range(200):
        h = int(rng.integers(cfg.n_q_heads)); g = h // cfg.group
        i = int(rng.integers(cfg.seqlen)); b = int(rng.integers(cfg.n_blocks))
        q = Q[h, i]
        s = np.maximum(q * _f(kmax[g, b]), q * _f(kmin[g, b])).sum()
        tok = K[g, b * 64:(b + 1) * 64] @ q
        assert s >= tok.max() - 1e-9
    # and the oracle's tile score inherits it: ts_quest[t,h,b] >= max_{r,j} q_r.k_j
    r = oracle.select(c1_inputs.Q, c1_meta, 64, "quest", 4, 0.0, want_scores=True)
    for (t, h, b) in [(5, 0, 2), (31, 3, 17), (10, 2, 10)]:
        g = h // cfg.group
        tok = (Q[h, t * 64:(t + 1) * 64] @ K[g, b * 64:(b + 1) * 64].T).max()
        assert r["tile_score"][t, h, b] >= tok * (1 - 1e-6)


def test_quest_equals_mean_on_constant_blocks():
    """Block of BLOCK_N copies of one key: kmin = kmax = kbar = k, so s_quest = q.k = sqrt(d) * s_mean
    and topk / quest must select identically (d = 64 -> 1/sqrt(d) = 2^-3 is exact)."""
    cfg = synth.CONFIGS["C1"].scaled(1024)
    inp = synth.make_inputs(cfg)
    K = inp.K.copy().reshape(2, 16, 64, 64)
    K[:] = K[:, :, :1, :]
    K = K.reshape(2, 1024, 64)
    meta = oracle.pool(K, 64)
    a = oracle.select(inp.Q, meta, 64, "topk", 4, 0.0, want_scores=True)
    b = oracle.select(inp.Q, meta, 64, "quest", 4, 0.0, want_scores=True)
    assert np.array_equal(a["kv_idx"], b["kv_idx"])
    assert np.array_equal(a["sigma"], b["sigma"])
    vis = np.isfinite(a["tile_score"])
    assert np.array_equal(a["tile_score"][vis] * np.float32(8.0), b["tile_score"][vis])


def test_route_vs_full_sort_and_counts():
    rng = np.random.default_rng(2)
    for T, H, q in [(32, 4, 0.25), (512, 28, 0.25), (1024, 28, 0.1), (2048, 16, 0.5), (2048, 7, 0.4),
                    (33, 3, 0.0), (33, 3, 1.0)]:
        sigma = rng.random((T, H)).astype(np.float32)
        sbar, tau, trig = oracle.route(sigma, "router_quest", q)
        # O8: sequential fp32 sum over heads, then / H
        acc = np.zeros(T, np.float32)
        for h in range(H):
            acc = acc + sigma[:, h]
        assert np.array_equal(sbar, acc / np.float32(H))
        m = min(max(math.ceil(q * T - 1e-9), 0), T)
        if m == 0:
            assert trig.sum() == 0
            continue
        srt = np.sort(sbar)
        assert tau == srt[m - 1]
        assert np.array_equal(trig.astype(bool), sbar <= srt[m - 1])
        if len(np.unique(sbar)) == T:
            assert trig.sum() == m                       # |Pi_q| = ceil(qT)  (L426)
        else:
            assert trig.sum() >= m
    # non-router policies never trigger
    _, tau, trig = oracle.route(rng.random((64, 4)).astype(np.float32), "topk", 0.5)
    assert trig.sum() == 0 and tau == -1.0
    # ties at tau all trigger (G15)
    sig = np.array([[0.5], [0.1], [0.1], [0.1], [0.9], [0.7], [0.3], [0.8]], np.float32)
    _, tau, trig = oracle.route(sig, "router", 0.25)
    assert tau == np.float32(0.1) and trig.sum() == 3


def test_fill_closed_form_and_superset():
    """Eq.14 rules, Eq.15 closed form E[attended] = k(1 + q'(rho-1)), superset (L424)."""
    cfg = synth.CONFIGS["C2"].scaled(8192)            # T = 128, k = 32 -> tiles with t+1 >= 64 are full
    inp = synth.make_inputs(cfg)
    meta = oracle.pool(inp.K, 64)
    k = 16
    r = oracle.select(inp.Q, meta, 64, "router_quest", k, 0.25)
    T, NB = 128, 128
    assert r["trigger"].sum() == math.ceil(0.25 * T)
    full = np.arange(T) + 1 >= 2 * k
    qprime = r["trigger"][full].mean()
    mean_cnt = r["kv_count"][:, full].mean()
    assert abs(mean_cnt - k * (1 + qprime * (oracle.RHO - 1))) < 1e-9
    base = oracle.select(inp.Q, meta, 64, "quest", k, 0.0)
    for t in range(T):
        for h in range(0, 28, 9):
            small = set(base["kv_idx"][h, t][: base["kv_count"][h, t]])
            big = set(r["kv_idx"][h, t][: r["kv_count"][h, t]])
            assert small <= big
            if not r["trigger"][t]:
                assert small == big                     # non-triggered tiles cost the same (L131)
            assert np.all(r["kv_idx"][h, t][r["kv_count"][h, t]:] == NB)
    assert np.all(np.isin(r["kv_count"], [min(k, t + 1) for t in range(T)] + [min(2 * k, t + 1) for t in range(T)]))
