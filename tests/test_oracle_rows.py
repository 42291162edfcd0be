"""Pins of the oracle's per-row scatter-into-bitmap selection (reading G18)."""
import math

import numpy as np

import oracle
from paper_2607_07724_b200 import synth


def _f32(x):
    return (np.asarray(x).astype(np.uint32) << np.uint32(16)).view(np.float32)


def _bits(bitmap, nb):
    return np.unpackbits(bitmap.view(np.uint8), axis=-1, bitorder="little")[..., :nb].astype(bool)


def _setup(n_tiles=12, name="C1rows"):
    cfg = synth.CONFIGS["C1"].scaled(64 * n_tiles, name)
    inp = synth.make_inputs(cfg)
    return cfg, inp, oracle.pool(inp.K, cfg.block)


def test_brute_force_numpy():
    cfg, inp, meta = _setup()
    kmean, kmin, kmax = meta
    T, H, G, Bn, d = cfg.n_blocks, cfg.n_q_heads, cfg.group, cfg.block, cfg.head_dim
    for policy, k_row in (("topk", 3), ("topk", 5), ("quest", 4)):
        bm, cnt = oracle.select_rows_bitmap(inp.Q, meta, Bn, policy, k_row)
        got = _bits(bm, T)
        for t in range(T):
            for h in range(H):
                g = h // G
                q = _f32(inp.Q[h, t * Bn:(t + 1) * Bn]).astype(np.float64)
                if policy == "quest":
                    s = (np.maximum(q, 0) @ _f32(kmax[g, :t + 1]).astype(np.float64).T +
                         np.minimum(q, 0) @ _f32(kmin[g, :t + 1]).astype(np.float64).T).astype(np.float32)
                else:
                    s = (q @ kmean[g, :t + 1].astype(np.float64).T).astype(np.float32) \
                        * np.float32(1.0 / math.sqrt(d))
                want = np.zeros(T, bool)
                want[0] = want[t] = True
                free = np.arange(1, t)
                keep = min(k_row - (1 if t == 0 else 2), len(free))
                for r in range(Bn):
                    if keep > 0:
                        order = np.lexsort((free, -s[r, 1:t].astype(np.float64)))   # score desc, index asc
                        want[free[order[:keep]]] = True
                assert np.array_equal(got[t, h], want), (policy, k_row, t, h)
                assert cnt[t, h] == want.sum()


def test_identical_rows_reduce_to_per_tile_selection():
    """If every row of a tile is the same vector, row score == tile score: the bitmap is exactly the set of
    the per-tile selection (Eq.3-10) with k = k_row."""
    cfg, inp, meta = _setup()
    Qc = inp.Q.copy()
    Qc[:] = Qc[:, ::cfg.block].repeat(cfg.block, axis=1)
    for policy, k in (("topk", 4), ("quest", 5)):
        bm, cnt = oracle.select_rows_bitmap(Qc, meta, cfg.block, policy, k)
        sel = oracle.select(Qc, meta, cfg.block, policy, k, 0.0)
        got = _bits(bm, cfg.n_blocks)
        for t in range(cfg.n_blocks):
            for h in range(cfg.n_q_heads):
                c = sel["kv_count"][h, t]
                assert set(np.nonzero(got[t, h])[0]) == set(sel["kv_idx"][h, t, :c].tolist())
                assert cnt[t, h] == c


def test_bounds_and_full_budget():
    cfg, inp, meta = _setup()
    T, Bn = cfg.n_blocks, cfg.block
    bm, cnt = oracle.select_rows_bitmap(inp.Q, meta, Bn, "topk", T + 5)       # k_row >= N_B: everything
    got = _bits(bm, T)
    for t in range(T):
        assert (got[t, :, :t + 1]).all() and not got[t, :, t + 1:].any()
    k_row = 4
    bm, cnt = oracle.select_rows_bitmap(inp.Q, meta, Bn, "quest", k_row)
    got = _bits(bm, T)
    tt = np.arange(T)
    assert got[:, :, 0].all() and got[tt, :, tt].all()                           # forced sink / self
    for t in range(T):
        assert not got[t, :, t + 1:].any()                                       # causal
        lo = min(k_row, t + 1)
        hi = min(t + 1, 2 + Bn * (k_row - 2))
        assert ((cnt[t] >= lo) & (cnt[t] <= hi)).all()
    kv, kc = oracle.bitmap_to_kv_idx(bm, T)
    assert np.array_equal(kc, cnt.T) and (kv[:, :, 0] == 0).all()
