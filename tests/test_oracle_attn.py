"""Pins for oracle O11/O12 (PAPER.md L43-47 softmax definition; L131, L342 kv_idx iteration)."""
import math

import numpy as np
import torch

import oracle
from paper_2607_07724_b200 import synth


def _t(x):
    return torch.from_numpy(synth.bf16_to_f32(x).astype(np.float64))


def test_dense_vs_torch_sdpa(c1_inputs):
    """Dense special case against a library routine (torch CPU SDPA, fp64, causal, GQA expanded)."""
    cfg = c1_inputs.cfg
    Q, K, V = _t(c1_inputs.Q), _t(c1_inputs.K), _t(c1_inputs.V)
    Kx = K.repeat_interleave(cfg.group, dim=0)
    Vx = V.repeat_interleave(cfg.group, dim=0)
    ref = torch.nn.functional.scaled_dot_product_attention(Q[None], Kx[None], Vx[None], is_causal=True)[0]
    O, lse = oracle.attn_full(c1_inputs.Q, c1_inputs.K, c1_inputs.V, cfg.block)
    assert np.abs(O - ref.numpy()).max() < 1e-6
    logits = (Q @ Kx.transpose(1, 2)) / math.sqrt(cfg.head_dim)
    logits = logits.masked_fill(torch.triu(torch.ones(cfg.seqlen, cfg.seqlen, dtype=torch.bool), 1), -math.inf)
    assert np.abs(lse - torch.logsumexp(logits, -1).numpy()).max() < 1e-5


def test_sparse_brute_force_masked_softmax(c1_inputs, c1_meta):
    """Sparse attention == dense softmax with every non-selected block masked out (numpy fp64)."""
    cfg = c1_inputs.cfg
    r = oracle.select(c1_inputs.Q, c1_meta, cfg.block, "router", cfg.k_budget, 0.25)
    Q, K, V = _t(c1_inputs.Q).numpy(), _t(c1_inputs.K).numpy(), _t(c1_inputs.V).numpy()
    pairs = [(0, 0), (1, 1), (7, 2), (31, 3), (20, 0), (13, 1)]
    O, lse = oracle.attn_pairs(c1_inputs.Q, c1_inputs.K, c1_inputs.V, 64, pairs, r["kv_idx"], r["kv_count"])
    for n, (t, h) in enumerate(pairs):
        g = h // cfg.group
        blocks = r["kv_idx"][h, t][: r["kv_count"][h, t]]
        rows = np.arange(t * 64, (t + 1) * 64)
        logits = Q[h, rows] @ K[g].T / math.sqrt(64)
        keep = np.zeros(cfg.seqlen, bool)
        for b in blocks:
            keep[b * 64:(b + 1) * 64] = True
        mask = keep[None, :] & (np.arange(cfg.seqlen)[None, :] <= rows[:, None])
        logits = np.where(mask, logits, -np.inf)
        p = np.exp(logits - logits.max(axis=1, keepdims=True))
        want = (p / p.sum(axis=1, keepdims=True)) @ V[g]
        assert np.abs(O[n] - want).max() < 1e-6
        want_lse = logits.max(axis=1) + np.log(p.sum(axis=1))
        assert np.abs(lse[n] - want_lse).max() < 1e-5


def test_full_budget_equals_dense(c1_inputs, c1_meta):
    """k_budget >= N_B  =>  sparse == dense (north_star invariant)."""
    cfg = c1_inputs.cfg
    r = oracle.select(c1_inputs.Q, c1_meta, cfg.block, "topk", cfg.n_blocks, 0.0)
    assert np.all(r["kv_count"] == np.arange(1, cfg.n_blocks + 1)[None, :])
    Os, ls = oracle.attn_full(c1_inputs.Q, c1_inputs.K, c1_inputs.V, 64, r["kv_idx"], r["kv_count"])
    Od, ld = oracle.attn_full(c1_inputs.Q, c1_inputs.K, c1_inputs.V, 64)
    assert np.array_equal(Os, Od) and np.array_equal(ls, ld)


def test_permutation_sentinel_and_bounds(c1_inputs, c1_meta):
    cfg = c1_inputs.cfg
    r = oracle.select(c1_inputs.Q, c1_meta, cfg.block, "router", cfg.k_budget, 0.25)
    pairs = [(9, 0), (30, 3)]
    O1, _ = oracle.attn_pairs(c1_inputs.Q, c1_inputs.K, c1_inputs.V, 64, pairs, r["kv_idx"], r["kv_count"])
    # permuting a kv_idx row (sentinels mixed in, no kv_count) leaves the output unchanged
    kv = r["kv_idx"].copy()
    rng = np.random.default_rng(3)
    for t, h in pairs:
        kv[h, t] = rng.permutation(kv[h, t])
    O2, _ = oracle.attn_pairs(c1_inputs.Q, c1_inputs.K, c1_inputs.V, 64, pairs, kv, None)
    assert np.array_equal(O1, O2)
    # every output coordinate is a convex combination of the attended V rows
    V = synth.bf16_to_f32(c1_inputs.V)
    for n, (t, h) in enumerate(pairs):
        g = h // cfg.group
        blocks = r["kv_idx"][h, t][: r["kv_count"][h, t]]
        rows = np.concatenate([V[g, b * 64:(b + 1) * 64] for b in blocks])
        assert np.all(O1[n] <= rows.max(axis=0) + 1e-6) and np.all(O1[n] >= rows.min(axis=0) - 1e-6)
    # tile 0, row 0 attends exactly one key: output == v_0
    O0, l0 = oracle.attn_pairs(c1_inputs.Q, c1_inputs.K, c1_inputs.V, 64, [(0, 1)], r["kv_idx"], r["kv_count"])
    assert np.array_equal(O0[0, 0], V[0, 0])
    q0 = synth.bf16_to_f32(c1_inputs.Q)[1, 0].astype(np.float64)
    k0 = synth.bf16_to_f32(c1_inputs.K)[0, 0].astype(np.float64)
    assert abs(l0[0, 0] - q0 @ k0 / 8.0) < 1e-5


def test_block128_dim256_gqa():
    cfg = synth.CONFIGS["C5"].scaled(1024)
    inp = synth.make_inputs(cfg)
    Q, K, V = _t(inp.Q), _t(inp.K), _t(inp.V)
    Kx = K.repeat_interleave(cfg.group, dim=0)
    Vx = V.repeat_interleave(cfg.group, dim=0)
    ref = torch.nn.functional.scaled_dot_product_attention(Q[None], Kx[None], Vx[None], is_causal=True)[0]
    O, _ = oracle.attn_full(inp.Q, inp.K, inp.V, 128)
    assert np.abs(O - ref.numpy()).max() < 1e-6
