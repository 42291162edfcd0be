"""Pins for oracle O1/O2 (Eq.1/Eq.6 L74,L293; Eq.2)."""
import numpy as np

import oracle
from paper_2607_07724_b200 import synth


def test_pool_brute_force(c1_inputs):
    K = c1_inputs.K
    kmean, kmin, kmax = oracle.pool(K, 64)
    Kf = synth.bf16_to_f32(K).astype(np.float64).reshape(2, 32, 64, 64)
    assert np.array_equal(kmean, Kf.mean(axis=2).astype(np.float32))
    assert np.array_equal(synth.bf16_to_f32(kmin), Kf.min(axis=2).astype(np.float32))
    assert np.array_equal(synth.bf16_to_f32(kmax), Kf.max(axis=2).astype(np.float32))


def test_pool_constant_block():
    K = np.full((1, 128, 16), synth.f32_to_bf16(np.array([1.5], np.float32))[0], np.uint16)
    K[0, 64:, :] = synth.f32_to_bf16(np.array([-0.25], np.float32))[0]
    kmean, kmin, kmax = oracle.pool(K, 64)
    assert np.all(kmean[0, 0] == 1.5) and np.all(kmean[0, 1] == -0.25)
    assert np.all(synth.bf16_to_f32(kmin)[0, 0] == 1.5) and np.all(synth.bf16_to_f32(kmax)[0, 1] == -0.25)


def test_pool_linearity(c1_inputs):
    """q . kbar_b == mean_j q . k_j  (Eq.1): pins the 1/BLOCK_N factor and the block boundaries."""
    K, Q = c1_inputs.K, c1_inputs.Q
    kmean, _, _ = oracle.pool(K, 64)
    Kf = synth.bf16_to_f32(K).astype(np.float64)
    q = synth.bf16_to_f32(Q[0, 100]).astype(np.float64)
    lhs = kmean[0].astype(np.float64) @ q
    rhs = (Kf[0] @ q).reshape(32, 64).mean(axis=1)
    assert np.allclose(lhs, rhs, rtol=0, atol=1e-5)


def test_pool_block128():
    K = synth.gauss_bf16(5, synth.TID_K, 1, 512, 32, 128)
    kmean, kmin, kmax = oracle.pool(K, 128)
    Kf = synth.bf16_to_f32(K).astype(np.float64).reshape(1, 4, 128, 32)
    assert kmean.shape == (1, 4, 32)
    assert np.array_equal(kmean, Kf.mean(axis=2).astype(np.float32))
    assert np.all(synth.bf16_to_f32(kmin) <= kmean) and np.all(synth.bf16_to_f32(kmax) >= kmean)
