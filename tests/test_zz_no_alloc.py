"""bsa_select_static -- the entry point that allocates nothing (include/bsa.h): its scratch (sigma_bar,
trigger) is a static __device__ array inside libbsa.  Collected last on purpose (pytest -x at the round's
end must not lose the other tests to a failure here).  Passes alone in a fresh process and after the other
GPU tests: it depends on nothing they leave behind."""
import ctypes

import pytest


def _shape(binding, batch, seqlen):
    s = binding.BsaShape()
    s.batch, s.seqlen, s.n_q_heads, s.n_kv_heads, s.head_dim, s.block = batch, seqlen, 4, 2, 64, 64
    s.q_stride_n = s.kv_stride_n = 64
    s.q_stride_h = s.kv_stride_h = seqlen * 64
    s.q_stride_b, s.kv_stride_b = 4 * s.q_stride_h, 2 * s.kv_stride_h
    return s


def test_static_limit_is_checked_on_the_host():
    """more tiles than the static array holds: a clear BSA_ERR_UNSUPPORTED before any device call"""
    from paper_2607_07724_b200 import binding
    lib = binding.load_library()
    one = ctypes.c_void_p(256)            # never dereferenced: the limit check comes first
    tiles = binding.BSA_STATIC_MAX_TILES // 4 + 1
    st = lib.bsa_select_static(ctypes.byref(_shape(binding, 4, tiles * 64)), one, one, 3, 16, 0.25, one, one,
                               one, one, None)
    assert st == 2                        # BSA_ERR_UNSUPPORTED
    msg = lib.bsa_last_error().decode()
    assert "bsa_select_static" in msg and str(binding.BSA_STATIC_MAX_TILES) in msg and str(4 * tiles) in msg
    st = lib.bsa_select_static(ctypes.byref(_shape(binding, 1, 4096)), None, one, 3, 16, 0.25, one, one, one,
                               one, None)
    assert st == 1                        # BSA_ERR_INVALID_ARG: Q is NULL


@pytest.mark.gpu
def test_static_scratch_select_matches_bsa_select():
    """two calls in a row (different shape, policy and budget, so the second one runs over the first one's
    leftovers in the shared array): kv_idx / kv_count bit-exact and sigma / tau bit-equal to bsa_select on the
    same inputs -- the same kernels run, only the scratch lives elsewhere; and no device memory is taken."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_07724_b200 import binding as bsa
    from paper_2607_07724_b200 import synth
    from parity_util import to_torch_bf16
    C = synth.CONFIGS
    calls = [(C["C2"].scaled(8192, "C2m"), "router_quest", 0.25),
             (C["C5"].scaled(4096, "C5m"), "router", 0.4),
             (C["C2"].scaled(8192, "C2m"), "topk", 0.0)]
    prepared = []
    for cfg, policy, q in calls:
        inp = synth.make_inputs(cfg)
        Q, K = to_torch_bf16(inp.Q)[None], to_torch_bf16(inp.K)[None]
        buf = bsa.bsa_build_block_meta(K, cfg.block, 3)
        ref = bsa.bsa_select(Q, buf, K, cfg.block, policy, cfg.k_budget, q)        # the existing path
        out = {n: torch.full_like(ref[n], -7) for n in ("kv_idx", "kv_count", "sigma", "tau")}
        prepared.append((cfg, policy, q, Q, K, buf, ref, out))
    torch.cuda.synchronize()
    # back to back on one stream, nothing in between
    for cfg, policy, q, Q, K, buf, ref, out in prepared:
        bsa.bsa_select_static(Q, buf, K, cfg.block, policy, cfg.k_budget, q, out)
    torch.cuda.synchronize()
    for cfg, policy, q, Q, K, buf, ref, out in prepared:
        for n in ("kv_idx", "kv_count"):
            assert torch.equal(out[n], ref[n]), (cfg.name, policy, n)
        for n in ("sigma", "tau"):                                                 # tests' sigma tolerance: 1e-4
            assert torch.allclose(out[n], ref[n], rtol=0, atol=1e-4), (cfg.name, policy, n)
            assert torch.equal(out[n].view(torch.int32), ref[n].view(torch.int32)), (cfg.name, policy, n)
    # a repeated call takes no device memory (every kernel is loaded by now, outputs exist)
    cfg, policy, q, Q, K, buf, ref, out = prepared[0]
    free0, _ = torch.cuda.mem_get_info()
    bsa.bsa_select_static(Q, buf, K, cfg.block, policy, cfg.k_budget, q, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    assert torch.equal(out["kv_idx"], ref["kv_idx"])
