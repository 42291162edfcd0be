"""CPU-side checks of the C-ABI library: it builds with nvcc (cross-compile, no GPU), loads, exports
every symbol include/bsa.h declares, and its host-only entry points and argument validation behave
as the header states.  No compute call is made here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "bsa.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2607_07724_b200 import binding, build
    build.build_lib()
    return binding.load_library()


def _declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(bsa_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared_symbols()
    assert {"bsa_build_block_meta", "bsa_select", "bsa_sparse_attn_fwd", "bsa_dense_attn_fwd",
            "bsa_block_meta_bytes", "bsa_kv_width", "bsa_select_workspace_bytes",
            "bsa_last_error", "bsa_version"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in bsa.h but not exported"


def test_no_torch_or_oracle_dependency():
    """the boundary is plain C: libbsa links neither torch nor the oracle"""
    import subprocess
    from paper_2607_07724_b200 import build
    out = subprocess.run(["ldd", build.LIB], capture_output=True, text=True).stdout
    assert "torch" not in out and "oracle" not in out
    pkg = os.path.join(ROOT, "paper_2607_07724_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".c")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert "bsa_oracle" not in txt, f


def _shape(binding, **kw):
    d = dict(batch=1, seqlen=2048, n_q_heads=4, n_kv_heads=2, head_dim=64, block=64)
    d.update(kw)
    s = binding.BsaShape()
    for k, v in d.items():
        setattr(s, k, v)
    s.q_stride_n = s.kv_stride_n = s.head_dim
    s.q_stride_h = s.kv_stride_h = s.seqlen * s.head_dim
    s.q_stride_b = s.n_q_heads * s.q_stride_h
    s.kv_stride_b = s.n_kv_heads * s.kv_stride_h
    return s


def test_host_only_entry_points(lib):
    from paper_2607_07724_b200 import binding
    assert lib.bsa_version().decode().startswith("bsa ")
    assert lib.bsa_kv_width(binding.POLICIES["topk"], 32) == 32
    assert lib.bsa_kv_width(binding.POLICIES["quest"], 32) == 32
    assert lib.bsa_kv_width(binding.POLICIES["router"], 32) == 64          # rho = 2
    assert lib.bsa_kv_width(binding.POLICIES["router_quest"], 33) == 66
    s = _shape(binding)
    n = 1 * 2 * 32 * 64
    nbytes = lib.bsa_block_meta_bytes(ctypes.byref(s), 3)
    assert nbytes >= n * (4 + 2 + 2)
    off = lib.bsa_block_meta_offset(ctypes.byref(s), binding.BSA_META_MINMAX)
    assert off >= n * 4 and off % 256 == 0
    assert lib.bsa_block_meta_offset(ctypes.byref(s), binding.BSA_META_MEAN) == 0
    assert lib.bsa_select_workspace_bytes(ctypes.byref(s), 1, 4) >= 32 * 5
    assert lib.bsa_block_meta_bytes(ctypes.byref(_shape(binding, seqlen=2000)), 3) == 0


@pytest.mark.parametrize("kw,code", [
    (dict(seqlen=2000), 1),            # seqlen % block
    (dict(n_q_heads=5), 1),            # heads % kv heads
    (dict(block=32), 2),               # unsupported block
    (dict(head_dim=96), 2),            # unsupported head_dim
])
def test_argument_validation_precedes_any_launch(lib, kw, code):
    from paper_2607_07724_b200 import binding
    s = _shape(binding, **kw)
    buf = ctypes.create_string_buffer(4096)
    p = ctypes.addressof(buf)
    p = (p + 255) // 256 * 256
    st = lib.bsa_build_block_meta(ctypes.byref(s), p, 3, p, None)
    assert st == code, lib.bsa_last_error()
    assert lib.bsa_last_error().decode() != ""
    st = lib.bsa_dense_attn_fwd(ctypes.byref(s), p, p, p, ctypes.c_float(0.0), p, None, None)
    assert st == code


def test_select_argument_validation(lib):
    from paper_2607_07724_b200 import binding
    s = _shape(binding)
    buf = ctypes.create_string_buffer(4096)
    p = (ctypes.addressof(buf) + 255) // 256 * 256
    args = lambda pol, k, q: (ctypes.byref(s), p, p, pol, k, ctypes.c_double(q), p, p, p, p, p, p, None, 0, None)
    assert lib.bsa_select(*args(1, 2, 0.25)) == 1          # k_budget < 3
    assert lib.bsa_select(*args(1, 4, 1.5)) == 1           # q_frac outside [0,1]
    assert lib.bsa_select(*args(7, 4, 0.25)) == 1          # unknown policy
    assert lib.bsa_select(ctypes.byref(s), None, p, 0, 4, ctypes.c_double(0.2), p, p, p, p, p, p,
                          None, 0, None) == 1              # NULL Q
    assert lib.bsa_sparse_attn_fwd(ctypes.byref(s), p, p, p, None, None, 4, ctypes.c_float(0), p, None,
                                   None) == 1              # NULL kv_idx
    assert lib.bsa_sparse_attn_fwd(ctypes.byref(s), p + 2, p, p, p, None, 4, ctypes.c_float(0), p, None,
                                   None) == 1              # misaligned Q


def test_round2_entry_points_validate_before_any_launch(lib):
    """bsa_select_diag, the varlen calls and the per-row bitmap calls: host-side validation only."""
    from paper_2607_07724_b200 import binding
    s = _shape(binding)
    buf = ctypes.create_string_buffer(4096)
    p = (ctypes.addressof(buf) + 255) // 256 * 256
    dbl = ctypes.c_double
    # diagnostics: a NULL diag struct, a NULL member and a NULL tau are refused
    sel = lambda diag, tau: lib.bsa_select_diag(ctypes.byref(s), p, p, 1, 4, dbl(0.25), p, p, p, p, p, tau,
                                                diag, None, 0, None)
    assert sel(None, p) == 1
    d = binding.BsaDiagOut(p, p, p, p, p, None)
    assert sel(ctypes.byref(d), p) == 1
    d = binding.BsaDiagOut(p, p, p, p, p, p)
    assert sel(ctypes.byref(d), None) == 1
    assert b"diagnostics" in lib.bsa_last_error()
    # per-row bitmap: policy must be a backbone (TOPK / QUEST), 3 <= k_row <= 64
    rows = lambda pol, k: lib.bsa_select_rows_bitmap(ctypes.byref(s), p, p, pol, k, p, p, None)
    assert rows(1, 8) == 1 and rows(3, 8) == 1            # router policies have no per-row meaning
    assert rows(0, 2) == 1                                # k_row < 3
    assert rows(2, 65) == 2                               # BSA_ERR_UNSUPPORTED
    assert lib.bsa_bitmap_words(ctypes.byref(s)) == (s.seqlen // s.block + 31) // 32
    assert lib.bsa_sparse_attn_fwd_bitmap(ctypes.byref(s), p, p, p, None, ctypes.c_float(0), p, None, None) == 1
    # varlen: cu_seqlens must run from 0 to seqlen in multiples of block, batch must be 1
    i32 = ctypes.c_int32
    cu = lambda *v: (i32 * len(v))(*v)
    N = s.seqlen
    ok = cu(0, N // 2, N // 2, N)                          # an empty sequence is allowed
    assert lib.bsa_block_meta_bytes_varlen(ctypes.byref(s), ok, 3, 3) > 0
    assert lib.bsa_block_meta_bytes_varlen(ctypes.byref(s), cu(0, N // 2 + 1, N), 2, 3) == 0
    bad = [cu(64, N), cu(0, N - 64), cu(0, 100, N), cu(0, N, N // 2)]
    for c in bad:
        n = len(c) - 1
        assert lib.bsa_build_block_meta_varlen(ctypes.byref(s), c, n, p, 3, p, None) == 1, list(c)
        assert lib.bsa_select_varlen(ctypes.byref(s), c, n, p, p, 1, 4, dbl(0.25), p, p, p, p, p, p, None) == 1
        assert lib.bsa_dense_attn_fwd_varlen(ctypes.byref(s), c, n, p, p, p, ctypes.c_float(0), p, None, None) == 1
    assert lib.bsa_select_varlen(ctypes.byref(s), ok, 3, p, p, 1, 4, dbl(0.25), p, p, p, None, p, p, None) == 1
    assert lib.bsa_sparse_attn_fwd_varlen(ctypes.byref(s), ok, 3, p, p, p, None, None, 4, ctypes.c_float(0), p,
                                          None, None) == 1
    s2 = _shape(binding, batch=2)
    assert lib.bsa_build_block_meta_varlen(ctypes.byref(s2), ok, 3, p, 3, p, None) == 1
    # limits of bsa_select are argument errors, not launches
    big = _shape(binding, seqlen=64 * 8256)
    assert lib.bsa_select(ctypes.byref(big), p, p, 0, 4, dbl(0.2), p, p, p, p, p, p, None, 0, None) == 2
    assert b"8192" in lib.bsa_last_error()
