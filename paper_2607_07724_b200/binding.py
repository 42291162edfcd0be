"""Thin ctypes binding of libbsa.so (include/bsa.h).  Argument marshalling only: every step of the
hot path runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory and streams.

Tensors: Q, O [B, Hq, N, d]; K, V [B, Hkv, N, d], bf16, CUDA, head_dim contiguous (any strides that
are multiples of 8 elements).  Functions keep the names of the C entry points.
"""
from __future__ import annotations

import ctypes
import os

import torch

from .build import LIB, build_lib

BSA_OK = 0
BSA_META_MEAN, BSA_META_MINMAX, BSA_META_SPLIT = 1, 2, 4
BSA_DIAG_SUMMARY_LEN = 16
DIAG_SUMMARY = ("n", "r_bar", "cv_r", "sigma_q", "gamma_q", "band_mass", "d2_q10", "d2_q50", "tau_hat",
                "zero_gap_frac", "g_q40_pos", "g_q40_pos_over_tau_hat")
BSA_RHO = 2
BSA_STATIC_MAX_TILES = 16384
POLICIES = {"topk": 0, "router": 1, "quest": 2, "router_quest": 3}
STATUS = {0: "BSA_OK", 1: "BSA_ERR_INVALID_ARG", 2: "BSA_ERR_UNSUPPORTED",
          3: "BSA_ERR_WORKSPACE_TOO_SMALL", 4: "BSA_ERR_CUDA"}


class BsaShape(ctypes.Structure):
    _fields_ = [("batch", ctypes.c_int32), ("seqlen", ctypes.c_int32), ("n_q_heads", ctypes.c_int32),
                ("n_kv_heads", ctypes.c_int32), ("head_dim", ctypes.c_int32), ("block", ctypes.c_int32),
                ("q_stride_b", ctypes.c_int64), ("q_stride_h", ctypes.c_int64),
                ("q_stride_n", ctypes.c_int64), ("kv_stride_b", ctypes.c_int64),
                ("kv_stride_h", ctypes.c_int64), ("kv_stride_n", ctypes.c_int64)]


class BsaDiagOut(ctypes.Structure):
    _fields_ = [(n, ctypes.c_void_p) for n in ("g", "G", "r", "d2", "rough", "summary")]


class BsaError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS.get(status, status)}: {message}")
        self.status = status


_lib = None


def load_library(path: str | None = None) -> ctypes.CDLL:
    """Load libbsa.so.  There is no fallback: a missing library is an error."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB
    if path is None:
        build_lib()  # no-op when libbsa.so matches the sources (hash); raises if the build fails
    lib = ctypes.CDLL(p)
    vp, sz, i32, sp = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int32, ctypes.POINTER(BsaShape)
    lib.bsa_block_meta_bytes.argtypes = [sp, ctypes.c_int]
    lib.bsa_block_meta_bytes.restype = sz
    lib.bsa_block_meta_offset.argtypes = [sp, ctypes.c_int]
    lib.bsa_block_meta_offset.restype = sz
    lib.bsa_build_block_meta.argtypes = [sp, vp, ctypes.c_int, vp, vp]
    lib.bsa_build_block_meta.restype = ctypes.c_int
    lib.bsa_kv_width.argtypes = [ctypes.c_int, i32]
    lib.bsa_kv_width.restype = i32
    lib.bsa_select_workspace_bytes.argtypes = [sp, ctypes.c_int, i32]
    lib.bsa_select_workspace_bytes.restype = sz
    lib.bsa_select.argtypes = [sp, vp, vp, ctypes.c_int, i32, ctypes.c_double, vp, vp, vp, vp, vp, vp,
                               vp, sz, vp]
    lib.bsa_select.restype = ctypes.c_int
    lib.bsa_select_static.argtypes = [sp, vp, vp, ctypes.c_int, i32, ctypes.c_double, vp, vp, vp, vp, vp]
    lib.bsa_select_static.restype = ctypes.c_int
    lib.bsa_select_diag.argtypes = [sp, vp, vp, ctypes.c_int, i32, ctypes.c_double, vp, vp, vp, vp, vp, vp,
                                    ctypes.POINTER(BsaDiagOut), vp, sz, vp]
    lib.bsa_select_diag.restype = ctypes.c_int
    lib.bsa_sparse_attn_fwd.argtypes = [sp, vp, vp, vp, vp, vp, i32, ctypes.c_float, vp, vp, vp]
    lib.bsa_sparse_attn_fwd.restype = ctypes.c_int
    lib.bsa_select_attn_fwd.argtypes = [sp, vp, vp, vp, vp, ctypes.c_int, i32, ctypes.c_double, vp, vp, vp, vp, vp,
                                        vp, ctypes.c_float, vp, vp, vp, sz, vp]
    lib.bsa_select_attn_fwd.restype = ctypes.c_int
    lib.bsa_dense_attn_fwd.argtypes = [sp, vp, vp, vp, ctypes.c_float, vp, vp, vp]
    lib.bsa_dense_attn_fwd.restype = ctypes.c_int
    ip = ctypes.POINTER(ctypes.c_int32)
    lib.bsa_block_meta_bytes_varlen.argtypes = [sp, ip, i32, ctypes.c_int]
    lib.bsa_block_meta_bytes_varlen.restype = sz
    lib.bsa_build_block_meta_varlen.argtypes = [sp, ip, i32, vp, ctypes.c_int, vp, vp]
    lib.bsa_build_block_meta_varlen.restype = ctypes.c_int
    lib.bsa_select_varlen.argtypes = [sp, ip, i32, vp, vp, ctypes.c_int, i32, ctypes.c_double, vp, vp, vp, vp,
                                      vp, vp, vp]
    lib.bsa_select_varlen.restype = ctypes.c_int
    lib.bsa_sparse_attn_fwd_varlen.argtypes = [sp, ip, i32, vp, vp, vp, vp, vp, i32, ctypes.c_float, vp, vp, vp]
    lib.bsa_sparse_attn_fwd_varlen.restype = ctypes.c_int
    lib.bsa_dense_attn_fwd_varlen.argtypes = [sp, ip, i32, vp, vp, vp, ctypes.c_float, vp, vp, vp]
    lib.bsa_dense_attn_fwd_varlen.restype = ctypes.c_int
    lib.bsa_bitmap_words.argtypes = [sp]
    lib.bsa_bitmap_words.restype = sz
    lib.bsa_select_rows_bitmap.argtypes = [sp, vp, vp, ctypes.c_int, i32, vp, vp, vp]
    lib.bsa_select_rows_bitmap.restype = ctypes.c_int
    lib.bsa_sparse_attn_fwd_bitmap.argtypes = [sp, vp, vp, vp, vp, ctypes.c_float, vp, vp, vp]
    lib.bsa_sparse_attn_fwd_bitmap.restype = ctypes.c_int
    lib.bsa_last_error.restype = ctypes.c_char_p
    lib.bsa_version.restype = ctypes.c_char_p
    if path is None:
        _lib = lib
    return lib


def _check(status: int):
    if status != BSA_OK:
        raise BsaError(status, load_library().bsa_last_error().decode())


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _ptr(t):
    return None if t is None else t.data_ptr()


def make_shape(Q: torch.Tensor | None, K: torch.Tensor, block: int, n_q_heads: int | None = None):
    """bsa_shape from the tensors (Q may be None for the pooling call)."""
    B, Hkv, N, d = K.shape
    assert K.dtype == torch.bfloat16 and K.stride(3) == 1
    s = BsaShape()
    s.batch, s.seqlen, s.n_kv_heads, s.head_dim, s.block = B, N, Hkv, d, block
    s.kv_stride_b, s.kv_stride_h, s.kv_stride_n = K.stride(0), K.stride(1), K.stride(2)
    if Q is not None:
        assert Q.dtype == torch.bfloat16 and Q.stride(3) == 1 and Q.shape[0] == B and Q.shape[2] == N
        s.n_q_heads = Q.shape[1]
        s.q_stride_b, s.q_stride_h, s.q_stride_n = Q.stride(0), Q.stride(1), Q.stride(2)
    else:
        s.n_q_heads = n_q_heads or Hkv
        s.q_stride_b, s.q_stride_h, s.q_stride_n = s.n_q_heads * N * d, N * d, d
    return s


def bsa_block_meta_bytes(shape: BsaShape, kinds: int = 3) -> int:
    return int(load_library().bsa_block_meta_bytes(ctypes.byref(shape), kinds))


def bsa_build_block_meta(K: torch.Tensor, block: int, kinds: int = 3, meta: torch.Tensor | None = None):
    """Pools K into the block metadata buffer (uint8 tensor).  Returns meta."""
    lib = load_library()
    shape = make_shape(None, K, block)
    nbytes = bsa_block_meta_bytes(shape, kinds)
    if nbytes == 0:
        _check(lib.bsa_build_block_meta(ctypes.byref(shape), _ptr(K), kinds, None, _stream()))
    if meta is None:
        meta = torch.empty(nbytes, dtype=torch.uint8, device=K.device)
    assert meta.numel() >= nbytes and meta.is_cuda
    _check(lib.bsa_build_block_meta(ctypes.byref(shape), _ptr(K), kinds, _ptr(meta), _stream()))
    return meta


def meta_views(meta: torch.Tensor, K_shape, block: int):
    """(kmean fp32, kmin bf16, kmax bf16) views of a meta buffer, each [B, Hkv, N_B, d]."""
    B, Hkv, N, d = K_shape
    NB = N // block
    n = B * Hkv * NB * d
    s = BsaShape(B, N, Hkv, Hkv, d, block, Hkv * N * d, N * d, d, Hkv * N * d, N * d, d)
    off = int(load_library().bsa_block_meta_offset(ctypes.byref(s), BSA_META_MINMAX))
    kmean = meta[:n * 4].view(torch.float32).view(B, Hkv, NB, d)
    kmin = meta[off:off + 2 * n].view(torch.bfloat16).view(B, Hkv, NB, d)
    kmax = meta[off + 2 * n:off + 4 * n].view(torch.bfloat16).view(B, Hkv, NB, d)
    return kmean, kmin, kmax


def meta_split_view(meta: torch.Tensor, K_shape, block: int):
    """The three bf16 planes hi, mid, lo (hi + mid + lo == kmean) as one view [3, B, Hkv, N_B, d]."""
    B, Hkv, N, d = K_shape
    NB = N // block
    n = B * Hkv * NB * d
    s = BsaShape(B, N, Hkv, Hkv, d, block, Hkv * N * d, N * d, d, Hkv * N * d, N * d, d)
    off = int(load_library().bsa_block_meta_offset(ctypes.byref(s), BSA_META_SPLIT))
    return meta[off:off + 6 * n].view(torch.bfloat16).view(3, B, Hkv, NB, d)


def bsa_kv_width(policy: str, k_budget: int) -> int:
    return int(load_library().bsa_kv_width(POLICIES[policy], k_budget))


def bsa_select(Q: torch.Tensor, meta: torch.Tensor, K_like: torch.Tensor, block: int, policy: str,
               k_budget: int, q_frac: float, out: dict | None = None, diag: bool = False,
               use_workspace: bool = False) -> dict:
    """Selection.  K_like only provides the K/V shape and strides.  Returns a dict with kv_idx
    [B,Hq,T,W] int32, kv_count [B,Hq,T] int32, sigma [B,Hq,T] f32, sigma_bar [B,T] f32,
    trigger [B,T] u8, tau [B] f32.  `out` may carry preallocated tensors of those names.
    diag=True calls bsa_select_diag and adds g, G, r, d2, rough [B,Hq,T] f32 and summary [B,16] f32.
    use_workspace=True passes sigma_bar = trigger = NULL and a workspace buffer instead (the results
    then stay inside the library's workspace; `sigma_bar` / `trigger` are absent from the dict)."""
    lib = load_library()
    shape = make_shape(Q, K_like, block)
    B, H, N, _ = Q.shape
    T = N // block
    W = bsa_kv_width(policy, k_budget)
    dev = Q.device
    o = dict(out) if out else {}
    o.setdefault("kv_idx", torch.empty((B, H, T, max(W, 1)), dtype=torch.int32, device=dev))
    o.setdefault("kv_count", torch.empty((B, H, T), dtype=torch.int32, device=dev))
    o.setdefault("sigma", torch.empty((B, H, T), dtype=torch.float32, device=dev))
    o.setdefault("tau", torch.empty((B,), dtype=torch.float32, device=dev))
    ws, ws_bytes = None, 0
    if use_workspace:
        ws_bytes = int(lib.bsa_select_workspace_bytes(ctypes.byref(shape), POLICIES[policy], k_budget))
        ws = torch.empty(ws_bytes, dtype=torch.uint8, device=dev)
        o["workspace"] = ws
        sb, tr = None, None
    else:
        o.setdefault("sigma_bar", torch.empty((B, T), dtype=torch.float32, device=dev))
        o.setdefault("trigger", torch.empty((B, T), dtype=torch.uint8, device=dev))
        sb, tr = o["sigma_bar"], o["trigger"]
    args = [ctypes.byref(shape), _ptr(Q), _ptr(meta), POLICIES[policy], k_budget, float(q_frac),
            _ptr(o["kv_idx"]), _ptr(o["kv_count"]), _ptr(o["sigma"]), _ptr(sb), _ptr(tr), _ptr(o["tau"])]
    if diag:
        for n in ("g", "G", "r", "d2", "rough"):
            o.setdefault(n, torch.empty((B, H, T), dtype=torch.float32, device=dev))
        o.setdefault("summary", torch.empty((B, BSA_DIAG_SUMMARY_LEN), dtype=torch.float32, device=dev))
        d = BsaDiagOut(*[_ptr(o[n]) for n in ("g", "G", "r", "d2", "rough", "summary")])
        _check(lib.bsa_select_diag(*args, ctypes.byref(d), _ptr(ws), ws_bytes, _stream()))
    else:
        _check(lib.bsa_select(*args, _ptr(ws), ws_bytes, _stream()))
    o["W"] = W
    return o


def bsa_select_static(Q: torch.Tensor, meta: torch.Tensor, K_like: torch.Tensor, block: int, policy: str,
                      k_budget: int, q_frac: float, out: dict) -> dict:
    """bsa_select_static: the selection with its scratch in the library's static device array.  The C call
    allocates nothing, and neither does this wrapper: `out` must carry kv_idx [B,Hq,T,W] int32, kv_count
    [B,Hq,T] int32, sigma [B,Hq,T] f32 and tau [B] f32.  Returns `out`."""
    lib = load_library()
    shape = make_shape(Q, K_like, block)
    _check(lib.bsa_select_static(ctypes.byref(shape), _ptr(Q), _ptr(meta), POLICIES[policy], k_budget,
                                 float(q_frac), _ptr(out["kv_idx"]), _ptr(out["kv_count"]), _ptr(out["sigma"]),
                                 _ptr(out["tau"]), _stream()))
    return out


def bsa_sparse_attn_fwd(Q, K, V, kv_idx, kv_count, block: int, softmax_scale: float = 0.0,
                        O: torch.Tensor | None = None, lse: torch.Tensor | None = None,
                        want_lse: bool = False):
    lib = load_library()
    shape = make_shape(Q, K, block)
    assert V.shape == K.shape and V.stride() == K.stride()
    if O is None:
        O = torch.empty_like(Q)
    assert O.stride() == Q.stride()
    if lse is None and want_lse:
        lse = torch.empty(Q.shape[:3], dtype=torch.float32, device=Q.device)
    assert kv_idx.dtype == torch.int32 and kv_idx.is_contiguous()
    _check(lib.bsa_sparse_attn_fwd(ctypes.byref(shape), _ptr(Q), _ptr(K), _ptr(V), _ptr(kv_idx),
                                   _ptr(kv_count), kv_idx.shape[-1], float(softmax_scale), _ptr(O),
                                   _ptr(lse), _stream()))
    return O, lse


def bsa_select_attn_fwd(Q, K, V, meta, block: int, policy: str, k_budget: int, q_frac: float,
                        softmax_scale: float = 0.0, out: dict | None = None, O: torch.Tensor | None = None,
                        want_lse: bool = False):
    """bsa_select + bsa_sparse_attn_fwd in one call (the attention kernel as a programmatic dependent
    launch).  Returns (selection dict as bsa_select, O, lse)."""
    lib = load_library()
    shape = make_shape(Q, K, block)
    B, H, N, _ = Q.shape
    T = N // block
    W = bsa_kv_width(policy, k_budget)
    dev = Q.device
    o = dict(out) if out else {}
    o.setdefault("kv_idx", torch.empty((B, H, T, max(W, 1)), dtype=torch.int32, device=dev))
    o.setdefault("kv_count", torch.empty((B, H, T), dtype=torch.int32, device=dev))
    o.setdefault("sigma", torch.empty((B, H, T), dtype=torch.float32, device=dev))
    o.setdefault("sigma_bar", torch.empty((B, T), dtype=torch.float32, device=dev))
    o.setdefault("trigger", torch.empty((B, T), dtype=torch.uint8, device=dev))
    o.setdefault("tau", torch.empty((B,), dtype=torch.float32, device=dev))
    if O is None:
        O = torch.empty_like(Q)
    lse = torch.empty(Q.shape[:3], dtype=torch.float32, device=dev) if want_lse else None
    _check(lib.bsa_select_attn_fwd(ctypes.byref(shape), _ptr(Q), _ptr(K), _ptr(V), _ptr(meta), POLICIES[policy],
                                   k_budget, float(q_frac), _ptr(o["kv_idx"]), _ptr(o["kv_count"]),
                                   _ptr(o["sigma"]), _ptr(o["sigma_bar"]), _ptr(o["trigger"]), _ptr(o["tau"]),
                                   float(softmax_scale), _ptr(O), _ptr(lse), None, 0, _stream()))
    o["W"] = W
    return o, O, lse


def bsa_dense_attn_fwd(Q, K, V, block: int, softmax_scale: float = 0.0, O: torch.Tensor | None = None,
                       lse: torch.Tensor | None = None, want_lse: bool = False):
    lib = load_library()
    shape = make_shape(Q, K, block)
    assert V.shape == K.shape and V.stride() == K.stride()
    if O is None:
        O = torch.empty_like(Q)
    assert O.stride() == Q.stride()
    if lse is None and want_lse:
        lse = torch.empty(Q.shape[:3], dtype=torch.float32, device=Q.device)
    _check(lib.bsa_dense_attn_fwd(ctypes.byref(shape), _ptr(Q), _ptr(K), _ptr(V), float(softmax_scale),
                                  _ptr(O), _ptr(lse), _stream()))
    return O, lse


# ---- ragged batches: packed Q / O [1, Hq, total, d], K / V [1, Hkv, total, d] + cu_seqlens --------------
def _cu(cu_seqlens):
    arr = (ctypes.c_int32 * len(cu_seqlens))(*[int(x) for x in cu_seqlens])
    return arr, len(cu_seqlens) - 1


def bsa_build_block_meta_varlen(K: torch.Tensor, cu_seqlens, block: int, kinds: int = 3):
    lib = load_library()
    shape = make_shape(None, K, block)
    cu, n = _cu(cu_seqlens)
    nbytes = int(lib.bsa_block_meta_bytes_varlen(ctypes.byref(shape), cu, n, kinds))
    meta = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=K.device)
    _check(lib.bsa_build_block_meta_varlen(ctypes.byref(shape), cu, n, _ptr(K), kinds, _ptr(meta), _stream()))
    return meta


def bsa_select_varlen(Q, meta, K_like, cu_seqlens, block: int, policy: str, k_budget: int, q_frac: float):
    """Sequence-major outputs (include/bsa.h "Ragged batches"): kv_idx flat [Hq * total_T * W],
    kv_count / sigma flat [Hq * total_T], sigma_bar / trigger [total_T], tau [n_seqs]."""
    lib = load_library()
    shape = make_shape(Q, K_like, block)
    cu, n = _cu(cu_seqlens)
    H, total_T = Q.shape[1], Q.shape[2] // block
    W = bsa_kv_width(policy, k_budget)
    dev = Q.device
    o = dict(kv_idx=torch.empty(H * total_T * W, dtype=torch.int32, device=dev),
             kv_count=torch.empty(H * total_T, dtype=torch.int32, device=dev),
             sigma=torch.empty(H * total_T, dtype=torch.float32, device=dev),
             sigma_bar=torch.empty(total_T, dtype=torch.float32, device=dev),
             trigger=torch.empty(total_T, dtype=torch.uint8, device=dev),
             tau=torch.empty(n, dtype=torch.float32, device=dev), W=W)
    _check(lib.bsa_select_varlen(ctypes.byref(shape), cu, n, _ptr(Q), _ptr(meta), POLICIES[policy], k_budget,
                                 float(q_frac), _ptr(o["kv_idx"]), _ptr(o["kv_count"]), _ptr(o["sigma"]),
                                 _ptr(o["sigma_bar"]), _ptr(o["trigger"]), _ptr(o["tau"]), _stream()))
    return o


def bsa_sparse_attn_fwd_varlen(Q, K, V, cu_seqlens, kv_idx, kv_count, kv_width: int, block: int,
                               softmax_scale: float = 0.0, want_lse: bool = False):
    lib = load_library()
    shape = make_shape(Q, K, block)
    cu, n = _cu(cu_seqlens)
    O = torch.empty_like(Q)
    lse = torch.empty(Q.shape[1] * Q.shape[2], dtype=torch.float32, device=Q.device) if want_lse else None
    _check(lib.bsa_sparse_attn_fwd_varlen(ctypes.byref(shape), cu, n, _ptr(Q), _ptr(K), _ptr(V), _ptr(kv_idx),
                                          _ptr(kv_count), kv_width, float(softmax_scale), _ptr(O), _ptr(lse),
                                          _stream()))
    return O, lse


def bsa_dense_attn_fwd_varlen(Q, K, V, cu_seqlens, block: int, softmax_scale: float = 0.0,
                              want_lse: bool = False):
    lib = load_library()
    shape = make_shape(Q, K, block)
    cu, n = _cu(cu_seqlens)
    O = torch.empty_like(Q)
    lse = torch.empty(Q.shape[1] * Q.shape[2], dtype=torch.float32, device=Q.device) if want_lse else None
    _check(lib.bsa_dense_attn_fwd_varlen(ctypes.byref(shape), cu, n, _ptr(Q), _ptr(K), _ptr(V),
                                         float(softmax_scale), _ptr(O), _ptr(lse), _stream()))
    return O, lse


# ---- per-row selection scattered into a per-tile bitmap ----------------------------------
def bsa_select_rows_bitmap(Q, meta, K_like, block: int, policy: str, k_row: int):
    """Returns (bitmap int32-viewed uint32 [B,Hq,T,words], kv_count int32 [B,Hq,T])."""
    lib = load_library()
    shape = make_shape(Q, K_like, block)
    B, H, N, _ = Q.shape
    T = N // block
    words = int(lib.bsa_bitmap_words(ctypes.byref(shape)))
    bitmap = torch.empty((B, H, T, words), dtype=torch.int32, device=Q.device)
    count = torch.empty((B, H, T), dtype=torch.int32, device=Q.device)
    _check(lib.bsa_select_rows_bitmap(ctypes.byref(shape), _ptr(Q), _ptr(meta), POLICIES[policy], k_row,
                                      _ptr(bitmap), _ptr(count), _stream()))
    return bitmap, count


def bsa_sparse_attn_fwd_bitmap(Q, K, V, bitmap, block: int, softmax_scale: float = 0.0,
                               O: torch.Tensor | None = None, want_lse: bool = False):
    lib = load_library()
    shape = make_shape(Q, K, block)
    if O is None:
        O = torch.empty_like(Q)
    lse = torch.empty(Q.shape[:3], dtype=torch.float32, device=Q.device) if want_lse else None
    assert bitmap.dtype == torch.int32 and bitmap.is_contiguous()
    _check(lib.bsa_sparse_attn_fwd_bitmap(ctypes.byref(shape), _ptr(Q), _ptr(K), _ptr(V), _ptr(bitmap),
                                          float(softmax_scale), _ptr(O), _ptr(lse), _stream()))
    return O, lse


def version() -> str:
    return load_library().bsa_version().decode()
