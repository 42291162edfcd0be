"""ctypes wrapper around the CPU oracle (oracle/bsa_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package never imports this module and this
module never imports the product's CUDA binding.

All tensors are numpy arrays; bf16 tensors are uint16 bit patterns [heads, N, d].
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bsa_oracle.c")
_LIB = os.path.join(_HERE, "libbsa_oracle.so")
_lib = None

POLICIES = {"topk": 0, "router": 1, "quest": 2, "router_quest": 3}
RHO = 2


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        # -ffp-contract=off: no fused multiply-adds, the oracle rounds exactly where the C text says.
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99",
                               "-ffp-contract=off", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        i64, vp, dbl, ci = ctypes.c_int64, ctypes.c_void_p, ctypes.c_double, ctypes.c_int
        lib.orc_pool.argtypes = [vp, i64, i64, i64, i64, vp, vp, vp]
        lib.orc_pool.restype = None
        lib.orc_select_tiles.argtypes = [vp, vp, vp, vp, i64, i64, i64, i64, i64, ci, i64, vp, i64,
                                         vp, vp, vp, vp]
        lib.orc_select_tiles.restype = None
        lib.orc_select_from_scores.argtypes = [vp, i64, i64, i64, vp, vp]
        lib.orc_select_from_scores.restype = ctypes.c_float
        lib.orc_route.argtypes = [vp, i64, i64, ci, dbl, vp, vp, vp]
        lib.orc_route.restype = None
        lib.orc_fill.argtypes = [vp, vp, i64, i64, i64, i64, i64, vp, vp]
        lib.orc_fill.restype = None
        lib.orc_attn_pairs.argtypes = [vp, vp, vp, i64, i64, i64, i64, i64, vp, vp, i64, ci, dbl,
                                       vp, i64, vp, vp]
        lib.orc_attn_pairs.restype = None
        lib.orc_diag_cells.argtypes = [vp, vp, i64, i64, i64, vp, vp, vp, vp]
        lib.orc_diag_cells.restype = None
        lib.orc_roughness.argtypes = [vp, vp, vp, vp, i64, i64, i64, i64, i64, ci, vp, i64, vp]
        lib.orc_roughness.restype = None
        lib.orc_diag_summary.argtypes = [vp, vp, vp, vp, i64, i64, i64, i64, ci, ctypes.c_float, vp]
        lib.orc_diag_summary.restype = None
        lib.orc_select_rows_bitmap.argtypes = [vp, vp, vp, vp, i64, i64, i64, i64, i64, ci, i64, vp, i64, vp, vp]
        lib.orc_select_rows_bitmap.restype = None
        lib.orc_max_threads.restype = ci
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().orc_max_threads())


def _p(a):
    return None if a is None else a.ctypes.data


def _c(a, dt):
    a = np.ascontiguousarray(a, dtype=dt)
    return a


def kv_width(policy: str, k: int) -> int:
    return RHO * k if policy in ("router", "router_quest") else k


def pool(K: np.ndarray, block: int):
    """O1/O2: returns (kmean fp32, kmin bf16 bits, kmax bf16 bits), each [Hkv, N_B, d]."""
    K = _c(K, np.uint16)
    Hkv, N, d = K.shape
    NB = N // block
    kmean = np.empty((Hkv, NB, d), np.float32)
    kmin = np.empty((Hkv, NB, d), np.uint16)
    kmax = np.empty((Hkv, NB, d), np.uint16)
    _load().orc_pool(_p(K), Hkv, N, d, block, _p(kmean), _p(kmin), _p(kmax))
    return kmean, kmin, kmax


def select_tiles(Q, meta, block: int, policy: str, k: int, tiles, want_scores: bool = False):
    """O3-O7 for the listed tiles.  Returns dict(idx_sorted [n,H,2k], score_sorted [n,H,2k+1],
    sigma [n,H], tile_score [n,H,N_B] or None)."""
    Q = _c(Q, np.uint16)
    kmean, kmin, kmax = meta
    H, N, d = Q.shape
    Hkv = kmean.shape[0]
    NB = N // block
    tiles = _c(np.asarray(tiles), np.int64)
    n = len(tiles)
    W2 = RHO * k
    idx_sorted = np.empty((n, H, W2), np.int32)
    score_sorted = np.empty((n, H, W2 + 1), np.float32)
    sigma = np.empty((n, H), np.float32)
    tile_score = np.empty((n, H, NB), np.float32) if want_scores else None
    _load().orc_select_tiles(_p(Q), _p(_c(kmean, np.float32)), _p(_c(kmin, np.uint16)),
                             _p(_c(kmax, np.uint16)), H, Hkv, N, d, block, POLICIES[policy], k,
                             _p(tiles), n, _p(idx_sorted), _p(score_sorted), _p(sigma), _p(tile_score))
    return dict(idx_sorted=idx_sorted, score_sorted=score_sorted, sigma=sigma, tile_score=tile_score)


def select_from_scores(ts, t: int, n_blocks: int, k: int):
    """O5-O7 on caller-provided tile scores ts[0..t] (hand-worked examples)."""
    ts = _c(ts, np.float32)
    assert len(ts) >= t + 1
    W2 = RHO * k
    idx_sorted = np.empty(W2, np.int32)
    score_sorted = np.empty(W2 + 1, np.float32)
    sig = _load().orc_select_from_scores(_p(ts), t, n_blocks, k, _p(idx_sorted), _p(score_sorted))
    return float(np.float32(sig)), idx_sorted, score_sorted


def route(sigma_th: np.ndarray, policy: str, q_frac: float):
    """O8/O9 on sigma laid out [T, H].  Returns (sigma_bar [T], tau, trigger uint8 [T])."""
    sigma_th = _c(sigma_th, np.float32)
    T, H = sigma_th.shape
    sigma_bar = np.empty(T, np.float32)
    tau = np.empty(1, np.float32)
    trigger = np.empty(T, np.uint8)
    _load().orc_route(_p(sigma_th), T, H, POLICIES[policy], float(q_frac), _p(sigma_bar), _p(tau),
                      _p(trigger))
    return sigma_bar, float(tau[0]), trigger


def fill(idx_sorted_th: np.ndarray, trigger: np.ndarray, n_blocks: int, k: int, W: int):
    """O10 on idx_sorted [T, H, 2k].  Returns (kv_idx [H,T,W], kv_count [H,T])."""
    idx_sorted_th = _c(idx_sorted_th, np.int32)
    T, H, W2 = idx_sorted_th.shape
    assert W2 == RHO * k
    kv_idx = np.empty((H, T, W), np.int32)
    kv_count = np.empty((H, T), np.int32)
    _load().orc_fill(_p(idx_sorted_th), _p(_c(trigger, np.uint8)), T, H, n_blocks, k, W,
                     _p(kv_idx), _p(kv_count))
    return kv_idx, kv_count


def select(Q, meta, block: int, policy: str, k: int, q_frac: float, want_scores: bool = False):
    """Full selection O3-O10 of one sequence.  Returns a dict with kv_idx [H,T,W], kv_count [H,T],
    sigma [H,T], sigma_bar [T], trigger [T], tau, idx_sorted [T,H,2k], score_sorted [T,H,2k+1]."""
    H, N, d = Q.shape
    T = N // block
    r = select_tiles(Q, meta, block, policy, k, np.arange(T), want_scores)
    sigma_bar, tau, trigger = route(r["sigma"], policy, q_frac)
    W = kv_width(policy, k)
    kv_idx, kv_count = fill(r["idx_sorted"], trigger, T, k, W)
    return dict(kv_idx=kv_idx, kv_count=kv_count, sigma=np.ascontiguousarray(r["sigma"].T),
                sigma_bar=sigma_bar, trigger=trigger, tau=tau, idx_sorted=r["idx_sorted"],
                score_sorted=r["score_sorted"], tile_score=r["tile_score"], W=W)


def attn_pairs(Q, K, V, block: int, pairs, kv_idx=None, kv_count=None, scale: float | None = None,
               want_lse: bool = True):
    """O11 (kv_idx given) / O12 (kv_idx None = dense) for the listed (t, h) pairs.
    Returns (O [n_pairs, block, d] fp32, lse [n_pairs, block] fp32)."""
    Q, K, V = _c(Q, np.uint16), _c(K, np.uint16), _c(V, np.uint16)
    H, N, d = Q.shape
    Hkv = K.shape[0]
    pairs = _c(np.asarray(pairs).reshape(-1, 2), np.int64)
    n = len(pairs)
    O = np.empty((n, block, d), np.float32)
    lse = np.empty((n, block), np.float32) if want_lse else None
    if scale is None:
        scale = 1.0 / math.sqrt(d)
    dense = kv_idx is None
    W = 0
    if not dense:
        kv_idx = _c(kv_idx, np.int32)
        W = kv_idx.shape[-1]
        if kv_count is not None:
            kv_count = _c(kv_count, np.int32)
    _load().orc_attn_pairs(_p(Q), _p(K), _p(V), H, Hkv, N, d, block, _p(kv_idx), _p(kv_count), W,
                           1 if dense else 0, float(scale), _p(pairs), n, _p(O), _p(lse))
    return O, lse


def attn_full(Q, K, V, block: int, kv_idx=None, kv_count=None, scale=None):
    """All (t, h) pairs; returns O [H, N, d] fp32 and lse [H, N]."""
    H, N, d = Q.shape
    T = N // block
    pairs = np.array([(t, h) for h in range(H) for t in range(T)], np.int64)
    O, lse = attn_pairs(Q, K, V, block, pairs, kv_idx, kv_count, scale)
    return O.reshape(H, N, d), lse.reshape(H, N)


# ---- D.4 diagnostics (Eq.18) ------------------------------------------------------
DIAG_SUMMARY = ("n", "r_bar", "cv_r", "sigma_q", "gamma_q", "band_mass", "d2_q10", "d2_q50", "tau_hat",
                "zero_gap_frac", "g_q40_pos", "g_q40_pos_over_tau_hat")


def diag_cells(score_sorted: np.ndarray, tiles, k: int):
    """Per-cell g, G, r, d2 (each [n_tiles, H]) from select_tiles()['score_sorted'] [n, H, 2k+1]."""
    ss = _c(score_sorted, np.float32)
    n, H, w = ss.shape
    assert w == RHO * k + 1
    tiles = _c(np.asarray(tiles), np.int64)
    out = [np.empty((n, H), np.float32) for _ in range(4)]
    _load().orc_diag_cells(_p(ss), _p(tiles), n, H, k, *[_p(a) for a in out])
    return dict(g=out[0], G=out[1], r=out[2], d2=out[3])


def roughness(Q, meta, block: int, policy: str, tiles):
    """rough [n_tiles, H]: sum over visible blocks and adjacent rows of (s[i+1,b] - s[i,b])^2."""
    Q = _c(Q, np.uint16)
    kmean, kmin, kmax = meta
    H, N, d = Q.shape
    tiles = _c(np.asarray(tiles), np.int64)
    out = np.empty((len(tiles), H), np.float32)
    _load().orc_roughness(_p(Q), _p(_c(kmean, np.float32)), _p(_c(kmin, np.uint16)), _p(_c(kmax, np.uint16)),
                          H, kmean.shape[0], N, d, block, POLICIES[policy], _p(tiles), len(tiles), _p(out))
    return out


def diag_summary(g, r, d2, rough, k: int, block: int, router: bool, tau: float):
    """Per-layer aggregates (dict keyed by DIAG_SUMMARY) from per-cell arrays laid out [T, H]."""
    g, r, d2, rough = (_c(a, np.float32) for a in (g, r, d2, rough))
    T, H = g.shape
    out = np.empty(16, np.float32)
    _load().orc_diag_summary(_p(g), _p(r), _p(d2), _p(rough), T, H, k, block, 1 if router else 0,
                             float(tau), _p(out))
    return {name: float(out[i]) for i, name in enumerate(DIAG_SUMMARY)}, out


def diag(Q, meta, block: int, policy: str, k: int, q_frac: float):
    """Full D.4 pass of one sequence: cells [T, H], rough [T, H], summary."""
    H, N, d = Q.shape
    T = N // block
    tiles = np.arange(T)
    sel = select_tiles(Q, meta, block, policy, k, tiles)
    cells = diag_cells(sel["score_sorted"], tiles, k)
    rough = roughness(Q, meta, block, policy, tiles)
    _, tau, _ = route(sel["sigma"], policy, q_frac)
    router = policy in ("router", "router_quest") and tau >= 0
    summ, vec = diag_summary(cells["g"], cells["r"], cells["d2"], rough, k, block, router, tau)
    return dict(cells, rough=rough, summary=summ, summary_vec=vec, tau=tau)


# ---- per-row selection scattered into a per-tile bitmap --------------------------------
def select_rows_bitmap(Q, meta, block: int, policy: str, k_row: int, tiles=None):
    """Returns (bitmap uint32 [n_tiles, H, ceil(N_B/32)], count int32 [n_tiles, H])."""
    Q = _c(Q, np.uint16)
    kmean, kmin, kmax = meta
    H, N, d = Q.shape
    NB = N // block
    tiles = _c(np.arange(NB) if tiles is None else np.asarray(tiles), np.int64)
    n = len(tiles)
    bitmap = np.empty((n, H, (NB + 31) // 32), np.uint32)
    count = np.empty((n, H), np.int32)
    _load().orc_select_rows_bitmap(_p(Q), _p(_c(kmean, np.float32)), _p(_c(kmin, np.uint16)),
                                   _p(_c(kmax, np.uint16)), H, kmean.shape[0], N, d, block, POLICIES[policy],
                                   k_row, _p(tiles), n, _p(bitmap), _p(count))
    return bitmap, count


def bitmap_to_kv_idx(bitmap, n_blocks: int):
    """[n, H, NBW] -> (kv_idx [H, n, width] ascending block lists padded with n_blocks, kv_count [H, n])."""
    n, H, _ = bitmap.shape
    bits = np.unpackbits(bitmap.view(np.uint8), axis=-1, bitorder="little")[..., :n_blocks]
    cnt = bits.sum(-1).astype(np.int32)
    W = int(cnt.max()) if cnt.size else 1
    kv = np.full((H, n, max(W, 1)), n_blocks, np.int32)
    for i in range(n):
        for h in range(H):
            idx = np.nonzero(bits[i, h])[0]
            kv[h, i, :len(idx)] = idx
    return kv, np.ascontiguousarray(cnt.T)
