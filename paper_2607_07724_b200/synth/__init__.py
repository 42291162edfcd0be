"""Seeded synthetic inputs for the selection + sparse-attention prefill path.

Holds none of the method's arithmetic: only the counter-based Gaussian generator
(`synth.c`), the needle planting and the QK-Norm pre-processing of the input
recipe (shapes from PAPER.md L141-144,
block size L70/L90).  Used by the oracle's tests, the CUDA parity tests and
bench.py so every side sees identical bf16 bit patterns.

bf16 tensors are numpy ``uint16`` arrays of shape ``[heads, N, d]``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "synth.c")
_LIB = os.path.join(_HERE, "libbsa_synth.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile synth.c into libbsa_synth.so (gcc, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-ffp-contract=off",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        u64, i64, dbl, vp = ctypes.c_uint64, ctypes.c_int64, ctypes.c_double, ctypes.c_void_p
        lib.synth_u64.argtypes = [u64, u64, u64, u64, vp]
        lib.synth_gauss_f64.argtypes = [u64, u64, u64, u64, vp]
        lib.synth_gauss_bf16.argtypes = [u64, u64, u64, dbl, i64, i64, i64, i64, vp]
        lib.synth_rmsnorm_rows_bf16.argtypes = [vp, i64, i64, ctypes.c_float]
        for f in (lib.synth_u64, lib.synth_gauss_f64, lib.synth_gauss_bf16, lib.synth_rmsnorm_rows_bf16):
            f.restype = None
        _lib = lib
    return _lib


# tensor ids of the recipe
TID_Q, TID_K, TID_V, TID_KOFF, TID_QOFF, TID_NDIR, TID_NPOS = 1, 2, 3, 4, 5, 6, 7


def bf16_to_f32(x: np.ndarray) -> np.ndarray:
    return (x.astype(np.uint32) << np.uint32(16)).view(np.float32)


def f32_to_bf16(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16 bit patterns (finite inputs)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    u = u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))
    return (u >> np.uint32(16)).astype(np.uint16)


def u64(seed: int, tensor_id: int, start: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.uint64)
    _load().synth_u64(seed, tensor_id, start, n, out.ctypes.data)
    return out


def gauss_f64(seed: int, tensor_id: int, start: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.float64)
    _load().synth_gauss_f64(seed, tensor_id, start, n, out.ctypes.data)
    return out


def gauss_bf16(seed, tensor_id, heads, rows, d, block, off_tensor_id=0, off_scale=0.0) -> np.ndarray:
    out = np.empty((heads, rows, d), dtype=np.uint16)
    _load().synth_gauss_bf16(seed, tensor_id, off_tensor_id, float(off_scale), heads, rows, d, block,
                             out.ctypes.data)
    return out


def rmsnorm_rows_(x: np.ndarray, eps: float = 1e-6) -> None:
    assert x.dtype == np.uint16 and x.flags.c_contiguous
    d = x.shape[-1]
    _load().synth_rmsnorm_rows_bf16(x.ctypes.data, x.size // d, d, eps)


@dataclass(frozen=True)
class Config:
    """One workload of BASELINE.json `configs` (ids as in SURVEY.md 8: C1, C2, C3a, C3b, C4, C5)."""
    name: str
    number: int                 # seed = 7724*100 + number
    seqlen: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    block: int
    k_budget: int
    q_fracs: tuple = (0.25,)
    policies: tuple = ("topk", "router")
    structured: bool = False    # per-block mean offsets (std 0.5) on Q and K
    needles: str = "none"       # "none" | "single16" | "chain8"
    qk_norm: bool = False

    @property
    def seed(self) -> int:
        return 7724 * 100 + self.number

    @property
    def n_blocks(self) -> int:
        return self.seqlen // self.block

    @property
    def group(self) -> int:
        return self.n_q_heads // self.n_kv_heads

    def scaled(self, seqlen: int, name: str | None = None) -> "Config":
        """Same recipe at another sequence length (used by the small parity cases)."""
        from dataclasses import replace
        return replace(self, seqlen=seqlen, name=name or f"{self.name}@{seqlen}")


CONFIGS = {
    "C1": Config("C1", 1, 2048, 4, 2, 64, 64, 4, (0.25,), ("topk", "router")),
    "C2": Config("C2", 2, 32768, 28, 4, 128, 64, 32, (0.25,),
                 ("topk", "router", "quest", "router_quest"), True, "single16"),
    "C3a": Config("C3a", 3, 65536, 28, 4, 128, 64, 32, (0.25,),
                  ("router_quest", "topk"), True, "single16"),
    "C3b": Config("C3b", 3, 131072, 28, 4, 128, 64, 32, (0.25,),
                  ("router_quest", "topk"), True, "single16"),
    # 256K: the regime PAPER.md L271 names for selection fused into the attention kernel
    "C3c": Config("C3c", 3, 262144, 28, 4, 128, 64, 32, (0.25,),
                  ("router_quest", "topk"), True, "single16"),
    "C4": Config("C4", 4, 65536, 32, 8, 128, 64, 64, (0.1, 0.25, 0.5),
                 ("quest", "router_quest"), True, "single16"),
    "C5": Config("C5", 5, 131072, 16, 2, 256, 128, 16, (0.25,),
                 ("router", "router_quest"), False, "chain8", True),
}

NEEDLE_ALPHA = 3.0   # norm ratio of a planted key to its query (BASELINE.json fixes only cos 0.8)
NEEDLE_COS = 0.8


@dataclass
class Inputs:
    cfg: Config
    Q: np.ndarray               # uint16 [H, N, d]
    K: np.ndarray               # uint16 [Hkv, N, d]
    V: np.ndarray               # uint16 [Hkv, N, d]
    needles: list = field(default_factory=list)   # dicts: head, q_row, kv_head, key_row


def _aligned_key(q_row_bits: np.ndarray, dir_draw: np.ndarray) -> np.ndarray:
    """bf16( alpha*|q| * (0.8 q^ + 0.6 u^) ), u^ a unit vector orthogonal to q^ (double arithmetic)."""
    q = bf16_to_f32(q_row_bits).astype(np.float64)
    nq = np.linalg.norm(q)
    qh = q / nq
    u = dir_draw - np.dot(dir_draw, qh) * qh
    u /= np.linalg.norm(u)
    s = np.sqrt(1.0 - NEEDLE_COS ** 2)
    return f32_to_bf16((NEEDLE_ALPHA * nq * (NEEDLE_COS * qh + s * u)).astype(np.float32))


def _plant_single(cfg: Config, Q, K, n_needles=16):
    """16 single needles (SURVEY.md 8(d) 'Needles'): a key aligned (cos 0.8) to a late query row."""
    N, Bn, d, G = cfg.seqlen, cfg.block, cfg.head_dim, cfg.group
    draws = u64(cfg.seed, TID_NPOS, 0, 64 * n_needles)
    out, used, p = [], set(), 0
    if N // Bn < 8:          # too short to host a needle strictly between sink and self
        return out
    while len(out) < n_needles and p + 4 <= len(draws):
        h = int(draws[p] % np.uint64(cfg.n_q_heads))
        i = N // 2 + int(draws[p + 1] % np.uint64(N - N // 2))
        t = i // Bn
        b = 1 + int(draws[p + 2] % np.uint64(max(t - 1, 1)))      # in [1, t-1]
        o = int(draws[p + 3] % np.uint64(Bn))
        p += 4
        g = h // G
        if b >= t or (g, b) in used:
            continue
        used.add((g, b))
        n = len(out)
        dirv = gauss_f64(cfg.seed, TID_NDIR, n * d, d)
        K[g, Bn * b + o, :] = _aligned_key(Q[h, i, :], dirv)
        out.append(dict(head=h, q_row=i, kv_head=g, key_row=Bn * b + o))
    return out


def _plant_chain(cfg: Config, Q, K, n_pairs=8):
    """8 chained needle pairs (depth-2 pointer chase in the spirit of PAPER.md L356-358)."""
    N, d, G = cfg.seqlen, cfg.head_dim, cfg.group
    draws = u64(cfg.seed, TID_NPOS, 0, 4 * n_pairs)
    out = []
    if N < 1024:
        return out
    for n in range(n_pairs):
        h = int(draws[4 * n] % np.uint64(cfg.n_q_heads))
        i = 3 * N // 4 + int(draws[4 * n + 1] % np.uint64(N - 3 * N // 4))
        j1 = N // 4 + int(draws[4 * n + 2] % np.uint64(N // 2 - N // 4))
        j2 = 128 + int(draws[4 * n + 3] % np.uint64(N // 4 - 128))
        g = h // G
        K[g, j1, :] = _aligned_key(Q[h, i, :], gauss_f64(cfg.seed, TID_NDIR, (2 * n) * d, d))
        K[g, j2, :] = _aligned_key(Q[h, j1, :], gauss_f64(cfg.seed, TID_NDIR, (2 * n + 1) * d, d))
        out.append(dict(head=h, q_row=i, kv_head=g, key_row=j1))
        out.append(dict(head=h, q_row=j1, kv_head=g, key_row=j2))
    return out


def make_inputs(cfg: Config) -> Inputs:
    """Generate Q, K, V for `cfg` (deterministic in cfg.seed and the shape)."""
    N, d, Bn = cfg.seqlen, cfg.head_dim, cfg.block
    assert N % Bn == 0 and cfg.n_q_heads % cfg.n_kv_heads == 0
    if cfg.structured:
        Q = gauss_bf16(cfg.seed, TID_Q, cfg.n_q_heads, N, d, Bn, TID_QOFF, 0.5)
        K = gauss_bf16(cfg.seed, TID_K, cfg.n_kv_heads, N, d, Bn, TID_KOFF, 0.5)
    else:
        Q = gauss_bf16(cfg.seed, TID_Q, cfg.n_q_heads, N, d, Bn)
        K = gauss_bf16(cfg.seed, TID_K, cfg.n_kv_heads, N, d, Bn)
    V = gauss_bf16(cfg.seed, TID_V, cfg.n_kv_heads, N, d, Bn)
    if cfg.needles == "single16":
        needles = _plant_single(cfg, Q, K)
    elif cfg.needles == "chain8":
        needles = _plant_chain(cfg, Q, K)
    else:
        needles = []
    if cfg.qk_norm:
        rmsnorm_rows_(Q)
        rmsnorm_rows_(K)
    return Inputs(cfg, Q, K, V, needles)
