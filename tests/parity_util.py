"""Helpers for the GPU-vs-oracle parity tests: tensor conversion and the comparison protocol of
DESIGN.md "Parity protocol" (bit-exact kv_idx / routing; near-ties inside the 1e-5 relative band are
logged and resolved by set comparison; attention within max-abs 2e-2 / mean-abs 2e-3)."""
from __future__ import annotations

import numpy as np

TIE_REL = 1e-5          # north_star: fp32 block scores closer than this (relative) may swap
SIGMA_TOL = 1e-4        # sigma divides two small score differences
SIGMA_BAR_BAND = 2e-4   # |sigma_bar - tau| below which a trigger may flip: both sides are means of
                        # sigmas that are each within SIGMA_TOL (logged, counted, never hidden)
ATTN_MAX_ABS = 2e-2
ATTN_MEAN_ABS = 2e-3


def to_torch_bf16(bits: np.ndarray, device="cuda"):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16)
    return t.to(device)


def bf16_bits(t) -> np.ndarray:
    import torch
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


def bf16_to_f32(bits: np.ndarray) -> np.ndarray:
    return (bits.astype(np.uint32) << np.uint32(16)).view(np.float32)


def compare_select(gpu: dict, orc: dict, n_blocks: int, k: int, log: list | None = None):
    """gpu: numpy arrays kv_idx [H,T,W], kv_count [H,T], sigma [H,T], sigma_bar [T], trigger [T], tau.
    orc: oracle.select(..., want_scores=True) result.  Returns a dict of counters; raises on a
    mismatch outside the tie bands."""
    log = log if log is not None else []
    H, T, W = orc["kv_idx"].shape
    ts = orc["tile_score"]                      # [T, H, NB]
    stats = dict(rows=H * T, tie_rows=0, trigger_flips=0)

    # ---- routing ----
    tau = orc["tau"]
    flip = np.nonzero(gpu["trigger"].astype(np.uint8) != orc["trigger"].astype(np.uint8))[0]
    for t in flip:
        gap = abs(float(orc["sigma_bar"][t]) - tau)
        assert gap <= SIGMA_BAR_BAND, f"trigger differs at tile {t}: sigma_bar-tau gap {gap:g}"
        log.append(("trigger", int(t), gap))
    stats["trigger_flips"] = len(flip)
    flipped = np.zeros(T, bool)
    flipped[flip] = True
    assert len(flip) <= max(2, T // 100), f"{len(flip)} trigger flips"
    assert abs(float(gpu["tau"]) - tau) <= SIGMA_TOL, "tau"
    np.testing.assert_allclose(gpu["sigma_bar"], orc["sigma_bar"], rtol=0, atol=SIGMA_TOL)

    # ---- kv_count: exact wherever the trigger agrees ----
    ok_t = ~flipped
    assert np.array_equal(gpu["kv_count"][:, ok_t], orc["kv_count"][:, ok_t]), "kv_count mismatch"

    # ---- kv_idx ----
    same = (gpu["kv_idx"] == orc["kv_idx"]).all(axis=2)          # [H, T]
    sig_bad = np.abs(gpu["sigma"] - orc["sigma"]) > SIGMA_TOL
    for h, t in zip(*np.nonzero(~same)):
        if flipped[t]:
            continue
        cnt = int(orc["kv_count"][h, t])
        g_row, o_row = gpu["kv_idx"][h, t], orc["kv_idx"][h, t]
        assert (g_row[cnt:] == n_blocks).all(), f"padding not sentinel at h={h} t={t}"
        assert g_row[0] == 0 and (t == 0 or g_row[1] == t), f"forced blocks missing at h={h} t={t}"
        gs, os_ = set(g_row[:cnt].tolist()), set(o_row[:cnt].tolist())
        assert len(gs) == cnt and all(0 <= b <= t for b in gs), f"invalid blocks at h={h} t={t}"
        sc = ts[t, h]
        # every position where the rows differ must be a near-tie between the two blocks placed there
        for gb, ob in zip(g_row[:cnt], o_row[:cnt]):
            if gb != ob:
                a, b = float(sc[gb]), float(sc[ob])
                assert abs(a - b) <= TIE_REL * max(abs(a), abs(b)), \
                    f"kv_idx differs outside the tie band at h={h} t={t}: blocks {gb},{ob} scores {a},{b}"
        # set difference (cutoff swaps) must be near-ties with the boundary score
        for blk in gs ^ os_:
            bnd = float(sc[o_row[cnt - 1]])
            a = float(sc[blk])
            assert abs(a - bnd) <= TIE_REL * max(abs(a), abs(bnd)), \
                f"selected set differs outside the tie band at h={h} t={t}: block {blk}"
        stats["tie_rows"] += 1
        log.append(("kv_idx", int(h), int(t)))
    # sigma: 1e-4 absolute, except rows whose cutoff is itself inside the tie band
    for h, t in zip(*np.nonzero(sig_bad)):
        ss = orc["score_sorted"][t, h]
        f = 1 if t == 0 else 2
        den = float(ss[f]) - float(ss[k])
        scale = max(abs(float(ss[f])), abs(float(ss[k])))
        assert den <= 100 * TIE_REL * scale, \
            f"sigma differs at h={h} t={t}: {gpu['sigma'][h, t]} vs {orc['sigma'][h, t]} (den {den:g})"
        log.append(("sigma", int(h), int(t)))
    return stats


def compare_attn(O_gpu_f32: np.ndarray, O_ref: np.ndarray, what: str = ""):
    diff = np.abs(O_gpu_f32.astype(np.float64) - O_ref.astype(np.float64))
    mx, mean = float(diff.max()), float(diff.mean())
    assert np.isfinite(O_gpu_f32).all(), f"{what}: non-finite output"
    assert mx <= ATTN_MAX_ABS, f"{what}: max-abs {mx:g} > {ATTN_MAX_ABS}"
    assert mean <= ATTN_MEAN_ABS, f"{what}: mean-abs {mean:g} > {ATTN_MEAN_ABS}"
    return mx, mean
