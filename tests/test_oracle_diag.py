"""Pins of the oracle's D.4 diagnostics (oracle.diag_cells / roughness / diag_summary; App. D.4
L486-491, Eq.18): hand-worked examples, closed forms and an independently formulated brute force."""
import math
import os

import numpy as np

import oracle
from paper_2607_07724_b200 import synth

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "diag_examples.txt")


def _f32(x):
    return (np.asarray(x).astype(np.uint32) << np.uint32(16)).view(np.float32)


def _parse():
    cells, summ = [], []
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        p = [x.strip() for x in line.split("|")]
        if p[1] == "summary":
            summ.append(dict(name=p[0], T=int(p[2]), H=int(p[3]), k=int(p[4]), Bn=int(p[5]), tau=float(p[6]),
                             r=np.array(p[7].split(), np.float32), g=np.array(p[8].split(), np.float32),
                             d2=np.array(p[9].split(), np.float32), rough=float(p[10]),
                             want=np.array(p[11].split(), np.float64)))
        else:
            cells.append(dict(name=p[0], t=int(p[1]), nb=int(p[2]), k=int(p[3]),
                              ts=np.array(p[4].split(), np.float32),
                              want=[float(x) for x in p[5:9]]))
    return cells, summ


def test_hand_worked_cells():
    cells, _ = _parse()
    assert len(cells) == 5
    for e in cells:
        _, _, ss = oracle.select_from_scores(e["ts"], e["t"], e["nb"], e["k"])
        d = oracle.diag_cells(ss.reshape(1, 1, -1), [e["t"]], e["k"])
        got = [float(d[n][0, 0]) for n in ("g", "G", "r", "d2")]
        for a, b in zip(got, e["want"]):
            assert (math.isnan(a) and math.isnan(b)) or a == b, (e["name"], got, e["want"])


def test_hand_worked_summary():
    _, summ = _parse()
    assert len(summ) == 1
    e = summ[0]
    T, H, k = e["T"], e["H"], e["k"]
    full = lambda v: np.concatenate([np.full(2 * k, np.nan, np.float32), v]).reshape(T, H)
    rough = np.full((T, H), e["rough"], np.float32)
    s, vec = oracle.diag_summary(full(e["g"]), full(e["r"]), full(e["d2"]), rough, k, e["Bn"], True, e["tau"])
    np.testing.assert_allclose(vec[:12], e["want"], rtol=2e-7, atol=0)
    # non-router policy: the router's threshold, gamma_q and the band mass are undefined
    s2, _ = oracle.diag_summary(full(e["g"]), full(e["r"]), full(e["d2"]), rough, k, e["Bn"], False, -1.0)
    assert math.isnan(s2["sigma_q"]) and math.isnan(s2["gamma_q"]) and math.isnan(s2["band_mass"])
    assert s2["r_bar"] == s["r_bar"] and s2["d2_q50"] == s["d2_q50"]


def _row_scores(Q, meta, cfg, policy, t, h):
    """Independent formulation in numpy fp64: [Bn rows, t+1 blocks]."""
    kmean, kmin, kmax = meta
    g = h // cfg.group
    q = _f32(Q[h, t * cfg.block:(t + 1) * cfg.block]).astype(np.float64)
    if policy in ("quest", "router_quest"):
        qp, qn = np.maximum(q, 0), np.minimum(q, 0)
        s = qp @ _f32(kmax[g, :t + 1]).astype(np.float64).T + qn @ _f32(kmin[g, :t + 1]).astype(np.float64).T
        return s.astype(np.float32)
    s = (q @ kmean[g, :t + 1].astype(np.float64).T).astype(np.float32)
    return s * np.float32(1.0 / math.sqrt(cfg.head_dim))


def test_roughness_brute_force_and_invariants():
    cfg = synth.CONFIGS["C1"].scaled(64 * 12, "C1r")
    inp = synth.make_inputs(cfg)
    meta = oracle.pool(inp.K, cfg.block)
    tiles = [0, 1, 5, 11]
    for policy in ("router", "router_quest"):
        got = oracle.roughness(inp.Q, meta, cfg.block, policy, tiles)
        for i, t in enumerate(tiles):
            for h in range(cfg.n_q_heads):
                s = _row_scores(inp.Q, meta, cfg, policy, t, h).astype(np.float64)
                want = float((np.diff(s, axis=0) ** 2).sum())
                assert abs(got[i, h] - want) <= 1e-6 * want + 1e-30, (policy, t, h)
    # identical rows inside every tile: no roughness at all
    Qc = inp.Q.copy()
    Qc[:] = Qc[:, ::cfg.block].repeat(cfg.block, axis=1)
    assert (oracle.roughness(Qc, meta, cfg.block, "router", tiles) == 0).all()
    assert (oracle.roughness(Qc, meta, cfg.block, "router_quest", tiles) == 0).all()
    # rows alternating +q, -q (K-mean backbone): every adjacent pair differs by 2 s_b, so
    # rough = 4 (Bn - 1) sum_b s_b^2   -- closed form
    Qa = Qc.copy()
    Qa[:, 1::2] ^= np.uint16(0x8000)
    got = oracle.roughness(Qa, meta, cfg.block, "router", tiles)
    for i, t in enumerate(tiles):
        for h in range(cfg.n_q_heads):
            s = _row_scores(Qc, meta, cfg, "router", t, h)[0].astype(np.float64)
            want = 4.0 * (cfg.block - 1) * float((s ** 2).sum())
            assert abs(got[i, h] - want) <= 1e-6 * want


def test_cells_invariants_on_real_scores():
    """sigma = g / r (Eq.18), G >= g >= 0 (L422), d2 >= 0, NaN exactly on tiles with < rho k + 1 blocks."""
    cfg = synth.CONFIGS["C1"]
    inp = synth.make_inputs(cfg)
    meta = oracle.pool(inp.K, cfg.block)
    k = cfg.k_budget
    for policy in ("topk", "quest"):
        d = oracle.diag(inp.Q, meta, cfg.block, policy, k, 0.25)
        sel = oracle.select_tiles(inp.Q, meta, cfg.block, policy, k, np.arange(cfg.n_blocks))
        valid = np.arange(cfg.n_blocks) >= 2 * k
        assert np.isnan(d["g"][~valid]).all() and np.isfinite(d["g"][valid]).all()
        g, G, r = d["g"][valid], d["G"][valid], d["r"][valid]
        assert (g >= 0).all() and (G >= g).all() and (r >= g).all() and (d["d2"][valid] >= 0).all()
        sig = np.where(r == 0, np.float32(0), g / np.where(r == 0, 1, r)).astype(np.float32)
        assert np.array_equal(sig, sel["sigma"][valid])
        s = d["summary"]
        assert s["n"] == cfg.n_q_heads * (cfg.n_blocks - 2 * k)
        np.testing.assert_allclose(s["r_bar"], r.astype(np.float64).mean(), rtol=1e-6)
        np.testing.assert_allclose(s["cv_r"], r.astype(np.float64).std() / r.astype(np.float64).mean(), rtol=1e-5)
        assert math.isnan(s["band_mass"])          # non-router policy
    d = oracle.diag(inp.Q, meta, cfg.block, "router", k, 0.25)
    assert 0.0 <= d["summary"]["band_mass"] <= 1.0 and d["summary"]["sigma_q"] == np.float32(d["tau"])
