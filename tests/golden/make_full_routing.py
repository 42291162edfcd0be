#!/usr/bin/env python
"""Writes tests/golden/routing_<case>.json: the ORACLE's full-sequence routing of the large
BASELINE.json configs (C3a, C3b, C4, C5, and C3c = 256K), i.e. what needs every tile of the sequence and
therefore cannot be checked on a sample:

    sigma_bar[T]  (Eq.12)   -- fp32 bit patterns, hex
    amp_bar[T]    mean over heads of scale / (s~[f] - s~[k]), the factor by which sigma amplifies a
                  relative score error (tests/parity_util.py: sigma_amp) -- fp32, hex
    per q_frac:   m = ceil(qT - 1e-9), tau (Eq.5 / Eq.13) and trigger[T] (bit string)

Calls only `oracle/` and the seeded input generator (no CUDA code, no GPU).  The GPU parity test
`tests/test_gpu_parity.py::test_full_size_sampled` compares bsa_select's sigma_bar / tau / trigger with
these values instead of with the GPU's own sigma_bar.

    python tests/golden/make_full_routing.py            # every case (about 1e12 MAC each: minutes)
    python tests/golden/make_full_routing.py C3b/router_quest C5/router

Cost on the 8-core build box: C3a 40 s, C3b 3-5 min per backbone, C4 1 min, C5 1-3 min, C3c 15 min.
"""
from __future__ import annotations

import json
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

import oracle
from paper_2607_07724_b200 import synth

# (config, policy) -> q fractions.  Non-router policies store sigma_bar only.
CASES = {
    "C3a/router_quest": (0.25,),
    "C3b/router_quest": (0.25, 0.4),
    "C3b/topk": (),
    "C4/router_quest": (0.1, 0.25, 0.5),
    "C5/router": (0.25,),
    "C5/router_quest": (0.25,),
    "C3c/router_quest": (0.25,),
}


def path_of(case: str) -> str:
    return os.path.join(HERE, "routing_" + case.replace("/", "_") + ".json")


def make(case: str) -> dict:
    name, policy = case.split("/")
    cfg = synth.CONFIGS[name]
    inp = synth.make_inputs(cfg)
    t0 = time.time()
    meta = oracle.pool(inp.K, cfg.block)
    T = cfg.n_blocks
    r = oracle.select_tiles(inp.Q, meta, cfg.block, policy, cfg.k_budget, np.arange(T))
    sigma = r["sigma"]                                   # [T, H]
    out = {
        "case": case, "config": name, "policy": policy, "seed": cfg.seed, "seqlen": cfg.seqlen,
        "n_q_heads": cfg.n_q_heads, "n_kv_heads": cfg.n_kv_heads, "head_dim": cfg.head_dim,
        "block": cfg.block, "k_budget": cfg.k_budget, "T": T,
        "written_by": "tests/golden/make_full_routing.py (oracle only)",
        "routes": {},
    }
    sigma_bar, _, _ = oracle.route(sigma, policy, 0.0)
    out["sigma_bar_hex"] = sigma_bar.astype(np.float32).view(np.uint32).tobytes().hex()
    ss = r["score_sorted"].astype(np.float64)            # [T, H, 2k+1], forced = +inf
    k = cfg.k_budget
    amp = np.zeros((T, cfg.n_q_heads))
    for t in range(k, T):                                # t + 1 <= k: sigma = 1 by convention (G5)
        f = 1 if t == 0 else 2
        den = ss[t, :, f] - ss[t, :, k]
        scale = np.maximum(np.abs(ss[t, :, f]), np.abs(ss[t, :, k]))
        with np.errstate(divide="ignore", invalid="ignore"):
            amp[t] = np.where(den > 0, scale / den, np.inf)
    out["amp_bar_hex"] = amp.mean(axis=1).astype(np.float32).view(np.uint32).tobytes().hex()
    # per-head sigma of a few tiles, so a reader can spot-check the file against oracle.select_tiles
    probe = sorted({0, cfg.k_budget, T // 2, T - 1})
    out["sigma_probe"] = {str(t): [float(x) for x in sigma[t]] for t in probe}
    for q in CASES[case]:
        sb, tau, trig = oracle.route(sigma, policy, q)
        assert np.array_equal(sb.view(np.uint32), sigma_bar.view(np.uint32))
        out["routes"][repr(q)] = {
            "m": int(np.ceil(q * T - 1e-9)),
            "tau_hex": np.float32(tau).view(np.uint32).item().to_bytes(4, "little").hex(),
            "tau": float(tau),
            "n_trigger": int(trig.sum()),
            "trigger_bits": "".join("1" if x else "0" for x in trig),
        }
    out["oracle_seconds"] = round(time.time() - t0, 1)
    out["oracle_threads"] = oracle.max_threads()
    return out


def load(case: str):
    """Reader used by the tests: returns dict(sigma_bar fp32 [T], routes {q: (m, tau, trigger u8 [T])})."""
    p = path_of(case)
    if not os.path.exists(p):
        return None
    with open(p) as f:
        d = json.load(f)
    sb = np.frombuffer(bytes.fromhex(d["sigma_bar_hex"]), dtype=np.uint32).view(np.float32).copy()
    amp = np.frombuffer(bytes.fromhex(d["amp_bar_hex"]), dtype=np.uint32).view(np.float32).copy()
    routes = {}
    for q, r in d["routes"].items():
        tau = np.frombuffer(bytes.fromhex(r["tau_hex"]), dtype=np.uint32).view(np.float32)[0]
        trig = np.frombuffer(r["trigger_bits"].encode(), dtype=np.uint8) - ord("0")
        routes[float(q)] = (int(r["m"]), np.float32(tau), trig.astype(np.uint8))
    return dict(sigma_bar=sb, amp_bar=amp, routes=routes, meta=d)


if __name__ == "__main__":
    todo = sys.argv[1:] or list(CASES)
    for case in todo:
        if case.split("/")[0] not in synth.CONFIGS:
            print(f"skip {case}: unknown config")
            continue
        d = make(case)
        with open(path_of(case), "w") as f:
            json.dump(d, f)
            f.write("\n")
        print(f"{case}: T={d['T']} {d['oracle_seconds']} s -> {os.path.relpath(path_of(case), ROOT)}",
              flush=True)
