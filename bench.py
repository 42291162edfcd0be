#!/usr/bin/env python
"""bench.py -- one JSON line for the selection + sparse-attention prefill path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3b|C2|C3a|C3c|C4|C5|C1]
                    [--policy router_quest] [--q-frac 0.25] [--no-extra] [--impl reference]

A step is one pass of the whole hot path over one synthetic prefill layer:
bsa_build_block_meta -> bsa_select -> bsa_sparse_attn_fwd (rows 1-6, the "sparse prefill attention")
and bsa_dense_attn_fwd (row 7, the "x dense" denominator).  Each stage is bracketed by CUDA events on
the launching stream; L2 is flushed (512 MiB memset) before every step, outside the event pairs.
Default workload: C3b, the 128K Qwen2.5-7B-shaped layer with router_quest that BASELINE.json's
north_star names as the headline ("router_quest sparse prefill at 128K ... as a measured ratio of this
library's own dense kernel time").

  value        = ms of rows 1-6 (pool + select + sparse attention), mean over the K timed steps,
                 inputs resident in HBM; `stats` carries median and min per stage
  ms_per_step  = rows 1-7 (value + dense kernel)
  x_dense      = value / dense ms (the paper's "x dense wall time", attention only), phases timed apart,
                 each with its own clock record; x_dense_interleaved = the same ratio with the dense
                 kernel launched directly before every sparse pass (the other ordering)
  e2e          = the same rows 1-6 through the C ABI from pinned HOST buffers: H2D of Q, K, V and D2H of
                 O inside the timed region
  roofline     = the sparse attention kernel (dominant kernel of rows 1-6) against the measured bf16 peak
  cpu_baseline = the CPU oracle (oracle/), timed on this host's cores on a bounded sample of the same
                 workload; `measured_ms` is what was timed, `scale` the factor to the full workload,
                 `value` their product, labelled `extrapolated`
  extra        = the other BASELINE.json configs (C2, C3a, C4, C5, C3c) and the k_budget / q sweeps the
                 paper itself varies, fewer steps each

N > 1: the path does not shard (replicas only); every rank runs an independent
replica, the time is the max over ranks.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "sparse prefill attention ms (pool+select+sparse attn); x dense"
PEAKS_FALLBACK = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["_source"] = "measured"
        return d
    d = dict(PEAKS_FALLBACK)
    d["_source"] = "fallback"
    return d


# ---- clocks ---------------------------------------------------------------------------------------
class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self._stop, self._th = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True,
                                     timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.splitlines()[0].split(",")])
            except Exception:
                pass
            self._stop.wait(0.1)

    def start(self):
        self._th = threading.Thread(target=self._run, daemon=True)
        self._th.start()

    def stop(self) -> dict:
        self._stop.set()
        if self._th:
            self._th.join(timeout=6)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---- algorithmic work -----------------------------------------------------------------------------
def algorithmic(cfg, kv_count_sum: int):
    Bn, d, T, H = cfg.block, cfg.head_dim, cfg.n_blocks, cfg.n_q_heads
    return {
        "sparse_flops": 4.0 * Bn * Bn * d * kv_count_sum,               # diagonal block counted in full
        "dense_flops": 4.0 * Bn * Bn * d * H * (T * (T + 1) / 2.0),
        "pool_bytes": cfg.seqlen * cfg.n_kv_heads * d * 2.0,             # K read once
        "gather_bytes": 2.0 * Bn * d * 2.0 * kv_count_sum,              # K and V tile per selected block
    }


def ncu_traffic(key: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, taken from the
    committed `ncu --set full` capture of that kernel on this workload (profiles/traffic.json names the
    capture); None when no capture of this workload / policy is committed."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        ent = json.load(f).get(key)
    return None if ent is None else float(ent["dram_bytes_read"]) + float(ent["dram_bytes_write"])


# ---- the CPU oracle legs --------------------------------------------------------------------------
def golden_route(cfg, policy: str, q_frac: float):
    """(tau, trigger[T]) of the WHOLE sequence from the oracle-written golden (tests/golden/), or None."""
    case = f"{cfg.name}/{policy}"
    p = os.path.join(ROOT, "tests", "golden", "routing_" + case.replace("/", "_") + ".json")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        d = json.load(f)
    r = d["routes"].get(repr(float(q_frac)))
    if r is None or d["seed"] != cfg.seed or d["seqlen"] != cfg.seqlen:
        return None
    return float(r["tau"]), np.frombuffer(r["trigger_bits"].encode(), dtype=np.uint8) - ord("0")


def oracle_sample_ms(cfg, inp, policy: str, q_frac: float, stride: int = 16):
    """Oracle rows 1-6.  stride == 1: the whole workload, with the oracle's own routing.  stride > 1: a
    stratified sample of tiles (every stride-th, all heads); pooling runs in full; the trigger of the
    sampled tiles comes from the oracle's full-sequence routing (tests/golden/routing_*.json, written
    by oracle/ alone) when that file exists, else from the sample's own quantile (said in the text).
    Returns dict(measured_ms, scale, value, seconds, sample)."""
    import oracle
    oracle.max_threads()                       # builds / loads the oracle library outside the timed part
    T, H, k = cfg.n_blocks, cfg.n_q_heads, cfg.k_budget
    stride = max(1, min(stride, max(T // 2, 1)))
    tiles = np.arange(stride // 2, T, stride)
    n = len(tiles)
    router = policy in ("router", "router_quest")
    gold = golden_route(cfg, policy, q_frac) if (stride > 1 and router) else None
    t0 = time.perf_counter()
    meta = oracle.pool(inp.K, cfg.block)
    t1 = time.perf_counter()
    r = oracle.select_tiles(inp.Q, meta, cfg.block, policy, k, tiles)
    if gold is not None:
        trig = gold[1][tiles]
        how = "trigger of the sampled tiles from the oracle's full-sequence routing (tests/golden)"
    else:
        _, _, trig = oracle.route(r["sigma"], policy, q_frac)
        how = "oracle routing" if stride == 1 else "routing by the sample's own quantile"
    W = oracle.kv_width(policy, k)
    kv_idx = np.full((H, T, W), T, np.int32)
    kv_count = np.zeros((H, T), np.int32)
    for i, t in enumerate(tiles):
        cnt = min(2 * k if trig[i] else k, t + 1)
        kv_idx[:, t, :cnt] = r["idx_sorted"][i, :, :cnt]
        kv_count[:, t] = cnt
    t2 = time.perf_counter()
    pairs = [(int(t), h) for t in tiles for h in range(H)]
    oracle.attn_pairs(inp.Q, inp.K, inp.V, cfg.block, pairs, kv_idx, kv_count, want_lse=False)
    t3 = time.perf_counter()
    pool_ms, rest_ms = (t1 - t0) * 1e3, (t3 - t1) * 1e3
    scale = T / n
    if stride == 1:
        text = f"the whole workload: all {T} tiles x {H} heads, {how}"
    else:
        text = (f"pooling in full ({pool_ms:.0f} ms); scoring + top-k + sigma + fill + sparse attention on "
                f"{n} of {T} tiles (every {stride}th, all {H} heads; {rest_ms:.0f} ms measured, x{scale:.4g}); {how}")
    return {"measured_ms": pool_ms + rest_ms, "scale": scale, "value": pool_ms + rest_ms * scale,
            "extrapolated": stride > 1, "seconds": t3 - t0, "sample": text}


def reference_stride(cfg, steps_total: int, cores: int) -> int:
    """Tile stride (a power of two) that keeps the whole reference run near 2-3 minutes: the oracle does
    2.3e8 (C2 in full: 33 s on 16 cores) to 7e8 (128K samples) MAC/s per core; 4e8 is assumed."""
    work = cfg.n_blocks * (cfg.n_blocks + 1) / 2 * cfg.block * cfg.head_dim * cfg.n_q_heads * 4.0
    per_step_s = 150.0 / max(steps_total, 1)
    need = work / (4e8 * max(cores, 1) * per_step_s)
    return int(min(512, max(1, 2 ** math.ceil(math.log2(max(need, 1))))))


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on the host cores, same config / metric.  Each step
    is a bounded sample of the workload; `ms_per_step` is what a step really took, `value` the same metric
    as the GPU arm (ms for the full workload) = pooling + measured rest x scale, labelled extrapolated."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from paper_2607_07724_b200 import synth
    cfg = synth.CONFIGS[args.workload]
    inp = synth.make_inputs(cfg)
    oracle.build()
    stride = reference_stride(cfg, args.warmup + args.steps, oracle.max_threads())
    runs = []
    for i in range(args.warmup + args.steps):
        r = oracle_sample_ms(cfg, inp, args.policy, args.q_frac, stride)
        if i >= args.warmup:
            runs.append(r)
    v = float(np.mean([r["value"] for r in runs]))
    measured = float(np.mean([r["measured_ms"] for r in runs]))
    base = {"kind": "oracle", "cores": oracle.max_threads(), "sample": runs[-1]["sample"],
            "measured_ms": measured, "scale": runs[-1]["scale"], "extrapolated": runs[-1]["extrapolated"]}
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": "ms", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": measured, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64 accumulate, f32 results (CPU oracle)",
        "data": "synthetic",
        "config": workload_config(cfg, args),
        "cpu_baseline": dict(base, value=v, unit="ms"),
        "e2e": {"value": v, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
        "note": "value = ms for the full workload (extrapolated from the sample when scale > 1); "
                "ms_per_step = the measured time of one step of this arm",
    }
    print(json.dumps(line), flush=True)


def workload_config(cfg, args):
    return {"workload": f"{cfg.name}: B1 N={cfg.seqlen} Hq={cfg.n_q_heads} Hkv={cfg.n_kv_heads} "
                        f"d={cfg.head_dim} block={cfg.block} k_budget={cfg.k_budget}",
            "policy": args.policy, "q_frac": args.q_frac, "k_budget": cfg.k_budget, "seqlen": cfg.seqlen,
            "order": "K timed passes of rows 1-6, then K timed passes of row 7 (dense reference kernel), then 3 "
                     "interleaved passes (dense, sparse) for x_dense_interleaved",
            "l2": "flushed before every step (512 MiB memset outside the event pairs); "
                  "Q+K+V+O also exceed the 126 MB L2",
            "parallelism": "replicas only"}


def max_over_ranks(values, world: int, device: str):
    """Replicas only: every rank times the same independent workload; a multi-GPU
    number is the MAX over ranks of the device-timed milliseconds.  No data-path collective exists."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.tolist()]


# ---- the GPU arm ----------------------------------------------------------------------------------
class Runner:
    """Device tensors + preallocated outputs for one workload; step() enqueues rows 1-7."""

    def __init__(self, cfg, inp, policy, q_frac, torch, bsa):
        self.cfg, self.policy, self.q_frac, self.torch, self.bsa = cfg, policy, q_frac, torch, bsa

        def host(bits):
            t = torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16)[None]
            return t.pin_memory()

        self.hQ, self.hK, self.hV = host(inp.Q), host(inp.K), host(inp.V)
        self.Q, self.K, self.V = (x.cuda() for x in (self.hQ, self.hK, self.hV))
        self.O = torch.empty_like(self.Q)
        self.Od = torch.empty_like(self.Q)
        self.hO = torch.empty(self.Q.shape, dtype=torch.bfloat16).pin_memory()
        shape = bsa.make_shape(self.Q, self.K, cfg.block)
        self.meta = torch.empty(bsa.bsa_block_meta_bytes(shape, 3), dtype=torch.uint8, device="cuda")
        B, H, N, _ = self.Q.shape
        T, W = cfg.n_blocks, bsa.bsa_kv_width(policy, cfg.k_budget)
        dev = "cuda"
        self.sel = dict(kv_idx=torch.empty((B, H, T, W), dtype=torch.int32, device=dev),
                        kv_count=torch.empty((B, H, T), dtype=torch.int32, device=dev),
                        sigma=torch.empty((B, H, T), dtype=torch.float32, device=dev),
                        sigma_bar=torch.empty((B, T), dtype=torch.float32, device=dev),
                        trigger=torch.empty((B, T), dtype=torch.uint8, device=dev),
                        tau=torch.empty((B,), dtype=torch.float32, device=dev))
        self.kinds = 2 if policy in ("quest", "router_quest") else 1
        self.flush_buf = torch.empty(512 << 20, dtype=torch.uint8, device=dev)

    def flush_l2(self):
        self.flush_buf.zero_()

    def sparse_path(self, Q=None, K=None, V=None, ev=None):
        """rows 1-6; ev = list that receives events after each stage"""
        bsa, cfg, torch = self.bsa, self.cfg, self.torch
        Q = self.Q if Q is None else Q
        K = self.K if K is None else K
        V = self.V if V is None else V

        def mark():
            if ev is not None:
                e = torch.cuda.Event(enable_timing=True)
                e.record()
                ev.append(e)
        mark()
        bsa.bsa_build_block_meta(K, cfg.block, self.kinds, self.meta)
        mark()
        bsa.bsa_select(Q, self.meta, K, cfg.block, self.policy, cfg.k_budget, self.q_frac, out=self.sel)
        mark()
        bsa.bsa_sparse_attn_fwd(Q, K, V, self.sel["kv_idx"], self.sel["kv_count"], cfg.block, O=self.O)
        mark()

    def dense(self, ev=None):
        self.bsa.bsa_dense_attn_fwd(self.Q, self.K, self.V, self.cfg.block, O=self.Od)
        if ev is not None:
            e = self.torch.cuda.Event(enable_timing=True)
            e.record()
            ev.append(e)

    def timed_steps(self, steps, warmup, with_dense=True, clocks_index=None, interleaved=0):
        """Per-stage ms lists over `steps` steps: pool, select, sparse, dense (+ clock records per phase).

        The K timed steps run as K passes of rows 1-6 followed by K passes of row 7 (the dense
        kernel): a dense launch (full tensor-pipe power for 7-115 ms) directly in front of the sparse
        path drops the SM clock from 1965 to ~1665 MHz for the next kernels and inflates the sparse
        attention by 10-25 % (measured: 1.81 -> 2.13 ms at C2).  Both phases get their own clock
        record, and `interleaved` > 0 adds that many steps in the other ordering (dense, then sparse,
        back to back) so that both bounds of the ratio are on the line."""
        torch = self.torch

        def ev():
            e = torch.cuda.Event(enable_timing=True)
            e.record()
            return e

        for _ in range(warmup):
            self.flush_l2()
            self.sparse_path()
        torch.cuda.synchronize()
        clk = {}
        sampler = ClockSampler(clocks_index) if clocks_index is not None else None
        if sampler:
            sampler.start()
        all_ev, dense_ev, inter_ev = [], [], []
        for _ in range(steps):
            self.flush_l2()
            evs = []
            self.sparse_path(ev=evs)
            all_ev.append(evs)
        torch.cuda.synchronize()
        if sampler:
            clk["sparse_phase"] = sampler.stop()
        if with_dense:
            for _ in range(min(warmup, 3)):
                self.flush_l2()
                self.dense()
            torch.cuda.synchronize()
            sampler = ClockSampler(clocks_index) if clocks_index is not None else None
            if sampler:
                sampler.start()
            for _ in range(steps):
                self.flush_l2()
                e0 = ev()
                self.dense()
                dense_ev.append((e0, ev()))
            torch.cuda.synchronize()
            if sampler:
                clk["dense_phase"] = sampler.stop()
            for _ in range(interleaved):
                self.flush_l2()
                e0 = ev()
                self.dense()
                e1 = ev()
                self.flush_l2()
                evs = []
                self.sparse_path(ev=evs)
                inter_ev.append((e0, e1, evs))
            torch.cuda.synchronize()
        names = ["pool", "select", "sparse"]
        per = {n: [] for n in names}
        for evs in all_ev:
            for i, n in enumerate(names):
                per[n].append(evs[i].elapsed_time(evs[i + 1]))
        per["path"] = [evs[0].elapsed_time(evs[3]) for evs in all_ev]      # rows 1-6 incl. launch gaps
        if with_dense:
            per["dense"] = [a.elapsed_time(b) for a, b in dense_ev]
            if inter_ev:
                per["dense_interleaved"] = [a.elapsed_time(b) for a, b, _ in inter_ev]
                per["path_interleaved"] = [evs[0].elapsed_time(evs[3]) for _, _, evs in inter_ev]
        self.clocks = clk
        return per

    def e2e_steps(self, steps, warmup):
        """rows 1-6 from pinned host buffers: H2D Q,K,V + kernels + D2H O inside the timed region."""
        torch = self.torch
        times = []
        for i in range(warmup + steps):
            self.flush_l2()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            self.Q.copy_(self.hQ, non_blocking=True)
            self.K.copy_(self.hK, non_blocking=True)
            self.V.copy_(self.hV, non_blocking=True)
            self.sparse_path()
            self.hO.copy_(self.O, non_blocking=True)
            e1.record()
            torch.cuda.synchronize()
            if i >= warmup:
                times.append(e0.elapsed_time(e1))
        h2d = sum(x.numel() * 2 for x in (self.hQ, self.hK, self.hV))
        d2h = self.hO.numel() * 2
        return float(np.mean(times)), h2d, d2h


def stats_of(per: dict) -> dict:
    """mean / median / min per stage (SURVEY 8(d) "Timing procedure": >= 8 repetitions, median and min)."""
    return {n: {"mean": float(np.mean(v)), "median": float(np.median(v)), "min": float(np.min(v)), "n": len(v)}
            for n, v in per.items()}


def summarize(cfg, per: dict, kv_sum: int, peaks: dict) -> dict:
    """Per-config record: stage ms (mean), x dense, tokens/s, roofline fractions."""
    st = stats_of(per)
    m = {n: st[n]["mean"] for n in st}
    alg = algorithmic(cfg, kv_sum)
    path = m["pool"] + m["select"] + m["sparse"]
    peak_tf = peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"])
    rec = {"seqlen": cfg.seqlen, "sparse_path_ms": path, "pool_ms": m["pool"], "select_ms": m["select"],
           "sparse_attn_ms": m["sparse"], "stats": st, "kv_count_sum": kv_sum,
           "mean_blocks_per_tile": kv_sum / (cfg.n_q_heads * cfg.n_blocks),
           "tokens_per_s": cfg.seqlen / (path * 1e-3),
           "pool_gbs": alg["pool_bytes"] / (m["pool"] * 1e-3) / 1e9,
           "pool_frac_of_hbm_peak": alg["pool_bytes"] / (m["pool"] * 1e-3) / 1e9 / peaks["hbm_gbs"],
           "sparse_tflops": alg["sparse_flops"] / (m["sparse"] * 1e-3) / 1e12,
           "sparse_frac_of_bf16_peak": alg["sparse_flops"] / (m["sparse"] * 1e-3) / 1e12 / peak_tf}
    if "dense" in m:
        rec.update({"dense_attn_ms": m["dense"], "x_dense": path / m["dense"],
                    "x_dense_kernel_only": m["sparse"] / m["dense"],
                    "dense_tflops": alg["dense_flops"] / (m["dense"] * 1e-3) / 1e12,
                    "dense_frac_of_bf16_peak": alg["dense_flops"] / (m["dense"] * 1e-3) / 1e12 / peak_tf})
    if "dense_interleaved" in m:
        rec["x_dense_interleaved"] = m["path_interleaved"] / m["dense_interleaved"]
    return rec


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_2607_07724_b200 import binding as bsa
    from paper_2607_07724_b200 import synth

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback exists)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    bsa.load_library()     # raises if libbsa.so cannot be built / loaded
    peaks = load_peaks()

    cfg = synth.CONFIGS[args.workload]
    inp = synth.make_inputs(cfg)
    run = Runner(cfg, inp, args.policy, args.q_frac, torch, bsa)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    clocks = ClockSampler(local)
    barrier()
    clocks.start()
    t_wall0 = time.perf_counter()
    per = run.timed_steps(args.steps, args.warmup, clocks_index=local, interleaved=min(3, args.steps))
    barrier()
    wall_ms = (time.perf_counter() - t_wall0) * 1e3
    clk = clocks.stop()
    clk["phases"] = run.clocks

    mean = {n: float(np.mean(v)) for n, v in per.items()}
    sparse_ms = mean["pool"] + mean["select"] + mean["sparse"]
    step_ms = sparse_ms + mean["dense"]
    sparse_ms, step_ms = max_over_ranks([sparse_ms, step_ms], world, "cuda")

    kv_sum = int(run.sel["kv_count"].sum().item())
    alg = algorithmic(cfg, kv_sum)
    e2e_ms, h2d, d2h = run.e2e_steps(max(2, min(args.steps, 5)), 2)
    (e2e_ms,) = max_over_ranks([e2e_ms], world, "cuda")

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    head = summarize(cfg, per, kv_sum, peaks)
    tf_sparse, tf_dense = head["sparse_tflops"], head["dense_tflops"]
    peak_tf = peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"])
    gather_gbs = alg["gather_bytes"] / (mean["sparse"] * 1e-3) / 1e9
    sm_mhz = (run.clocks.get("sparse_phase") or {}).get("sm_mhz") or clk.get("sm_mhz") or 1965.0
    lts_peak_gbs = 64.0 * 148 * sm_mhz * 1e6 / 1e9
    n_sparse_launches = 5 if args.policy.startswith("router") else 4
    line = {
        "metric": METRIC, "value": sparse_ms, "unit": "ms", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "bf16 (fp32 accumulate / softmax; fp32 block scores)",
        "data": "synthetic",
        "config": workload_config(cfg, args),
        "tokens_per_s": cfg.seqlen * world / (sparse_ms * 1e-3),
        "x_dense": head["x_dense"],
        "x_dense_kernel_only": head["x_dense_kernel_only"],
        "x_dense_interleaved": head.get("x_dense_interleaved"),
        "stages_ms": {"pool": mean["pool"], "select": mean["select"], "sparse_attn": mean["sparse"],
                      "dense_attn": mean["dense"]},
        "stats": head["stats"],
        "wall_ms_timed_region": wall_ms,
        "kv_count_sum": kv_sum,
        "mean_blocks_per_tile": head["mean_blocks_per_tile"],
        "roofline": {"bound": "tensor",
                     "kernel": ("attn64p_kernel (bsa_sparse_attn_fwd; persistent, 64-token blocks)"
                                if cfg.block == 64 and cfg.k_budget * 2 <= 128 else
                                "attn_kernel<sparse> (bsa_sparse_attn_fwd)"),
                     "achieved": tf_sparse, "peak": peak_tf, "unit": "TFLOP/s", "frac": tf_sparse / peak_tf,
                     "traffic": ncu_traffic(f"attn_sparse/{args.workload}/{args.policy}"),
                     "peak_source": f"{peaks['_source']} bf16_tflops_sustained",
                     "algorithmic_flops_per_launch": alg["sparse_flops"]},
        # secondary ceiling of the same kernel: every selected block is gathered L2 -> shared memory
        # (K and V tile, 2*Bn*d*2 bytes) for 4*Bn*Bn*d flops = 64 flop/B at Bn=64.  The ceiling is the
        # SM's L2 read port, 64 B/clk/SM: the TMA-only ablation of this kernel (no MMA, no softmax)
        # measured 19.2-19.5 TB/s on B200 = 64 B/clk x 148 SMs x 1.965 GHz x 1.03.
        "roofline_l2_gather": {"bound": "l2", "achieved": gather_gbs, "peak": lts_peak_gbs, "unit": "GB/s",
                               "frac": gather_gbs / lts_peak_gbs,
                               "bytes_per_launch": alg["gather_bytes"],
                               "peak_source": "64 B/clk/SM x 148 SMs x SM clock of the sparse phase "
                                              "(TMA-only ablation of the same kernel reached it)"},
        "roofline_dense": {"bound": "tensor", "achieved": tf_dense, "peak": peak_tf, "unit": "TFLOP/s",
                           "frac": tf_dense / peak_tf},
        "roofline_pool": {"bound": "hbm", "achieved": head["pool_gbs"], "peak": peaks["hbm_gbs"],
                          "unit": "GB/s", "frac": head["pool_frac_of_hbm_peak"],
                          "algorithmic_bytes": alg["pool_bytes"], "note": "cold L2 (flushed before the step)"},
        "e2e": {"value": e2e_ms, "unit": "ms", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        # launches of libbsa kernels inside the timed region: K sparse passes (pool, score, route[,
        # finalize], attention), K dense, and the interleaved-order passes
        "gpu_launches": args.steps * (n_sparse_launches + 1) + min(3, args.steps) * (n_sparse_launches + 1),
        "clocks": clk,
    }

    # ---- the other BASELINE.json configs and the paper's own sweeps (fewer steps each) ------------------
    if not args.no_extra and world == 1:
        from dataclasses import replace
        del run
        torch.cuda.empty_cache()
        extra, sweeps, line_next = {}, {}, {}
        n_x, w_x = max(3, min(args.steps, 8)), 2
        plans = [("C2", ("router_quest", "topk", "quest", "router")), ("C3a", ("router_quest", "topk")),
                 ("C3b", ("topk",)), ("C4", ("router_quest", "quest")), ("C5", ("router_quest", "router")),
                 ("C3c", ("router_quest", "topk"))]
        for name, pols in plans:
            c = synth.CONFIGS[name]
            i2 = inp if name == args.workload else synth.make_inputs(c)
            dense_per = None
            for pol in pols:
                if name == args.workload and pol == args.policy:
                    continue
                r2 = Runner(c, i2, pol, args.q_frac, torch, bsa)
                # the dense kernel once per config (at 256K it alone is ~0.5 s per pass: 2 passes)
                want_dense = dense_per is None and not (name == args.workload)
                p2 = r2.timed_steps(2 if name == "C3c" else n_x, w_x, with_dense=want_dense, clocks_index=local)
                if want_dense:
                    dense_per = p2["dense"]
                elif dense_per is not None:
                    p2["dense"] = dense_per
                elif name == args.workload:
                    p2["dense"] = per["dense"]
                rec = summarize(c, p2, int(r2.sel["kv_count"].sum().item()), peaks)
                rec["clocks"] = r2.clocks
                extra[f"{name}/{pol}"] = rec
                del r2
                torch.cuda.empty_cache()
            if name == "C2":   # k_budget in {33..66} (Table 4), q in {.1...4} (L123)
                for kb, pol, qf in ([(kb, "router_quest", 0.4) for kb in (33, 40, 47, 52, 66)] +
                                    [(kb, "quest", 0.0) for kb in (33, 66)] +
                                    [(33, "router_quest", qf) for qf in (0.1, 0.2, 0.3)]):
                    r2 = Runner(replace(c, k_budget=kb), i2, pol, qf, torch, bsa)
                    p2 = r2.timed_steps(3, 1, with_dense=False)
                    p2["dense"] = dense_per
                    rec = summarize(replace(c, k_budget=kb), p2, int(r2.sel["kv_count"].sum().item()), peaks)
                    rec.pop("stats")
                    sweeps[f"k={kb}/{pol}/q={qf}"] = rec
                    del r2
                    torch.cuda.empty_cache()
            if name == "C2":   # SURVEY 8(f).3 / 8(f).4 on the 32K layer: diagnostics mode, per-row bitmap
                r2 = Runner(c, i2, "router_quest", args.q_frac, torch, bsa)
                next_rows = {}

                def timed(fn, n=5):
                    ts = []
                    for i in range(n + 2):
                        r2.flush_l2()
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        e0.record()
                        fn()
                        e1.record()
                        torch.cuda.synchronize()
                        if i >= 2:
                            ts.append(e0.elapsed_time(e1))
                    return float(np.median(ts))

                bsa.bsa_build_block_meta(r2.K, c.block, 3, r2.meta)
                next_rows["select_ms"] = timed(lambda: bsa.bsa_select(
                    r2.Q, r2.meta, r2.K, c.block, "router_quest", c.k_budget, args.q_frac, out=r2.sel))
                dsel = dict(r2.sel)
                next_rows["select_diag_ms"] = timed(lambda: dsel.update(bsa.bsa_select(
                    r2.Q, r2.meta, r2.K, c.block, "router_quest", c.k_budget, args.q_frac, out=dsel, diag=True)))
                next_rows["diag_summary"] = dict(zip(bsa.DIAG_SUMMARY, dsel["summary"][0].cpu().tolist()))
                for k_row in (4, 8):
                    box = {}
                    ms = timed(lambda: box.update(zip(("bm", "cnt"), bsa.bsa_select_rows_bitmap(
                        r2.Q, r2.meta, r2.K, c.block, "quest", k_row))))
                    cnt = int(box["cnt"].sum().item())
                    ms_a = timed(lambda: bsa.bsa_sparse_attn_fwd_bitmap(r2.Q, r2.K, r2.V, box["bm"], c.block, O=r2.O))
                    a2 = algorithmic(c, cnt)
                    next_rows[f"rows_bitmap/quest/k_row={k_row}"] = {
                        "select_rows_bitmap_ms": ms, "bitmap_attn_ms": ms_a,
                        "mean_blocks_per_tile": cnt / (c.n_q_heads * c.n_blocks),
                        "bitmap_attn_tflops": a2["sparse_flops"] / (ms_a * 1e-3) / 1e12}
                line_next = next_rows
                del r2, dsel
                torch.cuda.empty_cache()
            del i2
        # bsa_select_attn_fwd (one call, attention as a programmatic dependent launch)
        # beside the two-call path, rows 2-6 with the pooled planes already built
        one_call = {}
        for name in ("C3b", "C3c"):
            c = synth.CONFIGS[name]
            i2 = inp if name == args.workload else synth.make_inputs(c)
            r2 = Runner(c, i2, "router_quest", args.q_frac, torch, bsa)
            bsa.bsa_build_block_meta(r2.K, c.block, r2.kinds, r2.meta)

            def two():
                bsa.bsa_select(r2.Q, r2.meta, r2.K, c.block, "router_quest", c.k_budget, args.q_frac, out=r2.sel)
                bsa.bsa_sparse_attn_fwd(r2.Q, r2.K, r2.V, r2.sel["kv_idx"], r2.sel["kv_count"], c.block, O=r2.O)

            def one():
                bsa.bsa_select_attn_fwd(r2.Q, r2.K, r2.V, r2.meta, c.block, "router_quest", c.k_budget,
                                        args.q_frac, out=r2.sel, O=r2.O)
            ts = {"two_calls_ms": [], "one_call_ms": []}
            for i in range(16):                      # alternate the two paths: clock drift hits both alike
                label, fn = (("two_calls_ms", two), ("one_call_ms", one))[i & 1]
                r2.flush_l2()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                fn()
                e1.record()
                torch.cuda.synchronize()
                if i >= 4:
                    ts[label].append(e0.elapsed_time(e1))
            res = {k: float(np.median(v)) for k, v in ts.items()}
            one_call[name + "/router_quest"] = res
            del r2, i2
            torch.cuda.empty_cache()
        line["extra"] = {"configs": extra, "sweeps": sweeps, "next_rows_c2": line_next,
                         "select_attn_one_call": one_call,
                         "note": f"{n_x} timed steps after {w_x} warm-ups per entry (C3c: 2), dense kernel timed "
                                 "once per config; sweeps at C2 (32K), 3 steps"}

    # ---- CPU oracle on this host's cores --------------------------------------------------------------
    import oracle
    cores = oracle.max_threads()
    work = cfg.n_blocks * (cfg.n_blocks + 1) / 2 * cfg.block * cfg.head_dim * cfg.n_q_heads * 4.0
    stride = int(min(512, max(1, 2 ** math.ceil(math.log2(max(work / (4e8 * cores * 20.0), 1))))))
    cb = oracle_sample_ms(cfg, inp, args.policy, args.q_frac, stride)
    line["cpu_baseline"] = {"value": cb["value"], "unit": "ms", "cores": cores, "kind": "oracle",
                            "sample": cb["sample"], "measured_ms": cb["measured_ms"], "scale": cb["scale"],
                            "extrapolated": cb["extrapolated"], "cpu_seconds_spent": cb["seconds"]}
    if args.workload != "C2" and not args.no_extra and world == 1:
        # the sparse pipeline timed IN FULL where that is affordable (C2, 32K)
        c2 = synth.CONFIGS["C2"]
        cb2 = oracle_sample_ms(c2, synth.make_inputs(c2), args.policy, args.q_frac, 1)
        line["cpu_baseline_c2_full"] = {"value": cb2["value"], "unit": "ms", "cores": cores, "kind": "oracle",
                                        "sample": cb2["sample"], "extrapolated": False,
                                        "cpu_seconds_spent": cb2["seconds"]}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C3b")
    ap.add_argument("--policy", default="router_quest")
    ap.add_argument("--q-frac", type=float, default=0.25)
    ap.add_argument("--impl", default="bsa", choices=["bsa", "reference"])
    ap.add_argument("--no-extra", action="store_true",
                    help="skip the other configs, the k_budget / q_frac sweeps and the full C2 oracle run")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
