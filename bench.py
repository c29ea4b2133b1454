#!/usr/bin/env python
"""bench.py — FlashCP per-CP-rank hot path on B200 (see DESIGN.md section 7 for the contract).

A "step" is one pass of the whole hot path over one packed batch of the named config: host
plan + rank layouts + tile schedules, then for every virtual CP rank, one after another on the
GPU: sharding-aware KV gather -> attention forward -> attention backward.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 8b] [--impl fcp|reference]

metric = document-masked attention fwd+bwd useful TFLOP/s (14*D*Hq*sum W) over
the WHOLE step time (gather and host planning included); side reports: per-phase TFLOP/s,
gather GB/s, plan statistics (Eq. 4 / Eq. 5, imbalance), roofline, CPU oracle baseline.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import fcp_inputs  # noqa: E402

METRIC = "doc-masked attn fwd+bwd useful TFLOP/s"
NOMINAL_BF16_TFLOPS = 2250.0
FALLBACK_BF16_TFLOPS = 1590.0
FALLBACK_HBM_GBS = 6650.0


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            j = json.load(open(p))
            return {"bf16": float(j["bf16_tflops"]), "bf16_sustained": float(j.get(
                "bf16_tflops_sustained", j["bf16_tflops"])), "hbm": float(j["hbm_gbs"]),
                "source": "measured"}
        except Exception:
            pass
    return {"bf16": FALLBACK_BF16_TFLOPS, "bf16_sustained": 1400.0, "hbm": FALLBACK_HBM_GBS,
            "source": "fallback"}


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx,
                "reasons": sorted(reasons), "samples": len(sm)}


def useful_flops(cfg, d):
    pairs = sum(x * (x + 1) // 2 for x in d)           # sum_shards W is plan independent
    return 4 * cfg.D * cfg.Hq * pairs, 10 * cfg.D * cfg.Hq * pairs


# ------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle, as it stands, on the host cores
# ------------------------------------------------------------------------------------------
def oracle_sample(cfg, d, seed):
    """One bounded sample: every virtual rank, ONE GQA group (1 kv head + its G query heads);
    heads are independent units, so useful flops scale by 1/Hkv.  Returns (flops, seconds)."""
    from oracle import attention as OA, kvselect as OKV, planner as OP
    G = cfg.Hq // cfg.Hkv
    rng = np.random.default_rng(seed)
    Q = rng.standard_normal((cfg.C, G, cfg.D))
    K = rng.standard_normal((cfg.C, 1, cfg.D))
    V = rng.standard_normal((cfg.C, 1, cfg.D))
    dO = rng.standard_normal((cfg.C, G, cfg.D))
    scale = 1.0 / math.sqrt(cfg.D)
    t0 = time.perf_counter()
    pl = OP.plan(d, cfg.N)
    for r in range(cfg.N):
        lay = OKV.rank_layout(pl, r)
        qi, gi = OKV.q_token_index(pl, r), OKV.gather_index(pl, r)
        kg, vg = K[gi], V[gi]
        args = (lay.cu_seqlens_q, lay.q_pos_off, lay.shard_seg, lay.cu_seqlens_k, scale)
        o, lse = OA.rank_fwd(Q[qi], kg, vg, *args)
        OA.rank_bwd(Q[qi], kg, vg, o, lse, dO[qi], *args)
    dt = time.perf_counter() - t0
    f, b = useful_flops(cfg, d)
    return (f + b) / cfg.Hkv, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = fcp_inputs.CONFIGS[args.config]
    d = fcp_inputs.doc_lengths(args.config, args.seed)
    cores = len(os.sched_getaffinity(0))
    for _ in range(args.warmup):
        oracle_sample(fcp_inputs.CONFIGS["tiny"], fcp_inputs.doc_lengths("tiny"), 0)
    flops, secs = 0.0, 0.0
    for s in range(args.steps):
        f, t = oracle_sample(cfg, d, args.seed + s)
        flops += f
        secs += t
    val = flops / secs / 1e12
    sample = "per step: all %d virtual ranks, one GQA group (1 of %d kv heads), fp64 numpy" % (
        cfg.N, cfg.Hkv)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": "TFLOP/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.config, "C": cfg.C, "cp_ranks": cfg.N, "Hq": cfg.Hq,
                   "Hkv": cfg.Hkv, "D": cfg.D},
        "cpu_baseline": {"value": val, "unit": "TFLOP/s", "cores": cores, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": val, "unit": "TFLOP/s", "h2d_bytes_per_step": 0,
                "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))
