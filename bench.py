#!/usr/bin/env python
"""bench.py - loss+grad tokens/s of the fused AsyncWebRL token loss at V = 151,936 bf16.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config C]

One "step" = one pass of the whole hot path (segment expansion,
group advantage, log-sum-exp + gather, decoupled ratio / clip / normalizer, gradient write) over
one synthetic batch = one `awr_loss_fwd_bwd` call through the C ABI (include/awr.h).

Workload at N = 1: BASELINE.json configs[1] (8 groups x 8 trajectories, 40,960 tokens,
bf16 [40,960, 151,936] logits; eps 0.2, normalizer const 1/k with k = 10).  Inputs (12.4 GB of
logits, 12.4 GB of gradient) are far larger than the 126 MB L2, so no flush between steps.
N > 1: the path does not shard (BASELINE.json: "one GPU ... no inter-GPU collectives"):
N independent replicas, one per rank, each on its own seeded batch ("replicas only", weak
scaling); the only collectives are the timing barrier and the max-over-ranks of the time.

The JSON line:
  value         tokens/s, inputs resident in HBM, CUDA-event time over exactly K steps
  e2e           tokens/s through `awr_loss_fwd_bwd_host`: HOST (pinned) buffers, the H2D copy of
                every input and the D2H copy of every output inside the timed region
  roofline      the row kernel (a2+a3+a4): algorithmic bytes / its CUDA-event duration, measured
                live in the timed region (awr_outputs.ev_row_begin / ev_row_end of that call)
  cpu_baseline  the fp64 oracle (oracle/, as it stands) on the host cores, bounded sample
  --impl reference   times the oracle alone (this tier's reference arm)
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "loss+grad tokens/s at V=151,936 bf16"
UNIT = "tokens/s"
CPU_SAMPLE_TOK = 3072      # rows of the bounded oracle sample (about 10-30 s of CPU work)
REF_STEP_TOK = 256         # rows per step of the --impl reference arm
HEAD_CPU_SAMPLE_TOK = 2048  # rows of the fused-head oracle sample (three fp64 GEMMs of 2048 x 151,936)


def algorithmic_bytes_per_token(V: int, esz: int) -> int:
    """read the logits row once + write the gradient row once, + 24 B of
    per-token scalars (id, b, q in; l_t, term, flag/coef out)."""
    return 2 * V * esz + 24


# ---------------------------------------------------------------------------- rank plumbing
def dist_env():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init_dist(backend: str):
    import torch.distributed as dist
    rank, _, world = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29517")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def barrier(world: int):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def aggregate(local_ms: float, local_tokens: int, world: int, device="cpu"):
    """Whole-job numbers from per-rank ones: time = MAX over ranks, tokens = SUM over ranks.
    No data-path collective exists; this is the only communication of the benchmark."""
    if world == 1:
        return local_ms, local_tokens
    import torch
    import torch.distributed as dist
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    n = torch.tensor([local_tokens], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return float(t.item()), int(n.item())


# ---------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock + throttle reasons of one GPU through NVML while a region runs."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
               0x4: "sw_power_cap", 0x80: "hw_power_brake_slowdown"}

    def __init__(self, index: int, period_s: float = 0.005):
        self.period = period_s
        self.sm, self.reasons, self.power = [], set(), []
        self._stop = threading.Event()
        self._thr = None
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception as e:  # no NVML: say so in the JSON rather than invent numbers
            self.nv = None
            self.err = repr(e)

    def _loop(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                bits = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for b, name in self.REASONS.items():
                    if bits & b:
                        self.reasons.add(name)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if self.nv is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": statistics.median(self.sm) if self.sm else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.sm),
                "power_w_max": max(self.power) if self.power else None}


# ---------------------------------------------------------------------------- oracle legs
def oracle_sample(cfg: int, n_tok: int, seed: int):
    """A bounded sample of the bench workload: the same laws (gen/workloads.py) cut to n_tok."""
    from gen import workloads as W
    over = {} if cfg == 0 else dict(n_tok=n_tok)
    if cfg != 0 and n_tok < 1024:          # keep >= 1 token per step: fewer, same-law groups
        over.update(n_groups=2, group_size=8)
    w = W.workload(cfg, **over)
    host = W.to_host(W.make_batch(w, seed=seed, device="cpu"))
    return W.oracle_args(host), host


def time_oracle(args_kw, repeats: int = 1):
    from oracle import awr_oracle as O
    args, kw = args_kw
    fn = O.awr_loss_fwd_bwd_fused_head if len(args) == 9 else O.awr_loss_fwd_bwd   # config 4: hidden, W
    t0 = time.perf_counter()
    for _ in range(repeats):
        out = fn(*args, **kw)
    dt = time.perf_counter() - t0
    return dt / repeats, out


def host_threads_used() -> int:
    """The oracle is numpy elementwise code: one thread does the work."""
    return 1


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; rank 0 only."""
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    import numpy as np  # noqa: F401
    akw, host = oracle_sample(args.config, REF_STEP_TOK, seed=1234)
    n_tok = host["n_tok"]
    for _ in range(max(1, min(args.warmup, 2))):
        time_oracle(akw)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        time_oracle(akw)
    dt = time.perf_counter() - t0
    ms = dt / args.steps * 1e3
    val = n_tok / (ms / 1e3)
    sample = "config-%d laws cut to %d tokens per step, V=%d, fp64 numpy" % (
        args.config, n_tok, host["V"])
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT,
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[%d]" % args.config,
                       "n_tok_per_step": n_tok, "V": host["V"], "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": host_threads_used(),
                             "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------- the CUDA arm
def run_cuda(args):
    import torch

    import paper_2606_05597_b200 as A
    from gen import workloads as W

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a B200: there is no CPU path (use --impl reference "
                         "for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    init_dist("nccl")

    over = {}
    if args.n_tok:
        over["n_tok"] = args.n_tok
    w = W.workload(args.config, **over)
    if args.normalizer is not None:
        w.params["normalizer"] = args.normalizer
    batch = W.make_batch(w, seed=1000 + rank, device=dev)
    n_tok, V = batch["n_tok"], batch["V"]
    logits = batch["logits"]
    esz = logits.element_size()
    params = dict(batch["params"])
    params["kernel"] = {"auto": A.KERNEL_AUTO, "generic": A.KERNEL_GENERIC,
                        "cluster": A.KERNEL_CLUSTER, "rf": A.KERNEL_CLUSTER_RF,
                        "rf4": A.KERNEL_CLUSTER_RF4}[args.kernel]
    call = A.LossCall(logits, batch["target_ids"], batch["behave_lp"], batch["prox_lp"],
                      batch["step_off"], batch["traj_off"], batch["group_off"],
                      batch["rewards"], want=("err_word",), **params)
    kern = A.select_kernel(V, batch["ld"], logits.dtype) if args.kernel == "auto" else params["kernel"]
    stream = torch.cuda.current_stream(dev)

    # ---- device-resident leg
    for _ in range(args.warmup):
        call.run()
    torch.cuda.synchronize(dev)
    assert int(call.out["err_word"][0]) == 0
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(args.steps)]
    for a, b in evs:           # give every event a handle before the timed region
        a.record(stream)
        b.record(stream)
    t_beg, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(dev)
    barrier(world)
    with ClockSampler(local_rank) as clk:
        t_beg.record(stream)
        for a, b in evs:
            call.run(row_events=(a, b))
        t_end.record(stream)
        torch.cuda.synchronize(dev)
    barrier(world)
    local_ms = t_beg.elapsed_time(t_end)
    row_ms = [a.elapsed_time(b) for a, b in evs]
    total_ms, total_tok = aggregate(local_ms, n_tok * args.steps, world, dev)
    ms_per_step = total_ms / args.steps
    value = total_tok / (total_ms / 1e3)
    loss = float(call.out["loss"][0])
    clips = int(call.out["clip_count"][0])

    # ---- roofline of the dominant kernel (this rank's)
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        with open(peaks_path) as f:
            peak, peak_src = float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    else:
        peak, peak_src = 6650.0, "B200_PROFILING.md fallback (of fallback)"
    alg_bytes = algorithmic_bytes_per_token(V, esz) * n_tok
    row_avg_ms = sum(row_ms) / len(row_ms)
    achieved = alg_bytes / (row_avg_ms / 1e3) / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": load_traffic(args.config),
                "kernel": {A.KERNEL_GENERIC: "rows_generic_kernel",
                           A.KERNEL_CLUSTER: "rows_cluster_kernel",
                           A.KERNEL_CLUSTER_RF: "rows_rf_kernel<NU,2>",
                           A.KERNEL_CLUSTER_RF4: "rows_rf_kernel<NU,4>"}[kern],
                "kernel_ms": row_avg_ms, "kernel_share_of_step": row_avg_ms / (local_ms / args.steps),
                "algorithmic_bytes_per_launch": alg_bytes, "peak_source": peak_src}

    # ---- end-to-end leg: host buffers through awr_loss_fwd_bwd_host
    e2e = None
    if not args.no_e2e:
        e2e_steps = args.e2e_steps or args.steps
        host_in = {}
        for k in ("logits", "target_ids", "behave_lp", "prox_lp", "step_off", "traj_off",
                  "group_off", "rewards"):
            host_in[k] = torch.empty(batch[k].shape, dtype=batch[k].dtype,
                                     pin_memory=True).copy_(batch[k])
        del call, logits
        batch.pop("logits")
        torch.cuda.empty_cache()
        hparams = dict(params)
        hcall = A.HostLossCall(host_in["logits"], host_in["target_ids"], host_in["behave_lp"],
                               host_in["prox_lp"], host_in["step_off"], host_in["traj_off"],
                               host_in["group_off"], host_in["rewards"], device=dev, V=V,
                               **hparams)
        for _ in range(max(1, min(args.warmup, 2))):
            hcall.run()
        torch.cuda.synchronize(dev)
        barrier(world)
        t0 = time.perf_counter()
        e_beg, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e_beg.record(stream)
        for _ in range(e2e_steps):
            hcall.run()                 # returns once the results are in the host buffers
        e_end.record(stream)
        torch.cuda.synchronize(dev)
        wall_ms = (time.perf_counter() - t0) * 1e3
        barrier(world)
        # the host call synchronises internally on its own streams: wall clock is the honest
        # end-to-end time; the event pair on the caller's stream is recorded for reference
        e_ms, e_tok = aggregate(wall_ms, n_tok * e2e_steps, world, dev)
        assert int(hcall.out["err_word"][0]) == 0
        e_loss = float(hcall.out["loss"][0])
        e2e = {"value": e_tok / (e_ms / 1e3), "unit": UNIT,
               "h2d_bytes_per_step": int(hcall.h2d_bytes), "d2h_bytes_per_step": int(hcall.d2h_bytes),
               "steps": e2e_steps, "ms_per_step": e_ms / e2e_steps,
               "api": "awr_loss_fwd_bwd_host (pinned host buffers, 256 MB row panels)",
               "loss_matches_device_leg": e_loss == loss}

    # ---- CPU baseline: the oracle on a bounded sample (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        akw, host = oracle_sample(args.config, CPU_SAMPLE_TOK, seed=1234)
        dt, _ = time_oracle(akw)
        cpu = {"value": host["n_tok"] / dt, "unit": UNIT, "cores": host_threads_used(),
               "kind": "oracle", "seconds": dt,
               "sample": "config-%d laws cut to %d tokens, V=%d, one pass of "
                         "oracle.awr_loss_fwd_bwd (fp64 numpy)" % (args.config, host["n_tok"],
                                                                    host["V"])}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "bf16 in/out, f32 math" if esz == 2 else "f32",
                "data": "synthetic",
                "config": {"workload": ("BASELINE.json configs[%d] (%s)" if args.config < 5 else
                                        "not in BASELINE.json: workload %d (%s)") % (args.config, w.name),
                           "n_tok_per_gpu": n_tok, "V": V, "n_groups": w.n_groups,
                           "group_size": w.group_size, "normalizer":
                               "1/k" if params["normalizer"] == A.NORM_CONST_K else "1/|tau_i|",
                           "k_norm": params["k_norm"], "clip_eps": params["clip_eps"],
                           "stale_cap": params["stale_cap"],
                           "parallelism": "replicas only x%d" % world,
                           "l2": "inputs (%.1f GB/step) larger than L2, no flush" % (alg_bytes / 1e9)},
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
                "gpu_launches": A.launches_per_call() * args.steps,
                "clocks": clk.summary(), "loss": loss, "clip_count": clips}
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return 0


def run_head(args):
    """--config 4: the fused LM-head variant (a5).  A step = one awr_loss_fwd_bwd_fused_head call
    (hidden [32,768, 2048] and W_head [2048, 151,936] in, loss / dhidden / dw_head out).  The
    roofline is the tensor pipe: algorithmic flops 6 K V per token (logits, dH, dW).  The default
    mode executes exactly those (the fp32 logits of one row panel are kept for a streaming dS
    pass); --head-kernel 1cta / 2cta recompute the logits tile instead (8 K V executed)."""
    import torch

    import paper_2606_05597_b200 as A
    from gen import workloads as W

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a B200: there is no CPU path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    init_dist("nccl")
    over = {}
    if args.n_tok:
        over["n_tok"] = args.n_tok
    w = W.workload(4, **over)
    batch = W.make_batch(w, seed=1000 + rank, device=dev)
    n_tok, V, K = batch["n_tok"], batch["V"], w.hidden
    call = A.HeadLossCall(batch["hidden"], batch["w_head"], batch["target_ids"],
                          batch["behave_lp"], batch["prox_lp"], batch["step_off"],
                          batch["traj_off"], batch["group_off"], batch["rewards"],
                          want=("err_word",),
                          **dict(batch["params"], kernel={"auto": A.KERNEL_AUTO, "1cta": A.KERNEL_HEAD_1CTA,
                                                          "2cta": A.KERNEL_HEAD_2CTA,
                                                          "stored": A.KERNEL_HEAD_2CTA_STORED}[args.head_kernel]))
    stream = torch.cuda.current_stream(dev)
    for _ in range(args.warmup):
        call.run()
    torch.cuda.synchronize(dev)
    assert int(call.out["err_word"][0]) == 0
    t_beg, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(world)
    with ClockSampler(local_rank) as clk:
        t_beg.record(stream)
        for _ in range(args.steps):
            call.run()
        t_end.record(stream)
        torch.cuda.synchronize(dev)
    barrier(world)
    local_ms = t_beg.elapsed_time(t_end)
    total_ms, total_tok = aggregate(local_ms, n_tok * args.steps, world, dev)
    ms_per_step = total_ms / args.steps
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        with open(peaks_path) as f:
            peak = float(json.load(f)["bf16_tflops_sustained"])
        peak_src = "MEASURED_PEAKS.json bf16_tflops_sustained (of measured)"
    else:
        peak, peak_src = 1400.0, "B200_PROFILING.md fallback (of fallback)"
    # ---- end-to-end leg: pinned host hidden / W_head in, dhidden / dw_head / loss out, through
    # the public binding; copies inside the timed region, every step
    e2e = None
    if not args.no_e2e:
        e2e_steps = args.e2e_steps or args.steps
        hin = {k: torch.empty(batch[k].shape, dtype=batch[k].dtype, pin_memory=True).copy_(batch[k])
               for k in ("hidden", "w_head", "target_ids", "behave_lp", "prox_lp")}
        hout = {k: torch.empty(call.out[k].shape, dtype=call.out[k].dtype, pin_memory=True)
                for k in ("dhidden", "dw_head", "loss", "token_lp", "clip_count")}
        h2d = sum(t.numel() * t.element_size() for t in hin.values())
        d2h = sum(t.numel() * t.element_size() for t in hout.values())

        def e2e_step():
            for k, t in hin.items():
                batch[k].copy_(t, non_blocking=True)
            call.run()
            for k, t in hout.items():
                t.copy_(call.out[k], non_blocking=True)

        e2e_step()
        torch.cuda.synchronize(dev)
        barrier(world)
        e_beg, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e_beg.record(stream)
        for _ in range(e2e_steps):
            e2e_step()
        e_end.record(stream)
        torch.cuda.synchronize(dev)
        barrier(world)
        e_ms, e_tok = aggregate(e_beg.elapsed_time(e_end), n_tok * e2e_steps, world, dev)
        e2e = {"value": e_tok / (e_ms / 1e3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "steps": e2e_steps, "ms_per_step": e_ms / e2e_steps,
               "api": "awr_loss_fwd_bwd_fused_head on device buffers refilled from pinned host "
                      "memory each step; dhidden, dw_head, loss, token_lp copied back",
               "loss_matches_device_leg": float(hout["loss"][0]) == float(call.out["loss"][0])}

    # ---- CPU baseline: the fused-head oracle on a bounded sample (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        from oracle import awr_oracle as O
        ws = W.workload(4, n_groups=2, group_size=8, n_tok=HEAD_CPU_SAMPLE_TOK)
        host = W.to_host(W.make_batch(ws, seed=1234, device="cpu"))
        oargs, okw = W.oracle_args(host)
        t0 = time.perf_counter()
        O.awr_loss_fwd_bwd_fused_head(*oargs, **okw)
        dt = time.perf_counter() - t0
        cpu = {"value": host["n_tok"] / dt, "unit": UNIT, "cores": len(os.sched_getaffinity(0)),
               "kind": "oracle", "seconds": dt,
               "sample": "config-4 laws cut to %d tokens, K=%d, V=%d, one pass of "
                         "oracle.awr_loss_fwd_bwd_fused_head (fp64 numpy; its three matmuls use "
                         "the BLAS threads numpy was built with)" % (host["n_tok"], K, V)}

    alg_flops = 6.0 * K * V * n_tok
    exe_ratio = 1.0 if args.head_kernel in ("auto", "stored") else 8.0 / 6.0
    achieved = alg_flops / (local_ms / args.steps / 1e3) / 1e12
    if rank == 0:
        line = {"metric": METRIC + " (fused LM-head variant)", "value": total_tok / (total_ms / 1e3),
                "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "bf16 x bf16 -> f32 (TMEM)", "data": "synthetic",
                "config": {"workload": "BASELINE.json configs[4] (%s)" % w.name,
                           "n_tok_per_gpu": n_tok, "V": V, "K": K, "w_layout": "K_BY_V",
                           "parallelism": "replicas only x%d" % world,
                           "l2": "W_head (622 MB) + dS panels (1.4-2.9 GB) larger than L2, no flush"},
                "roofline": {"bound": "tensor", "achieved": achieved, "peak": peak,
                             "unit": "TFLOP/s", "frac": achieved / peak, "traffic": None,
                             "kernel": "head_gemm_kernel<epi, %s> (%s), whole step" % (
                                 "1" if args.head_kernel == "1cta" else "2",
                                 "3 GEMMs + dS streaming pass per panel" if exe_ratio == 1.0
                                 else "4 GEMMs, logits recomputed"),
                             "algorithmic_flops_per_step": alg_flops,
                             "executed_flops_per_step": alg_flops * exe_ratio,
                             "executed_tflops": achieved * exe_ratio, "peak_source": peak_src},
                "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": call.launches * args.steps,
                "clocks": clk.summary(), "loss": float(call.out["loss"][0]),
                "clip_count": int(call.out["clip_count"][0])}
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return 0


def load_traffic(cfg: int):
    """dram bytes (read + write) per launch of the row kernel from the committed `ncu --set full`
    capture (profiles/r1_traffic.txt, JSON text written by hand from the capture named there), or null."""
    p = os.path.join(ROOT, "profiles", "r1_traffic.txt")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        d = json.load(f)
    return d.get("config%d" % cfg, {}).get("dram_bytes_per_launch")


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=1, choices=[0, 1, 2, 3, 4, 5],
                    help="BASELINE.json configs[i]; 5 = the Thinking-variant shapes (SURVEY 8(f) rank 4)")
    ap.add_argument("--n-tok", type=int, default=0, help="override the config's token count")
    ap.add_argument("--normalizer", type=int, default=None, choices=[0, 1])
    ap.add_argument("--kernel", default="auto", choices=["auto", "generic", "cluster", "rf", "rf4"])
    ap.add_argument("--head-kernel", default="auto", choices=["auto", "1cta", "2cta", "stored"],
                    help="config 4: tcgen05 shape / backward mode (auto = stored: CTA pairs, fp32 "
                         "logits of one row panel kept for the dS pass; 1cta / 2cta recompute)")
    ap.add_argument("--e2e-steps", type=int, default=0, help="default: --steps")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args(argv)
    if args.warmup < 3 and args.impl == "cuda":
        args.warmup = 3                   # timing rule: at least 3 warm-up steps
    _, _, world = dist_env()
    if world != args.gpus and world == 1 and args.gpus > 1:
        raise SystemExit("launch N > 1 with: python -m torch.distributed.run --nnodes=1 "
                         "--nproc-per-node N --master-addr 127.0.0.1 bench.py --gpus N ...")
    if args.impl == "reference":
        return run_reference(args)
    if args.config == 4:
        return run_head(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
