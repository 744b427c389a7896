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
  cpu_baseline  the fp64 oracle (oracle/, as it stands) on the host cores, bounded sample: the
                rows split over one worker thread per core of the box (numpy releases the GIL;
                fixed-order final sum), the core count stated, a 1-thread figure beside it
  others        (N = 1, default config only) the same measurement for the other BASELINE.json
                configs and for the forward-only path, each with its own roofline and clocks:
                config 2 under 1/k and under 1/|tau_i|, config 3 into a separate gradient buffer and
                in place, config 4 (fused LM head, tensor roofline), awr_loss_fwd on config 1
  --impl reference   times the oracle alone (this tier's reference arm)
  --regimes [--kernel rfs|rfs_late]   diagnostic, its own JSON object: per-call kernel times of
                config 1 against the board's clock state
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
CPU_ROWS_PER_CORE = 512    # rows of the bounded oracle sample per host core (a few seconds of work on
CPU_MAX_ROWS = 24576       # ... capped (the sample batch lives in host memory: 3.7 GB of bf16 values
                           # widened to fp32 at the cap)
CPU_1T_ROWS = 1024         # rows of the 1-thread figure
OTHER_STEPS = 5            # timed steps of every "others" leg (3 warm-ups)
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


def host_cores() -> int:
    return len(os.sched_getaffinity(0))


def time_oracle_rows(host, n_threads: int):
    """The oracle's own per-row functions (unchanged: O.token_logprob, O.token_terms,
    O.dlogits_rows, i.e. steps O3..O8 of oracle/awr_oracle.py in the order its awr_loss_fwd_bwd
    chains them) over all rows of `host`, the rows split into contiguous chunks over `n_threads`
    worker threads (numpy releases the GIL inside exp / sum), then the fixed-order fp64 sum of
    the per-token terms in token order (O7).  Returns (seconds, loss)."""
    import numpy as np
    from concurrent.futures import ThreadPoolExecutor
    from oracle import awr_oracle as O
    p = host["params"]
    z, y = host["logits"], host["target_ids"].astype(np.int64)
    n_tok, V = z.shape
    t0 = time.perf_counter()
    seg = O.segment_expand(host["step_off"], host["traj_off"], host["group_off"])
    adv = O.group_advantage(host["rewards"], host["group_off"], p.get("flags", 0))
    scale = O.traj_scale(host["step_off"], host["traj_off"], host["group_off"], p["k_norm"],
                         p["normalizer"], p.get("loss_scale", 1.0), host["rewards"], p.get("flags", 0))
    tt = seg["tok_traj"]
    term = np.zeros(n_tok)
    rows_per = max(1, min(64, -(-n_tok // n_threads)))

    def work(lo):
        hi = min(n_tok, lo + rows_per)
        lse, lp, zy = O.token_logprob(z[lo:hi], y[lo:hi])
        valid = (y[lo:hi] >= 0) & (y[lo:hi] < V)
        t, c, trig, r, w = O.token_terms(lp, host["prox_lp"][lo:hi], host["behave_lp"][lo:hi],
                                         adv[tt[lo:hi]], scale[tt[lo:hi]], p["clip_eps"],
                                         p["stale_cap"], valid, p.get("dual_clip_c", 0.0))
        g = O.dlogits_rows(z[lo:hi], y[lo:hi], lse, c)
        term[lo:hi] = t
        return float(g[0, 0])

    if n_threads == 1:
        for lo in range(0, n_tok, rows_per):
            work(lo)
    else:
        with ThreadPoolExecutor(n_threads) as ex:
            list(ex.map(work, range(0, n_tok, rows_per)))
    loss = 0.0
    for t in range(n_tok):
        loss -= term[t]
    return time.perf_counter() - t0, loss


def cpu_baseline_rows(cfg: int):
    """cpu_baseline of the logits path: all host cores, and one thread beside it."""
    cores = host_cores()
    n = min(CPU_MAX_ROWS, CPU_ROWS_PER_CORE * cores)
    _, host = oracle_sample(cfg, n, seed=1234)
    dt, _ = time_oracle_rows(host, cores)
    n1 = min(CPU_1T_ROWS, host["n_tok"])
    host1 = dict(host)
    for k in ("logits", "target_ids", "behave_lp", "prox_lp"):
        host1[k] = host[k][:n1]
    so = host["step_off"]
    keep = int((so <= n1).sum())                 # whole steps inside the first n1 rows
    host1 = None if keep < 2 else host1
    dt1 = None
    if host1 is not None:
        _, h1 = oracle_sample(cfg, n1, seed=1234)
        dt1, _ = time_oracle_rows(h1, 1)
        n1 = h1["n_tok"]
    return {"value": host["n_tok"] / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "seconds": dt,
            "sample": "config-%d laws cut to %d tokens, V=%d; oracle steps O1..O8 (fp64 numpy) with "
                      "the rows split over %d worker threads, fixed-order sum" % (
                          cfg, host["n_tok"], host["V"], cores),
            "one_thread": None if dt1 is None else {"value": n1 / dt1, "unit": UNIT, "cores": 1,
                                                    "seconds": dt1, "rows": n1}}


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
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1,
                             "kind": "oracle", "sample": sample + " (one thread: oracle.awr_loss_fwd_bwd "
                                                                  "as it stands)"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------- measurement helpers
def measured_peaks():
    """Roofline denominators: MEASURED_PEAKS.json (driver-written on this pool's B200s), else the
    fallback B200_PROFILING.md states."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return {"hbm": float(d["hbm_gbs"]), "tensor": float(d["bf16_tflops_sustained"]),
                "tensor_burst": float(d["bf16_tflops"]), "src": "MEASURED_PEAKS.json (of measured)"}
    return {"hbm": 6650.0, "tensor": 1400.0, "tensor_burst": 1590.0,
            "src": "B200_PROFILING.md fallback (of fallback)"}


KERNEL_NAMES = {1: "rows_generic_kernel", 2: "rows_cluster_kernel", 3: "rows_rf_kernel<NU,2>",
                4: "rows_rf_kernel<NU,4>", 8: "rows_fwd_kernel", 10: "rows_rfs_kernel<NU>",
                12: "rows_rfs_kernel<NU> (late statistics)"}


def load_traffic(leg: str):
    """dram bytes (read + write) per launch of the leg's dominant kernel from a committed
    `ncu --set full` capture: profiles/r2_traffic.txt (JSON text; every entry names its capture).
    Returns (bytes, capture) or (None, reason) - never a number for a leg it was not taken on."""
    p = os.path.join(ROOT, "profiles", "r2_traffic.txt")
    if not os.path.exists(p):
        return None, "no ncu --set full capture committed"
    with open(p) as f:
        d = json.load(f)
    e = d.get(leg)
    if not e:
        return None, "no ncu --set full capture of this leg"
    return e.get("dram_bytes_per_launch"), e.get("capture")


def rows_leg(torch, A, W, dev, cfg, steps, warmup, *, seed=1000, normalizer=None, in_place=False,
             backward=True, kernel=None, n_tok=None, leg="", batch=None, rank_barrier=None):
    """One timed leg of the logits path: `steps` awr_loss_fwd_bwd (or awr_loss_fwd) calls on a
    device-resident batch of BASELINE.json configs[cfg]; CUDA events on the launching stream around
    the region and (through awr_outputs.ev_row_*) around the row kernel of every step; NVML clock
    samples during the region.  Returns the leg's numbers and the batch (for reuse)."""
    over = {} if not n_tok else dict(n_tok=n_tok)
    w = W.workload(cfg, **over)
    if normalizer is not None:
        w.params["normalizer"] = normalizer
    if batch is None:
        batch = W.make_batch(w, seed=seed, device=dev)
    n, V = batch["n_tok"], batch["V"]
    logits = batch["logits"]
    esz = logits.element_size()
    params = dict(batch["params"])
    params["normalizer"] = w.params["normalizer"]
    if kernel is not None:
        params["kernel"] = kernel
    kw = dict(dlogits=logits) if (in_place and backward) else {}
    call = A.LossCall(logits, batch["target_ids"], batch["behave_lp"], batch["prox_lp"],
                      batch["step_off"], batch["traj_off"], batch["group_off"], batch["rewards"],
                      want=("err_word",), backward=backward, **kw, **params)
    stream = torch.cuda.current_stream(dev)
    for _ in range(max(3, warmup)):
        call.run()
    torch.cuda.synchronize(dev)
    assert int(call.out["err_word"][0]) == 0
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(steps)]
    for a, b in evs:           # give every event a handle before the timed region
        a.record(stream)
        b.record(stream)
    t_beg, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(dev)
    if rank_barrier:
        rank_barrier()
    with ClockSampler(dev.index or 0) as clk:
        t_beg.record(stream)
        for ev in evs:
            call.run(row_events=ev)
        t_end.record(stream)
        torch.cuda.synchronize(dev)
    if rank_barrier:
        rank_barrier()
    local_ms = t_beg.elapsed_time(t_end)
    row_ms = sum(a.elapsed_time(b) for a, b in evs) / len(evs)
    peaks = measured_peaks()
    per_tok = algorithmic_bytes_per_token(V, esz) if backward else V * esz + 24
    alg_bytes = per_tok * n
    achieved = alg_bytes / (row_ms / 1e3) / 1e9
    if kernel in (None, A.KERNEL_AUTO):
        kern = A.KERNEL_FWD_STREAM if (not backward and A.select_kernel(V, batch["ld"], logits.dtype)
                                       != A.KERNEL_GENERIC) else A.select_kernel(V, batch["ld"], logits.dtype)
    else:
        kern = kernel
    traffic, capture = load_traffic(leg)
    res = {"ms_per_step": local_ms / steps, "tokens_per_s": n * steps / (local_ms / 1e3),
           "n_tok": n, "V": V, "steps": steps,
           "normalizer": "1/k" if params["normalizer"] == A.NORM_CONST_K else "1/|tau_i|",
           "in_place": bool(in_place and backward), "entry": call._name,
           "roofline": {"bound": "hbm", "achieved": achieved, "peak": peaks["hbm"], "unit": "GB/s",
                        "frac": achieved / peaks["hbm"], "frac_of_8tbs_data_sheet": achieved / 8000.0,
                        "traffic": traffic, "traffic_source": capture,
                        "kernel": KERNEL_NAMES.get(kern, str(kern)), "kernel_ms": row_ms,
                        "kernel_share_of_step": row_ms / (local_ms / steps),
                        "algorithmic_bytes_per_launch": alg_bytes, "peak_source": peaks["src"]},
           "clocks": clk.summary(), "loss": float(call.out["loss"][0]),
           "clip_count": int(call.out["clip_count"][0]),
           "gpu_launches": A.launches_per_call() * steps}
    return res, batch, call, local_ms


def head_leg(torch, A, W, dev, steps, warmup, *, seed=1000, head_kernel="auto", n_tok=None,
             rank_barrier=None):
    """One timed leg of the fused LM head (BASELINE.json configs[4]): tensor roofline over the
    whole step (6 K V algorithmic flops per token: logits, dhidden, dw_head)."""
    over = {} if not n_tok else dict(n_tok=n_tok)
    w = W.workload(4, **over)
    batch = W.make_batch(w, seed=seed, device=dev)
    n, V, K = batch["n_tok"], batch["V"], w.hidden
    kcode = {"auto": A.KERNEL_AUTO, "1cta": A.KERNEL_HEAD_1CTA, "2cta": A.KERNEL_HEAD_2CTA,
             "stored": A.KERNEL_HEAD_2CTA_STORED, "e16": A.KERNEL_HEAD_2CTA_E16,
             "rowref": A.KERNEL_HEAD_2CTA_ROWREF}[head_kernel]
    call = A.HeadLossCall(batch["hidden"], batch["w_head"], batch["target_ids"], batch["behave_lp"],
                          batch["prox_lp"], batch["step_off"], batch["traj_off"], batch["group_off"],
                          batch["rewards"], want=("err_word",), **dict(batch["params"], kernel=kcode))
    stream = torch.cuda.current_stream(dev)
    for _ in range(max(3, warmup)):
        call.run()
    torch.cuda.synchronize(dev)
    assert int(call.out["err_word"][0]) == 0
    t_beg, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if rank_barrier:
        rank_barrier()
    with ClockSampler(dev.index or 0) as clk:
        t_beg.record(stream)
        for _ in range(steps):
            call.run()
        t_end.record(stream)
        torch.cuda.synchronize(dev)
    if rank_barrier:
        rank_barrier()
    local_ms = t_beg.elapsed_time(t_end)
    peaks = measured_peaks()
    alg_flops = 6.0 * K * V * n
    exe_ratio = 1.0 if head_kernel in ("auto", "stored", "e16", "rowref") else 8.0 / 6.0
    achieved = alg_flops / (local_ms / steps / 1e3) / 1e12
    res = {"ms_per_step": local_ms / steps, "tokens_per_s": n * steps / (local_ms / 1e3),
           "n_tok": n, "V": V, "K": K, "steps": steps, "entry": "awr_loss_fwd_bwd_fused_head",
           "workspace_bytes": int(call.ws_bytes),
           "roofline": {"bound": "tensor", "achieved": achieved, "peak": peaks["tensor"],
                        "unit": "TFLOP/s", "frac": achieved / peaks["tensor"], "traffic": None,
                        "traffic_source": "null: tensor-bound leg of several kernels; dram bytes per kernel "
                                          "of one panel are in profiles/r2_head.md",
                        "kernel": "head_gemm_kernel<epi, %s> (%s), whole step" % (
                            "1" if head_kernel == "1cta" else "2",
                            "4 GEMMs, logits recomputed" if exe_ratio != 1.0 else
                            ("3 GEMMs per panel, row-reference E, no dS pass" if head_kernel in ("auto", "rowref")
                             else "3 GEMMs + dS streaming pass per panel")),
                        "algorithmic_flops_per_step": alg_flops,
                        "executed_flops_per_step": alg_flops * exe_ratio,
                        "executed_tflops": achieved * exe_ratio,
                        "peak_source": peaks["src"] + ": bf16_tflops_sustained (a kernel timed "
                                                      "inside a long step)"},
           "clocks": clk.summary(), "loss": float(call.out["loss"][0]),
           "clip_count": int(call.out["clip_count"][0]), "gpu_launches": call.launches * steps}
    return res, batch, call, local_ms


def other_legs(torch, A, W, dev):
    """The "others" object of the default line (N = 1): every other BASELINE.json config and the
    forward-only entry, OTHER_STEPS timed steps each after 3 warm-ups, inputs resident in HBM."""
    out = {}

    def free():
        import gc
        gc.collect()
        torch.cuda.empty_cache()

    def leg(name, fn):
        try:
            out[name] = fn()
        except Exception as e:                   # a leg that cannot run says so; the line survives
            out[name] = {"error": repr(e)[:300]}
        free()

    def cfg1_fwd():
        r, b, c, _ = rows_leg(torch, A, W, dev, 1, OTHER_STEPS, 3, backward=False, leg="config1_fwd")
        return r

    def cfg2():
        r1, b, c, _ = rows_leg(torch, A, W, dev, 2, OTHER_STEPS, 3, normalizer=A.NORM_CONST_K, leg="config2")
        del c
        r2, b, c, _ = rows_leg(torch, A, W, dev, 2, OTHER_STEPS, 3, normalizer=A.NORM_PER_TRAJ, batch=b,
                               leg="config2")
        return r1, r2

    leg("config1_forward_only", cfg1_fwd)
    try:
        out["config2_norm_1_over_k"], out["config2_norm_1_over_tau"] = cfg2()
    except Exception as e:
        out["config2_norm_1_over_k"] = out["config2_norm_1_over_tau"] = {"error": repr(e)[:300]}
    free()

    def cfg3(in_place):
        r, b, c, _ = rows_leg(torch, A, W, dev, 3, OTHER_STEPS, 3, in_place=in_place, leg="config3")
        return r

    leg("config3_separate_buffer", lambda: cfg3(False))
    leg("config3_in_place", lambda: cfg3(True))
    leg("config4_fused_head", lambda: head_leg(torch, A, W, dev, OTHER_STEPS, 3)[0])
    return out


# ---------------------------------------------------------------------------- the CUDA arm
def run_cuda(args):
    import torch

    import paper_2606_05597_b200 as A
    from gen import workloads as W

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a B200: there is no CPU path (use --impl reference "
                         "for the oracle)")
    # ---- CPU baseline first (rank 0, N = 1 only): before the GPU holds tens of GB and while the
    # host cores are idle; the oracle on a bounded sample, rows over all cores + a 1-thread figure
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu = cpu_baseline_rows(args.config)
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    init_dist("nccl")

    kernel = {"auto": A.KERNEL_AUTO, "generic": A.KERNEL_GENERIC, "cluster": A.KERNEL_CLUSTER,
              "rf": A.KERNEL_CLUSTER_RF, "rf4": A.KERNEL_CLUSTER_RF4, "rfs": A.KERNEL_CLUSTER_RFS,
              "rfs_late": A.KERNEL_CLUSTER_RFS_LATE}[args.kernel]
    leg, batch, call, local_ms = rows_leg(torch, A, W, dev, args.config, args.steps, args.warmup,
                                          seed=1000 + rank, normalizer=args.normalizer, kernel=kernel,
                                          n_tok=args.n_tok or None, backward=not args.forward_only,
                                          leg=("config%d_fwd" if args.forward_only else "config%d") % args.config,
                                          rank_barrier=lambda: barrier(world))
    w = W.workload(args.config)
    n_tok, V = batch["n_tok"], batch["V"]
    params = dict(batch["params"])
    if args.normalizer is not None:
        params["normalizer"] = args.normalizer
    params["kernel"] = kernel
    esz = batch["logits"].element_size()
    total_ms, total_tok = aggregate(local_ms, n_tok * args.steps, world, dev)
    ms_per_step = total_ms / args.steps
    value = total_tok / (total_ms / 1e3)
    loss, clips = leg["loss"], leg["clip_count"]
    stream = torch.cuda.current_stream(dev)

    # ---- end-to-end leg: host buffers through awr_loss_fwd_bwd_host
    e2e = None
    if not args.no_e2e and not args.forward_only:
        e2e_steps = args.e2e_steps or args.steps
        host_in = {}
        for k in ("logits", "target_ids", "behave_lp", "prox_lp", "step_off", "traj_off",
                  "group_off", "rewards"):
            host_in[k] = torch.empty(batch[k].shape, dtype=batch[k].dtype,
                                     pin_memory=True).copy_(batch[k])
        del call
        batch.pop("logits")
        torch.cuda.empty_cache()
        hcall = A.HostLossCall(host_in["logits"], host_in["target_ids"], host_in["behave_lp"],
                               host_in["prox_lp"], host_in["step_off"], host_in["traj_off"],
                               host_in["group_off"], host_in["rewards"], device=dev, V=V,
                               **params)
        for _ in range(max(1, min(args.warmup, 2))):
            hcall.run()
        torch.cuda.synchronize(dev)
        barrier(world)
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            hcall.run()                 # returns once the results are in the host buffers
        torch.cuda.synchronize(dev)
        wall_ms = (time.perf_counter() - t0) * 1e3
        barrier(world)
        # the host call synchronises internally on its own streams: wall clock is the honest
        # end-to-end time
        e_ms, e_tok = aggregate(wall_ms, n_tok * e2e_steps, world, dev)
        assert int(hcall.out["err_word"][0]) == 0
        e_loss = float(hcall.out["loss"][0])
        e2e = {"value": e_tok / (e_ms / 1e3), "unit": UNIT,
               "h2d_bytes_per_step": int(hcall.h2d_bytes), "d2h_bytes_per_step": int(hcall.d2h_bytes),
               "steps": e2e_steps, "ms_per_step": e_ms / e2e_steps,
               "api": "awr_loss_fwd_bwd_host (pinned host buffers, 256 MB row panels)",
               "loss_matches_device_leg": e_loss == loss}
        del hcall, host_in
    else:
        del call
    batch.clear()
    import gc
    gc.collect()
    torch.cuda.empty_cache()

    # ---- the other configs and the forward-only entry (N = 1, default workload only)
    others = None
    if rank == 0 and world == 1 and args.config == 1 and not args.no_others and not args.n_tok \
            and not args.forward_only:
        others = other_legs(torch, A, W, dev)

    if rank == 0:
        line = {"metric": METRIC if not args.forward_only else "forward-only tokens/s at V=151,936 bf16",
                "value": value, "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "bf16 in/out, f32 math" if esz == 2 else "f32",
                "data": "synthetic",
                "config": {"workload": ("BASELINE.json configs[%d] (%s)" if args.config < 5 else
                                        "not in BASELINE.json: workload %d (%s)") % (args.config, w.name),
                           "n_tok_per_gpu": n_tok, "V": V, "n_groups": w.n_groups,
                           "group_size": w.group_size, "normalizer": leg["normalizer"],
                           "k_norm": params["k_norm"], "clip_eps": params["clip_eps"],
                           "stale_cap": params["stale_cap"],
                           "parallelism": "replicas only x%d" % world,
                           "l2": "inputs (%.1f GB/step) larger than L2, no flush" % (
                               leg["roofline"]["algorithmic_bytes_per_launch"] / 1e9)},
                "roofline": leg["roofline"], "cpu_baseline": cpu, "e2e": e2e,
                "gpu_launches": leg["gpu_launches"],
                "clocks": leg["clocks"], "loss": loss, "clip_count": clips, "others": others}
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return 0


def run_regimes(args):
    """--regimes: how the fwd+bwd row kernel of config 1 behaves as the board's clocks move (DESIGN.md
    section 4, "Clock regimes"; a diagnostic, not the bench line).  (a) `--steps` back-to-back calls
    from an idle board: kernel time of every call (events the call records around its row kernel)
    and an NVML trace of the SM clock; (b) three calls after each of six 0.25 s bursts of dense
    bf16 GEMMs (torch.matmul 8192^3 as the load generator): the state a training step leaves the
    board in.  Prints one JSON object."""
    import torch

    import paper_2606_05597_b200 as A
    from gen import workloads as W

    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    batch = W.make_batch(W.workload(1), seed=1000, device=dev)
    kern = {"auto": A.KERNEL_AUTO, "rfs": A.KERNEL_CLUSTER_RFS, "rfs_late": A.KERNEL_CLUSTER_RFS_LATE,
            "rf": A.KERNEL_CLUSTER_RF, "rf4": A.KERNEL_CLUSTER_RF4, "cluster": A.KERNEL_CLUSTER,
            "generic": A.KERNEL_GENERIC}[args.kernel]
    call = A.LossCall(batch["logits"], batch["target_ids"], batch["behave_lp"], batch["prox_lp"],
                      batch["step_off"], batch["traj_off"], batch["group_off"], batch["rewards"],
                      want=("err_word",), **dict(batch["params"], kernel=kern))
    stream = torch.cuda.current_stream(dev)

    def events(n):
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        for a, b in evs:
            a.record(stream)
            b.record(stream)
        return evs

    for _ in range(2):
        call.run()
    steps = max(20, args.steps)
    evs = events(steps)
    torch.cuda.synchronize(dev)
    time.sleep(1.0)                                  # idle board: boost clock
    trace = []
    with ClockSampler(dev.index or 0, period_s=0.001) as clk:
        clk.trace = trace
        t0 = time.perf_counter()
        for ev in evs:
            call.run(row_events=ev)
        torch.cuda.synchronize(dev)
        wall_ms = (time.perf_counter() - t0) * 1e3
    ms = [a.elapsed_time(b) for a, b in evs]
    n_sm = len(clk.sm)
    blocks = []
    for i in range(0, steps, 20):
        blk = ms[i:i + 20]
        lo, hi = i * n_sm // steps, max(i * n_sm // steps + 1, (i + len(blk)) * n_sm // steps)
        blocks.append({"calls": "%d-%d" % (i, i + len(blk) - 1), "kernel_ms_mean": round(sum(blk) / len(blk), 3),
                       "kernel_ms_min": round(min(blk), 3), "kernel_ms_max": round(max(blk), 3),
                       "sm_mhz_median": statistics.median(clk.sm[lo:hi]) if clk.sm else None})
    x = torch.randn(8192, 8192, device=dev, dtype=torch.bfloat16)
    y = torch.randn(8192, 8192, device=dev, dtype=torch.bfloat16)
    bursts = []
    with ClockSampler(dev.index or 0) as clk2:
        for _ in range(6):
            for _ in range(300):
                torch.matmul(x, y)
            evs = events(3)
            for ev in evs:
                call.run(row_events=ev)
            torch.cuda.synchronize(dev)
            bursts.append([round(a.elapsed_time(b), 3) for a, b in evs])
    assert int(call.out["err_word"][0]) == 0
    flat = [v for r in bursts[1:] for v in r]
    print(json.dumps({"regimes": {
        "workload": "BASELINE.json configs[1], awr_loss_fwd_bwd, kernel %s" % KERNEL_NAMES.get(
            kern if kern != A.KERNEL_AUTO else A.select_kernel(batch["V"], batch["ld"], batch["logits"].dtype)),
        "back_to_back": {"calls": steps, "wall_ms": round(wall_ms, 1), "by_20_calls": blocks,
                         "reasons": sorted(clk.reasons)},
        "between_gemm_bursts": {"kernel_ms": bursts, "mean_ms_after_first_burst": round(sum(flat) / len(flat), 3),
                                "clocks": clk2.summary()}}}), flush=True)
    return 0


def run_head(args):
    """--config 4: the fused LM-head variant (a5).  A step = one awr_loss_fwd_bwd_fused_head call
    (hidden [32,768, 2048] and W_head [2048, 151,936] in, loss / dhidden / dw_head out).  The
    roofline is the tensor pipe: algorithmic flops 6 K V per token (logits, dH, dW).  The default
    mode executes exactly those; --head-kernel 1cta / 2cta recompute the logits tile instead
    (8 K V executed)."""
    import torch

    import paper_2606_05597_b200 as A
    from gen import workloads as W

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a B200: there is no CPU path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    init_dist("nccl")
    leg, batch, call, local_ms = head_leg(torch, A, W, dev, args.steps, args.warmup, seed=1000 + rank,
                                          head_kernel=args.head_kernel, n_tok=args.n_tok or None,
                                          rank_barrier=lambda: barrier(world))
    w = W.workload(4)
    n_tok, V, K = leg["n_tok"], leg["V"], leg["K"]
    total_ms, total_tok = aggregate(local_ms, n_tok * args.steps, world, dev)
    ms_per_step = total_ms / args.steps
    stream = torch.cuda.current_stream(dev)
    # ---- end-to-end leg: pinned host hidden / W_head in, dhidden / dw_head / loss out, through
    # the C-ABI host entry (awr_loss_fwd_bwd_fused_head_host); copies inside the timed region
    e2e = None
    if not args.no_e2e:
        e2e_steps = args.e2e_steps or args.steps
        hin = {k: torch.empty(batch[k].shape, dtype=batch[k].dtype, pin_memory=True).copy_(batch[k])
               for k in ("hidden", "w_head", "target_ids", "behave_lp", "prox_lp", "step_off",
                         "traj_off", "group_off", "rewards")}
        dev_loss = float(call.out["loss"][0])
        hcall = A.HostHeadLossCall(hin["hidden"], hin["w_head"], hin["target_ids"], hin["behave_lp"],
                                   hin["prox_lp"], hin["step_off"], hin["traj_off"], hin["group_off"],
                                   hin["rewards"], device=dev, workspace=call.workspace,
                                   **dict(batch["params"], kernel=call.params.kernel))
        hcall.run()
        torch.cuda.synchronize(dev)
        barrier(world)
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            hcall.run()
        torch.cuda.synchronize(dev)
        wall_ms = (time.perf_counter() - t0) * 1e3
        barrier(world)
        e_ms, e_tok = aggregate(wall_ms, n_tok * e2e_steps, world, dev)
        e2e = {"value": e_tok / (e_ms / 1e3), "unit": UNIT, "h2d_bytes_per_step": int(hcall.h2d_bytes),
               "d2h_bytes_per_step": int(hcall.d2h_bytes), "steps": e2e_steps,
               "ms_per_step": e_ms / e2e_steps,
               "api": "awr_loss_fwd_bwd_fused_head_host (pinned host hidden / W_head in; dhidden, "
                      "dw_head, loss, token_lp back)",
               "loss_matches_device_leg": float(hcall.out["loss"][0]) == dev_loss}

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
        cpu = {"value": host["n_tok"] / dt, "unit": UNIT, "cores": host_cores(),
               "kind": "oracle", "seconds": dt,
               "sample": "config-4 laws cut to %d tokens, K=%d, V=%d, one pass of "
                         "oracle.awr_loss_fwd_bwd_fused_head (fp64 numpy; its three matmuls use "
                         "the BLAS threads numpy was built with, the rest one thread)" % (
                             host["n_tok"], K, V)}

    if rank == 0:
        line = {"metric": METRIC + " (fused LM-head variant)", "value": total_tok / (total_ms / 1e3),
                "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "bf16 x bf16 -> f32 (TMEM)", "data": "synthetic",
                "config": {"workload": "BASELINE.json configs[4] (%s)" % w.name,
                           "n_tok_per_gpu": n_tok, "V": V, "K": K, "w_layout": "K_BY_V",
                           "parallelism": "replicas only x%d" % world,
                           "workspace_bytes": leg["workspace_bytes"],
                           "l2": "W_head (622 MB) + the dS panel larger than L2, no flush"},
                "roofline": leg["roofline"],
                "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": leg["gpu_launches"],
                "clocks": leg["clocks"], "loss": leg["loss"], "clip_count": leg["clip_count"]}
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return 0


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
    ap.add_argument("--kernel", default="auto", choices=["auto", "generic", "cluster", "rf", "rf4", "rfs", "rfs_late"])
    ap.add_argument("--head-kernel", default="auto", choices=["auto", "1cta", "2cta", "stored", "e16", "rowref"],
                    help="config 4: tcgen05 shape / backward mode (auto = rowref: CTA pairs, bf16 exp(z - "
                         "row reference) of one row panel kept, no dS pass; e16: exp(z - tile max) + an "
                         "in-place dS pass; stored: fp32 logits panel; 1cta / 2cta recompute)")
    ap.add_argument("--e2e-steps", type=int, default=0, help="default: --steps")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--forward-only", action="store_true",
                    help="time awr_loss_fwd (PAPER.md:436 prox-lp recompute) instead of awr_loss_fwd_bwd")
    ap.add_argument("--no-others", action="store_true",
                    help="skip the legs for the other configs / the forward-only entry")
    ap.add_argument("--regimes", action="store_true",
                    help="diagnostic: per-call kernel times of config 1 against the board's clock state "
                         "(back to back from idle; between bursts of dense GEMMs); prints its own JSON object")
    args = ap.parse_args(argv)
    if args.regimes:
        return run_regimes(args)
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
