"""Seeded synthetic inputs shaped like the paper's training batches (BASELINE.json configs 0-4).

This module serves BOTH the oracle-side tests and the CUDA-side tests / bench as a source of
*bytes*; it holds none of the method's arithmetic (no advantage, ratio, clip, normalizer, loss
or gradient).  The only numerical routine it calls is the library ``torch.log_softmax`` that
the recipe itself prescribes for drawing behave / prox log-probs ("perturbed log-softmax",
BASELINE.json configs 0-2).

The paper measures on WebGym with Qwen3-VL-8B; neither is available here, so
these inputs stand in for them using only the statistics the paper prints: 30-40 % success
(PAPER.md:122), failures ~12.5 steps vs successes ~5.1, G = 8 rollouts per task
and 16 groups per batch, a few hundred response tokens per step
(PAPER.md:106).  Recipe and the readings chosen: DESIGN.md "Input recipe".

Determinism: structure arrays come from ``numpy.random.Generator(PCG64(seed))`` on the host;
per-token tensors from ``torch.Generator(device).manual_seed(seed * 2**20 + chunk)`` per
1,024-row chunk.  CPU and CUDA torch generators give different streams; any one test or bench
run draws its inputs once and hands the same bytes to both sides.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
import torch

NORM_CONST_K = 0
NORM_PER_TRAJ = 1

V_QWEN = 151_936        # BASELINE.json: metric is quoted at V = 151,936
CHUNK_ROWS = 1024
GUARD_BAND = 1e-4       # keep log r_t away from log(1 +- eps)


@dataclass
class Workload:
    """Shape + distribution parameters of one config (BASELINE.json ``configs[i]``)."""
    name: str
    n_groups: int
    group_size: int
    n_tok: int | None            # "cut to Ntok": rescale step lengths so the total is exact
    V: int
    dtype: torch.dtype
    logit_std: float
    target_boost: float
    lp_mode: str                 # "perturb" | "lag" | "drift"
    p_equal_groups: float = 0.0  # config 3: share of groups forced to all-equal rewards
    fixed: bool = False          # config 0: hand-written structure
    tok_lo: int = 32             # response tokens per step ~ U{tok_lo..tok_hi}
    tok_hi: int = 256
    horizon: int | None = None   # step cap of a trajectory (PAPER.md:73: 10 / 20 / 30; :321-331)
    hidden: int | None = None    # config 4
    params: dict = field(default_factory=dict)


def workload(cfg: int, **over) -> Workload:
    """The five BASELINE.json configs.  ``over`` shrinks a config for parity tests while
    keeping its laws (e.g. ``workload(1, n_groups=2, n_tok=300)``)."""
    base = dict(k_norm=10.0, clip_eps=0.2, stale_cap=0.0, normalizer=NORM_CONST_K, flags=0,
                loss_scale=1.0)
    if cfg == 0:
        w = Workload("config0_tiny", 1, 4, 256, 1024, torch.float32, 2.0, 0.0, "perturb",
                     fixed=True, params=dict(base, stale_cap=2.0))
    elif cfg == 1:
        w = Workload("config1_microbatch", 8, 8, 40_960, V_QWEN, torch.bfloat16, 3.0, 4.0,
                     "perturb", params=dict(base))
    elif cfg == 2:
        w = Workload("config2_large", 16, 16, 65_536, V_QWEN, torch.bfloat16, 3.0, 4.0, "lag",
                     params=dict(base))
    elif cfg == 3:
        w = Workload("config3_stress", 32, 16, 131_072, V_QWEN, torch.bfloat16, 3.0, 4.0,
                     "drift", p_equal_groups=0.25,
                     params=dict(base, stale_cap=2.0, normalizer=NORM_PER_TRAJ))
    elif cfg == 4:
        w = Workload("config4_fused_head", 16, 16, 32_768, V_QWEN, torch.bfloat16, 0.0, 0.0,
                     "lag", hidden=2048, params=dict(base))
    elif cfg == 5:
        # not a BASELINE.json config: SURVEY.md 8(f) rank 4, the Thinking-variant shapes
        # (400-900 response tokens per step) under the long horizons (:321-331)
        # 2 groups x 8 with uncut step lengths (~90k tokens, ~28 GB of logits): cutting 16 groups
        # to a token budget would shrink the very step lengths this workload is about
        w = Workload("next_thinking_shapes", 2, 8, None, V_QWEN, torch.bfloat16, 3.0, 4.0, "lag",
                     tok_lo=400, tok_hi=900, horizon=40, params=dict(base))
    else:
        raise ValueError(cfg)
    for k, v in over.items():
        if k in w.params:
            w.params[k] = v
        else:
            setattr(w, k, v)
    return w


# ------------------------------------------------------------------ structure (host, numpy)
def make_structure(w: Workload, seed: int):
    """step_off (token index), traj_off (step index), group_off (trajectory index), rewards,
    and a per-step policy-version lag in {0,1,2,3} (used by lp_mode == "lag")."""
    rng = np.random.Generator(np.random.PCG64(seed))
    if w.fixed:
        steps = np.array([2, 3, 5, 6], dtype=np.int64)
        rewards = np.array([1.0, 0.0, 0.0, 1.0], dtype=np.float32)
        tok_per_step = np.full(int(steps.sum()), 16, dtype=np.int64)
        group_off = np.array([0, 4], dtype=np.int32)
    else:
        n_traj = w.n_groups * w.group_size
        rewards = (rng.random(n_traj) < 0.4).astype(np.float32)
        if w.p_equal_groups > 0:
            forced = rng.random(w.n_groups) < w.p_equal_groups
            common = (rng.random(w.n_groups) < 0.4).astype(np.float32)
            for g in np.nonzero(forced)[0]:
                rewards[g * w.group_size:(g + 1) * w.group_size] = common[g]
        lam = np.where(rewards > 0, 4.1, 11.5)          # 1 + Poisson: means 5.1 / 12.5
        steps = 1 + rng.poisson(lam).astype(np.int64)
        if w.horizon is not None:
            steps = np.minimum(steps, w.horizon)
        tok_per_step = rng.integers(w.tok_lo, w.tok_hi + 1, size=int(steps.sum())).astype(np.int64)
        group_off = (np.arange(w.n_groups + 1) * w.group_size).astype(np.int32)
    if w.n_tok is not None and not w.fixed:
        # "cut to Ntok": keep every group / trajectory / step, rescale the step lengths
        total = int(tok_per_step.sum())
        scaled = np.maximum(1, (tok_per_step * w.n_tok) // total)
        diff = w.n_tok - int(scaled.sum())
        if diff > 0:
            q, r = divmod(diff, scaled.size)
            scaled += q
            scaled[:r] += 1
        elif diff < 0:
            for i in range(scaled.size):        # only when min-1 clamping overshoots
                take = min(int(scaled[i]) - 1, -diff)
                scaled[i] -= take
                diff += take
                if diff == 0:
                    break
        tok_per_step = scaled
    step_off = np.concatenate([[0], np.cumsum(tok_per_step)]).astype(np.int32)
    traj_off = np.concatenate([[0], np.cumsum(steps)]).astype(np.int32)
    lag_step = rng.integers(0, 4, size=int(steps.sum())).astype(np.int64)
    return dict(step_off=step_off, traj_off=traj_off, group_off=group_off, rewards=rewards,
                lag_step=lag_step, n_tok=int(step_off[-1]))


# ------------------------------------------------------------------ per-token tensors (torch)
def _guard(lp, q, eps, gen, sigma):
    """Redraw q for tokens whose log r = lp - q is within GUARD_BAND of log(1 +- eps)."""
    lo, hi = math.log1p(-eps), math.log1p(eps)
    for _ in range(64):
        lr = lp - q
        bad = ((lr - lo).abs() < GUARD_BAND) | ((lr - hi).abs() < GUARD_BAND)
        if not bool(bad.any()):
            break
        fresh = torch.randn(q.shape, generator=gen, device=q.device, dtype=torch.float32)
        q = torch.where(bad, lp + max(sigma, 0.02) * fresh, q)
    return q


def make_batch(w: Workload, seed: int, device="cpu", ld: int | None = None, guard=True,
               masked_frac: float = 0.0):
    """Draw one batch.  Returns a dict of torch tensors on ``device`` plus ``params``.

    logits [n_tok, ld] (columns >= V hold a large sentinel that a correct kernel never
    reads), target_ids int32, behave_lp / prox_lp f32, offsets int32, rewards f32.
    For config 4 ``hidden`` [n_tok, K] and ``w_head`` [K, V] replace ``logits``."""
    st = make_structure(w, seed)
    n_tok, V = st["n_tok"], w.V
    dev = torch.device(device)
    eps = float(w.params["clip_eps"])
    ld = V if ld is None else ld
    assert ld >= V
    fused = w.hidden is not None
    ids = torch.empty(n_tok, dtype=torch.int32, device=dev)
    b = torch.empty(n_tok, dtype=torch.float32, device=dev)
    q = torch.empty(n_tok, dtype=torch.float32, device=dev)
    tok_step = torch.from_numpy(
        np.repeat(np.arange(st["step_off"].size - 1), np.diff(st["step_off"]))).to(dev)
    lag_tok = torch.from_numpy(st["lag_step"]).to(dev)[tok_step].to(torch.float32)
    if fused:
        g0 = torch.Generator(dev).manual_seed(seed * 2 ** 20 + 2 ** 19)
        H = torch.randn(n_tok, w.hidden, generator=g0, device=dev).to(torch.bfloat16)
        Wh = (0.02 * torch.randn(w.hidden, V, generator=g0, device=dev)).to(torch.bfloat16)
        logits = None
    else:
        logits = torch.empty(n_tok, ld, dtype=w.dtype, device=dev)
        if ld > V:
            logits[:, V:] = 3.0e4
    prev_tf32 = torch.backends.cuda.matmul.allow_tf32
    torch.backends.cuda.matmul.allow_tf32 = False
    try:
        for c, lo in enumerate(range(0, n_tok, CHUNK_ROWS)):
            hi = min(n_tok, lo + CHUNK_ROWS)
            n = hi - lo
            g = torch.Generator(dev).manual_seed(seed * 2 ** 20 + c)
            y = torch.randint(0, V, (n,), generator=g, device=dev)
            ar = torch.arange(n, device=dev)
            if fused:
                zf = H[lo:hi].float() @ Wh.float()
            else:
                z = torch.randn(n, V, generator=g, device=dev) * w.logit_std
                z[ar, y] += w.target_boost
                logits[lo:hi, :V] = z.to(w.dtype)
                zf = logits[lo:hi, :V].float()        # the already-rounded values
                del z
            lp = torch.log_softmax(zf, dim=1)[ar, y]
            if w.lp_mode == "perturb":
                nb = torch.randn(n, V, generator=g, device=dev) * 0.05
                bb = torch.log_softmax(zf + nb, dim=1)[ar, y]
                nb = torch.randn(n, V, generator=g, device=dev) * 0.02
                qq = torch.log_softmax(zf + nb, dim=1)[ar, y]
                del nb
                sig = 0.02
            elif w.lp_mode == "lag":
                nb = torch.randn(n, V, generator=g, device=dev) * 0.02
                qq = torch.log_softmax(zf + nb, dim=1)[ar, y]
                del nb
                bb = qq + 0.05 * lag_tok[lo:hi] * torch.randn(n, generator=g, device=dev)
                sig = 0.02
            elif w.lp_mode == "drift":
                qq = lp + 0.3 * torch.randn(n, generator=g, device=dev)
                bb = None
                sig = 0.3
            else:
                raise ValueError(w.lp_mode)
            if guard:
                q_new = _guard(lp, qq, eps, g, sig)
                if w.lp_mode == "lag":
                    bb = bb + (q_new - qq)            # keep b - q as drawn
                qq = q_new
            if w.lp_mode == "drift":
                bb = qq + 0.3 * torch.randn(n, generator=g, device=dev)
            ids[lo:hi] = y.to(torch.int32)
            b[lo:hi] = bb
            q[lo:hi] = qq
            del zf
    finally:
        torch.backends.cuda.matmul.allow_tf32 = prev_tf32
    if masked_frac > 0:
        gm = torch.Generator(dev).manual_seed(seed * 2 ** 20 + 2 ** 19 + 1)
        m = torch.rand(n_tok, generator=gm, device=dev) < masked_frac
        ids = torch.where(m, torch.full_like(ids, -1), ids)
    out = dict(n_tok=n_tok, V=V, ld=ld, target_ids=ids, behave_lp=b, prox_lp=q,
               step_off=torch.from_numpy(st["step_off"]).to(dev),
               traj_off=torch.from_numpy(st["traj_off"]).to(dev),
               group_off=torch.from_numpy(st["group_off"]).to(dev),
               rewards=torch.from_numpy(st["rewards"]).to(dev),
               params=dict(w.params), name=w.name)
    if fused:
        out.update(hidden=H, w_head=Wh)
    else:
        out.update(logits=logits)
    return out


def to_host(batch: dict) -> dict:
    """Exact host copies as numpy arrays (bf16 widened to float32, which is exact)."""
    out = {}
    for k, v in batch.items():
        if torch.is_tensor(v):
            t = v.detach().cpu()
            if t.dtype == torch.bfloat16:
                t = t.float()
            out[k] = t.numpy()
        else:
            out[k] = v
    if "logits" in out:
        out["logits"] = out["logits"][:, :batch["V"]]
    return out


def oracle_args(host: dict) -> tuple[tuple, dict]:
    """Positional / keyword arguments in the order every loss entry point takes them."""
    first = (host["hidden"], host["w_head"]) if "hidden" in host else (host["logits"],)
    args = first + (host["target_ids"], host["behave_lp"], host["prox_lp"], host["step_off"],
                    host["traj_off"], host["group_off"], host["rewards"])
    return args, dict(host["params"])
