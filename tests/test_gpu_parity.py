"""GPU parity: the CUDA path (through the C ABI / binding) against the fp64 oracle on the same
seeded inputs, element by element.  Run on the B200 box: pytest -m gpu."""
import numpy as np
import pytest
import torch

import paper_2606_05597_b200 as A
from gen import workloads as W
from oracle import awr_oracle as O
import parity_util as P

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _require_gpu():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (run them with gpurun)")


@pytest.fixture(autouse=True, scope="module")
def _gpu():
    _require_gpu()
    assert torch.cuda.get_device_capability(0)[0] == 10, "sm_100 only"
    yield


# ------------------------------------------------------------------ config 0 (fp32, V = 1024)
@pytest.mark.parametrize("norm", [A.NORM_CONST_K, A.NORM_PER_TRAJ])
@pytest.mark.parametrize("over", [dict(), dict(clip_eps=0.01), dict(stale_cap=1.02),
                                  dict(k_norm=4.0), dict(flags=A.FLAG_SAMPLE_STD)])
def test_config0_tiny(norm, over):
    """BASELINE.json configs[0]: 1 group, k = 4, steps {2,3,5,6}, 16 tokens/step, fp32
    [256, 1024]; eps 0.2, cap 2.0, both normalizers; parity-only reruns."""
    w = W.workload(0, normalizer=norm, **over)
    batch = W.make_batch(w, seed=0, device=DEV)
    gpu, ora = P.full_check(batch)
    if over.get("clip_eps") == 0.01:
        assert ora["clip_count"] > 0


def test_config0_all_ratios_one():
    """P2/P3 on the GPU: b = q = l -> loss is exactly 0 in exact arithmetic, gradient is not."""
    w = W.workload(0)
    batch = W.make_batch(w, seed=0, device=DEV)
    lp = A.awr_loss_fwd(batch["logits"], batch["target_ids"], batch["behave_lp"],
                        batch["prox_lp"], batch["step_off"], batch["traj_off"],
                        batch["group_off"], batch["rewards"], **batch["params"])["token_lp"]
    batch["prox_lp"] = lp.clone()
    batch["behave_lp"] = lp.clone()
    gpu, ora = P.full_check(batch)
    assert int(gpu["clip_count"][0]) == 0
    assert abs(float(gpu["loss"][0])) < 1e-6
    assert float(gpu["dlogits"].abs().max()) > 1e-4


# ------------------------------------------------------------------ generic kernel, odd shapes
@pytest.mark.parametrize("V,ld,dtype", [(1003, 1008, torch.bfloat16), (4096, 4096, torch.bfloat16),
                                        (777, 780, torch.float32), (8, 8, torch.bfloat16),
                                        (5, 8, torch.float32)])
@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_generic_small(V, ld, dtype, cfg):
    w = W.workload(cfg, n_groups=5, group_size=4, n_tok=700, V=V, dtype=dtype)
    batch = W.make_batch(w, seed=11 + cfg, device=DEV, ld=ld, masked_frac=0.05)
    batch["params"]["kernel"] = A.KERNEL_GENERIC
    P.full_check(batch)
    P.full_check(batch, backward=False)


# ------------------------------------------------------------------ cluster kernel
CLUSTER_SHAPES = [(151_936, 151_936), (40_000, 40_008), (32_768, 32_768), (65_544, 65_560),
                  (131_072, 131_072)]


CLUSTER_KERNELS = [A.KERNEL_CLUSTER, A.KERNEL_CLUSTER_RF, A.KERNEL_CLUSTER_RF4, A.KERNEL_CLUSTER_RFS,
                   A.KERNEL_CLUSTER_RFS_LATE]


@pytest.mark.parametrize("kernel", CLUSTER_KERNELS)
@pytest.mark.parametrize("V,ld", CLUSTER_SHAPES)
def test_cluster_vs_oracle(V, ld, kernel):
    """bf16 rows resident in the shared memory (CLUSTER) or the register files (CLUSTER_RF) of a
    2-CTA cluster; 300+ rows = several rows per cluster plus a ragged tail; masked tokens,
    zero-advantage groups, clip triggers."""
    assert A.select_kernel(V, ld, torch.bfloat16) in CLUSTER_KERNELS
    w = W.workload(3, n_groups=6, group_size=4, n_tok=331, V=V)
    batch = W.make_batch(w, seed=5, device=DEV, ld=ld, masked_frac=0.04)
    batch["params"]["kernel"] = kernel
    gpu, ora = P.full_check(batch)
    assert ora["clip_count"] > 0 and (ora["coef"] == 0).sum() > ora["clip_count"]
    P.full_check(batch, backward=False)


# ------------------------------------------------------------------ forward-only streaming kernel
@pytest.mark.parametrize("V,ld,n_tok", [(151_936, 151_936, 331), (40_000, 40_008, 700), (32_768, 32_768, 150),
                                        (65_544, 65_560, 149), (16_384, 16_384, 300), (1000, 1000, 257),
                                        (8, 8, 40), (2048 * 8, 2048 * 8 + 8, 77), (163_840, 163_840, 60)])
@pytest.mark.parametrize("entropy", [False, True])
def test_forward_stream_kernel(V, ld, n_tok, entropy):
    """awr_loss_fwd's streaming kernel (the proximal log-prob recomputation): rows
    shorter than one 32 KB stage, exactly one / several stages, ragged last stages, more and fewer
    rows than CTAs, masked tokens, -inf logits, clip triggers and the dual clip; every per-token
    output against the oracle, the entropy within 1e-4."""
    w = W.workload(3, n_groups=6, group_size=4, n_tok=n_tok, V=V)
    batch = W.make_batch(w, seed=V % 97, device=DEV, ld=ld, masked_frac=0.04)
    z = batch["logits"]
    if V > 64:
        z[::3, 5:V:97] = float("-inf")
        ids = batch["target_ids"].long().clamp(min=0)
        ar = torch.arange(z.shape[0], device=DEV)
        z[ar, ids] = z[ar, ids].nan_to_num(neginf=0.0)
    params = dict(batch["params"], kernel=A.KERNEL_FWD_STREAM, dual_clip_c=3.0)
    want = A.OPTIONAL_OUTPUTS + (("token_entropy",) if entropy else ())
    out = A.awr_loss_fwd(z, batch["target_ids"], batch["behave_lp"], batch["prox_lp"], batch["step_off"],
                         batch["traj_off"], batch["group_off"], batch["rewards"], V=V, want=want, **params)
    torch.cuda.synchronize()
    ora = P.run_oracle(batch, want_dlogits=False, want_entropy=True, dual_clip_c=3.0)
    P.check_scalars(out, ora, label="forward stream V=%d" % V)
    if entropy:
        H = out["token_entropy"].cpu().numpy().astype(np.float64)
        assert np.isfinite(H).all() and np.abs(H - ora["token_entropy"]).max() <= 1e-4
        assert np.all(H[batch["target_ids"].cpu().numpy() < 0] == 0.0)
    # deterministic (static row schedule, fixed merge order)
    again = A.awr_loss_fwd(z, batch["target_ids"], batch["behave_lp"], batch["prox_lp"], batch["step_off"],
                           batch["traj_off"], batch["group_off"], batch["rewards"], V=V, want=want, **params)
    torch.cuda.synchronize()
    for k in out:
        assert torch.equal(out[k], again[k]), k


def test_forward_stream_is_the_auto_choice_and_refuses_backward():
    w = W.workload(1, n_groups=2, group_size=4, n_tok=200)
    batch = W.make_batch(w, seed=5, device=DEV)
    args = (batch["logits"], batch["target_ids"], batch["behave_lp"], batch["prox_lp"], batch["step_off"],
            batch["traj_off"], batch["group_off"], batch["rewards"])
    a = A.awr_loss_fwd(*args, **batch["params"])                                   # AUTO
    b = A.awr_loss_fwd(*args, **dict(batch["params"], kernel=A.KERNEL_FWD_STREAM))
    c = A.awr_loss_fwd(*args, **dict(batch["params"], kernel=A.KERNEL_GENERIC))
    torch.cuda.synchronize()
    assert torch.equal(a["token_lp"], b["token_lp"]) and float(a["loss"][0]) == float(b["loss"][0])
    assert float((a["token_lp"] - c["token_lp"]).abs().max()) <= 2e-5
    assert int(a["clip_count"][0]) == int(c["clip_count"][0])
    with pytest.raises(A.AwrError) as ei:
        A.awr_loss_fwd_bwd(*args, **dict(batch["params"], kernel=A.KERNEL_FWD_STREAM))
    assert ei.value.status == -5
    with pytest.raises(A.AwrError) as ei:                                          # fp32: unsupported
        A.awr_loss_fwd(batch["logits"].float(), *args[1:], **dict(batch["params"], kernel=A.KERNEL_FWD_STREAM))
    assert ei.value.status == -5


@pytest.mark.parametrize("kernel", CLUSTER_KERNELS)
@pytest.mark.parametrize("cfg", [1, 2])
def test_cluster_configs_small(cfg, kernel):
    w = W.workload(cfg, n_groups=4, group_size=8, n_tok=450)
    batch = W.make_batch(w, seed=cfg, device=DEV)
    batch["params"]["kernel"] = kernel
    P.full_check(batch)
    P.full_check(batch, normalizer=A.NORM_PER_TRAJ)


@pytest.mark.parametrize("kernel", CLUSTER_KERNELS)
@pytest.mark.parametrize("V", [151_936, 50_000])
def test_cluster_gradient_matches_generic_elementwise(kernel, V):
    """The 1e-3 rowmax floor of the north_star bar hides most non-target entries at V = 151,936
    (p_v << 1e-3), so the gradient STORES of the cluster kernels are also compared with the
    one-CTA-per-row kernel (whose gradient pass is separate code) element by element: both are
    bf16 roundings of the same c_t p_v (one rounding there, two in the register-file kernel), so
    they agree within 2 bf16 ulp EVERYWHERE - a zeroed or mis-scaled lane / part would not."""
    w = W.workload(3, n_groups=6, group_size=4, n_tok=331, V=V)
    batch = W.make_batch(w, seed=77, device=DEV, masked_frac=0.03)
    a = P.run_gpu(batch, kernel=kernel)["dlogits"][:, :V].float()
    b = P.run_gpu(batch, kernel=A.KERNEL_GENERIC)["dlogits"][:, :V].float()
    big = torch.maximum(a.abs(), b.abs())
    ulp = torch.exp2(torch.floor(torch.log2(big.clamp(min=2.0 ** -126))) - 7)
    bad = (a - b).abs() > 2 * ulp
    assert not bool(bad.any()), "%d entries differ by more than 2 bf16 ulp" % int(bad.sum())


@pytest.mark.parametrize("kernel", [A.KERNEL_GENERIC] + CLUSTER_KERNELS)
def test_peaked_logits_many_entries_above_the_floor(kernel):
    """A workload where hundreds of entries per row exceed the 1e-3 rowmax floor, so that the
    2-ulp part of the dlogits bar is what decides: 256 'hot' vocabulary entries 12 nats above the
    rest (p ~ 1/256 each), the target among them."""
    V, n_tok = 151_936, 300
    w = W.workload(3, n_groups=6, group_size=4, n_tok=n_tok, V=V)
    batch = W.make_batch(w, seed=13, device=DEV)
    g = torch.Generator(DEV).manual_seed(99)
    z = 0.3 * torch.randn(n_tok, V, generator=g, device=DEV)
    hot = torch.randperm(V, generator=g, device=DEV)[:256]
    z[:, hot] += 12.0
    y = hot[torch.randint(0, 256, (n_tok,), generator=g, device=DEV)]
    batch["logits"] = z.to(torch.bfloat16)
    batch["target_ids"] = y.to(torch.int32)
    lp = torch.log_softmax(batch["logits"].float(), 1)[torch.arange(n_tok, device=DEV), y]
    batch["prox_lp"] = lp + 0.05 * torch.randn(n_tok, generator=g, device=DEV)   # few clips
    batch["behave_lp"] = batch["prox_lp"] + 0.05 * torch.randn(n_tok, generator=g, device=DEV)
    lr = lp - batch["prox_lp"]
    near = ((lr - float(np.log1p(0.2))).abs() < 1e-4) | ((lr - float(np.log1p(-0.2))).abs() < 1e-4)
    batch["prox_lp"] = torch.where(near, batch["prox_lp"] + 0.01, batch["prox_lp"])
    batch["params"]["kernel"] = kernel
    gpu, ora = P.full_check(batch)
    G = np.abs(ora["dlogits"])
    above = (G > 1e-3 * G.max(axis=1, keepdims=True)).sum(axis=1)
    live = ora["coef"] != 0
    assert live.sum() > 100 and above[live].min() >= 200, "the 2-ulp branch must decide here"


def test_unguarded_clip_counts_banded():
    """every other parity input keeps log r_t at least 1e-4 away from
    log(1 +- eps) (generator guard band), so that bit-exact counts test indexing rather than
    rounding luck.  This is the run WITHOUT the guard band, at V = 151,936 with config 3's laws
    (drift 0.3: clips and cap both fire): fp32 and fp64 may then legitimately disagree on a
    token whose ratio sits within rounding of a threshold.  Required: identical trigger flags
    for every token whose oracle |log r - log(1 +- eps)| >= 1e-6, and a clip count that differs
    from the oracle's by at most the number of tokens inside that band.  Both are printed."""
    w = W.workload(3, n_groups=8, group_size=8, n_tok=20_480)
    batch = W.make_batch(w, seed=303, device=DEV, guard=False)
    params = dict(batch["params"])
    n_tok, V = batch["n_tok"], batch["V"]
    assert V == 151_936 and n_tok >= 20_000
    ora = P.oracle_terms_all_rows(
        P.oracle_forward_all_rows(batch, params, lambda lo, hi: batch["logits"][lo:hi, :V].float().cpu().numpy()),
        batch, params)
    gpu = P.run_gpu(batch)
    eps = float(np.float32(params["clip_eps"]))
    lr = ora["token_lp"] - batch["prox_lp"].cpu().numpy().astype(np.float64)
    band = (np.abs(lr - np.log1p(eps)) < 1e-6) | (np.abs(lr - np.log1p(-eps)) < 1e-6)
    coef = gpu["tok_coef"].cpu().numpy()
    term = gpu["tok_term"].cpu().numpy()
    flags = (coef == 0) & (term != 0)
    assert np.array_equal(flags[~band], ora["trig"][~band]), "a trigger flag differs outside the 1e-6 band"
    d = abs(int(gpu["clip_count"][0]) - ora["clip_count"])
    print("unguarded run: %d tokens, clip_count gpu %d / oracle %d, %d tokens inside the 1e-6 band, "
          "%d flags differ (all inside the band)" % (n_tok, int(gpu["clip_count"][0]), ora["clip_count"],
                                                     int(band.sum()), int((flags != ora["trig"]).sum())))
    assert d <= int(band.sum())
    assert ora["clip_count"] > 0.1 * n_tok
    lp = gpu["token_lp"].cpu().numpy().astype(np.float64)
    assert np.abs(lp - ora["token_lp"]).max() <= P.LP_ATOL
    P.check_loss(gpu["loss"][0], ora["loss"], ora["term"], "unguarded config-3 laws")


@pytest.mark.parametrize("kernel", CLUSTER_KERNELS)
def test_cluster_matches_generic_bitwise_on_integers(kernel):
    """All row kernels give the same integers and the same zero pattern."""
    w = W.workload(3, n_groups=6, group_size=4, n_tok=500, V=50_000)
    batch = W.make_batch(w, seed=9, device=DEV, ld=50_000)
    a = P.run_gpu(batch, kernel=kernel)
    b = P.run_gpu(batch, kernel=A.KERNEL_GENERIC)
    assert torch.equal(a["tok_traj"], b["tok_traj"])
    assert torch.equal(a["target_logit"], b["target_logit"])
    assert int(a["clip_count"][0]) == int(b["clip_count"][0])
    assert torch.equal(a["tok_coef"] == 0, b["tok_coef"] == 0)
    assert float((a["token_lp"] - b["token_lp"]).abs().max()) < 2e-5


@pytest.mark.parametrize("horizon", [20, 40, 60])
def test_thinking_shapes_workload(horizon):
    """the Thinking-variant raggedness (400-900 tokens per step; the long
    horizons 20 / 40 / 60 of PAPER.md:154, :321-331) through the same kernels, cut to a size the
    oracle finishes in seconds."""
    w = W.workload(5, n_groups=3, group_size=4, n_tok=700, horizon=horizon)
    st = W.make_structure(W.workload(5, horizon=horizon, n_groups=32), seed=0)
    per_step = np.diff(st["step_off"])
    steps = np.diff(st["traj_off"])
    assert 400 <= per_step.min() and per_step.max() <= 900 and steps.max() <= horizon
    if horizon == 20:      # 256 trajectories, 1 + Poisson(11.5) steps for failures: the cap binds
        assert (steps == 20).any(), "the horizon-20 cap should bind for some failed trajectory"
    batch = W.make_batch(w, seed=71 + horizon, device=DEV)
    assert A.select_kernel(batch["V"], batch["ld"], torch.bfloat16) == A.KERNEL_CLUSTER_RFS
    P.full_check(batch, dual_clip_c=3.0)
    P.full_check(batch, normalizer=A.NORM_PER_TRAJ, flags=A.FLAG_SKIP_UNIFORM)


def test_coupled_flag_does_not_read_prox_lp():
    """include/awr.h: with AWR_FLAG_COUPLED prox_lp is not read and may be NULL (device entry and
    host-buffer entry); the result equals the call that passes behave_lp as prox_lp."""
    w = W.workload(3, n_groups=4, group_size=4, n_tok=200, V=40_000)
    batch = W.make_batch(w, seed=12, device=DEV)
    args = lambda q: (batch["logits"], batch["target_ids"], batch["behave_lp"], q, batch["step_off"],
                      batch["traj_off"], batch["group_off"], batch["rewards"])
    params = dict(batch["params"], flags=A.FLAG_COUPLED)
    a = A.awr_loss_fwd_bwd(*args(None), **params)
    b = A.awr_loss_fwd_bwd(*args(batch["prox_lp"]), **params)
    torch.cuda.synchronize()
    for k in ("loss", "token_lp", "tok_term", "tok_coef", "clip_count", "dlogits"):
        assert torch.equal(a[k], b[k]), k
    with pytest.raises(A.AwrError) as ei:
        A.awr_loss_fwd_bwd(*args(None), **batch["params"])        # decoupled: prox_lp is required
    assert ei.value.status == -1
    host = [None if t is None else t.cpu() for t in args(None)]
    h = A.awr_loss_fwd_bwd_host(*host, device=DEV, pin=False, **params)
    assert torch.equal(h["dlogits"], a["dlogits"].cpu()) and float(h["loss"][0]) == float(a["loss"][0])


def test_dynamic_sampling_flag():
    """SURVEY 8(f) rank 4 / PAPER.md:63: uniform groups skipped on the device, the mean over groups
    runs over the mixed ones; also through the fused head and with no mixed group at all."""
    w = W.workload(3, n_groups=12, group_size=4, n_tok=400, V=40_000, p_equal_groups=0.5)
    batch = W.make_batch(w, seed=61, device=DEV)
    gpu, ora = P.full_check(batch, flags=A.FLAG_SKIP_UNIFORM)
    base, _ = P.full_check(batch)
    mixed = O.mixed_groups(batch["rewards"].cpu().numpy(), batch["group_off"].cpu().numpy())
    assert 0 < mixed.sum() < mixed.size
    assert float(gpu["loss"][0]) == pytest.approx(float(base["loss"][0]) * mixed.size / mixed.sum(), rel=1e-5)
    P.full_check(batch, flags=A.FLAG_SKIP_UNIFORM | A.FLAG_SUCCESS_FILTER)
    batch["rewards"] = torch.ones_like(batch["rewards"])
    z, _ = P.full_check(batch, flags=A.FLAG_SKIP_UNIFORM | A.FLAG_SUCCESS_FILTER)
    assert float(z["loss"][0]) == 0.0 and not z["dlogits"].any()


@pytest.mark.parametrize("flags", [A.FLAG_SUCCESS_FILTER, A.FLAG_COUPLED,
                                   A.FLAG_SUCCESS_FILTER | A.FLAG_COUPLED])
@pytest.mark.parametrize("kernel", [A.KERNEL_GENERIC, A.KERNEL_CLUSTER_RF, A.KERNEL_CLUSTER_RFS,
                                    A.KERNEL_CLUSTER_RFS_LATE])
def test_baseline_variants(flags, kernel):
    """the paper's two comparison losses by flag - RAFT++ (advantage =
    1[R > 0]; run at group size 1 as in :462 and at 4) and the coupled-ratio
    ablation.  The generator's guard band is around the decoupled ratio, so for
    the coupled runs tokens whose coupled ratio sits within 1e-4 of 1 +- eps get a nudge."""
    for gs in (1, 4):
        w = W.workload(3, n_groups=24 // gs, group_size=gs, n_tok=400, V=40_000,
                       normalizer=A.NORM_PER_TRAJ)
        batch = W.make_batch(w, seed=51 + gs, device=DEV)
        batch["params"]["kernel"] = kernel
        if flags & A.FLAG_COUPLED:
            lp = P.run_gpu(batch, backward=False)["token_lp"]
            lr = lp - batch["behave_lp"]
            near = ((lr - float(np.log1p(0.2))).abs() < 1e-4) | ((lr - float(np.log1p(-0.2))).abs() < 1e-4)
            batch["behave_lp"] = torch.where(near, batch["behave_lp"] - 0.01, batch["behave_lp"])
        gpu, ora = P.full_check(batch, flags=flags)
        if flags & A.FLAG_SUCCESS_FILTER:
            assert set(np.unique(ora["adv"]).tolist()) <= {0.0, 1.0} and ora["adv"].sum() > 0
        if gs > 1 or (flags & A.FLAG_SUCCESS_FILTER):     # single-member groups: A = 0 without the filter
            assert (ora["coef"] != 0).any()


@pytest.mark.parametrize("kernel", [A.KERNEL_GENERIC] + CLUSTER_KERNELS)
@pytest.mark.parametrize("norm", [A.NORM_CONST_K, A.NORM_PER_TRAJ])
def test_dual_clip(kernel, norm):
    """Eq. (2) (PAPER.md:270-275, c = 3.0 as in every GRPO run of the paper, :461): tokens with
    A < 0 whose ratio exploded past c are floored at c A, counted, and carry no gradient.  Every
    5th token gets its prox log-prob lowered by 1.5 (r x 4.5), keeping the generator's guard
    band around 1 +- eps and adding one around c."""
    w = W.workload(3, n_groups=6, group_size=4, n_tok=420, V=40_000, normalizer=norm)
    batch = W.make_batch(w, seed=31, device=DEV)
    q = batch["prox_lp"].clone()
    q[::5] -= 1.5
    batch["prox_lp"] = q
    batch["params"]["kernel"] = kernel
    lp = P.run_gpu(batch, backward=False)["token_lp"]
    near = ((lp - q) - float(np.log(3.0))).abs() < 1e-4          # keep log r away from log c
    batch["prox_lp"] = torch.where(near, q - 0.01, q)
    gpu, ora = P.full_check(batch, dual_clip_c=3.0)
    assert ora["dual_clip_count"] > 5 and ora["clip_count"] > 0
    off, _ = P.full_check(batch, dual_clip_c=0.0)
    assert int(off["dual_clip_count"][0]) == 0
    P.full_check(batch, backward=False, dual_clip_c=3.0)


@pytest.mark.parametrize("kernel,V,dtype", [(A.KERNEL_GENERIC, 1024, torch.float32),
                                            (A.KERNEL_GENERIC, 1003, torch.bfloat16),
                                            (A.KERNEL_GENERIC, 50_000, torch.bfloat16),
                                            (A.KERNEL_CLUSTER_RF, 151_936, torch.bfloat16),
                                            (A.KERNEL_CLUSTER_RF4, 151_936, torch.bfloat16),
                                            (A.KERNEL_CLUSTER_RF, 40_000, torch.bfloat16),
                                            (A.KERNEL_CLUSTER_RFS, 151_936, torch.bfloat16),
                                            (A.KERNEL_CLUSTER_RFS, 40_000, torch.bfloat16),
                                            (A.KERNEL_CLUSTER_RFS_LATE, 151_936, torch.bfloat16),
                                            (A.KERNEL_CLUSTER_RFS_LATE, 40_000, torch.bfloat16),
                                            (A.KERNEL_AUTO, 151_936, torch.bfloat16)])
@pytest.mark.parametrize("backward", [True, False])
def test_token_entropy(kernel, V, dtype, backward):
    """per-token entropy from the same streaming pass,
    forward-only (the proximal log-prob recomputation of :436) and with the gradient.  Some
    logits are set to -inf (p = 0 entries contribute nothing); masked tokens give 0.
    Bar: |dH| <= 1e-4 absolute (fp32 sums of e z next to the log-sum-exp)."""
    ld = (V + 7) // 8 * 8
    w = W.workload(3, n_groups=4, group_size=4, n_tok=300, V=V, dtype=dtype)
    batch = W.make_batch(w, seed=41, device=DEV, ld=ld, masked_frac=0.05)
    z = batch["logits"]
    z[::3, 5:V:97] = float("-inf")
    ids = batch["target_ids"].long().clamp(min=0)
    z[torch.arange(z.shape[0], device=DEV), ids] = z[torch.arange(z.shape[0], device=DEV), ids].nan_to_num(neginf=0.0)
    params = dict(batch["params"], kernel=kernel)
    fn = A.awr_loss_fwd_bwd if backward else A.awr_loss_fwd
    out = fn(z, batch["target_ids"], batch["behave_lp"], batch["prox_lp"], batch["step_off"],
             batch["traj_off"], batch["group_off"], batch["rewards"], V=V,
             want=A.OPTIONAL_OUTPUTS + ("token_entropy",), **params)
    torch.cuda.synchronize()
    ora = P.run_oracle(batch, want_dlogits=False, want_entropy=True)
    H = out["token_entropy"].cpu().numpy().astype(np.float64)
    assert np.isfinite(H).all()
    assert np.abs(H - ora["token_entropy"]).max() <= 1e-4
    assert np.all(H[batch["target_ids"].cpu().numpy() < 0] == 0.0)
    assert ora["token_entropy"].max() > 1.0
    # the other outputs are what they are without the entropy output
    ref = fn(z, batch["target_ids"], batch["behave_lp"], batch["prox_lp"], batch["step_off"],
             batch["traj_off"], batch["group_off"], batch["rewards"], V=V, **params)
    torch.cuda.synchronize()
    if kernel == A.KERNEL_AUTO and not backward:
        # forward-only AUTO streams with the one-CTA-per-row kernel unless the entropy is asked for
        assert float((out["token_lp"] - ref["token_lp"]).abs().max()) <= 2e-5
        assert int(out["clip_count"][0]) == int(ref["clip_count"][0])
    else:
        assert torch.equal(out["token_lp"], ref["token_lp"]) and float(out["loss"][0]) == float(ref["loss"][0])
    if backward:
        assert torch.equal(out["dlogits"][:, :V], ref["dlogits"][:, :V])


def test_token_entropy_not_offered_by_the_shared_memory_cluster_kernel():
    w = W.workload(1, n_groups=2, group_size=4, n_tok=64, V=40_000)
    batch = W.make_batch(w, seed=1, device=DEV)
    with pytest.raises(A.AwrError) as ei:
        A.awr_loss_fwd(batch["logits"], batch["target_ids"], batch["behave_lp"], batch["prox_lp"],
                       batch["step_off"], batch["traj_off"], batch["group_off"], batch["rewards"],
                       want=("token_entropy",), **dict(batch["params"], kernel=A.KERNEL_CLUSTER))
    assert ei.value.status == -5


@pytest.mark.parametrize("kernel", [A.KERNEL_GENERIC] + CLUSTER_KERNELS)
def test_in_place(kernel):
    """dlogits may alias logits exactly (include/awr.h)."""
    w = W.workload(3, n_groups=4, group_size=4, n_tok=300, V=40_000)
    batch = W.make_batch(w, seed=2, device=DEV)
    batch["params"]["kernel"] = kernel
    ref = P.run_gpu(batch)
    z = batch["logits"].clone()
    out = A.awr_loss_fwd_bwd(z, batch["target_ids"], batch["behave_lp"], batch["prox_lp"],
                             batch["step_off"], batch["traj_off"], batch["group_off"],
                             batch["rewards"], dlogits=z, **batch["params"])
    torch.cuda.synchronize()
    assert out["dlogits"].data_ptr() == z.data_ptr()
    assert torch.equal(z, ref["dlogits"])
    assert torch.equal(out["token_lp"], ref["token_lp"])
    assert float(out["loss"][0]) == float(ref["loss"][0])


def test_deterministic():
    """Fixed-order reductions: two runs give identical bits."""
    w = W.workload(2, n_groups=4, group_size=8, n_tok=600, V=151_936)
    batch = W.make_batch(w, seed=4, device=DEV)
    a = P.run_gpu(batch)
    b = P.run_gpu(batch)
    for k in a:
        assert torch.equal(a[k], b[k]), k


@pytest.mark.parametrize("V,ld", [(151_936, 151_936), (40_000, 40_008), (20_000, 20_000)])
def test_rfs_schedules_same_bits(V, ld):
    """AWR_KERNEL_CLUSTER_RFS takes the last register group's (max, sum) from the ring before that
    group's registers are free and writes exp back in place; AWR_KERNEL_CLUSTER_RFS_LATE does it in
    registers afterwards.  Same elements, same references, same fold order: every output, the
    gradient included, must be bit-identical (config-3 laws: clips, zero-advantage rows, masked
    tokens; NG = 4, 2 and 1 groups per row half)."""
    w = W.workload(3, n_groups=4, group_size=4, n_tok=700, V=V)
    batch = W.make_batch(w, seed=77, device=DEV, ld=ld, masked_frac=0.05)
    outs = []
    for kernel in (A.KERNEL_CLUSTER_RFS, A.KERNEL_CLUSTER_RFS_LATE):
        batch["params"]["kernel"] = kernel
        outs.append(P.run_gpu(batch, dual_clip_c=3.0))
    for k in outs[0]:
        a, b = outs[0][k], outs[1][k]
        if k == "dlogits":                       # the padding columns >= V are not written by anybody
            a, b = a[:, :V], b[:, :V]
        assert torch.equal(a, b), k


@pytest.mark.parametrize("kernel", [A.KERNEL_CLUSTER_RFS, A.KERNEL_CLUSTER_RFS_LATE])
@pytest.mark.parametrize("V,ld,n_tok", [(151_936, 151_936, 1500), (40_000, 40_008, 37)])
def test_rfs_soak_bit_identical(V, ld, n_tok, kernel):
    """300 back-to-back calls of the service-warp kernel (mbarrier hand-overs between 15 data warps,
    the service warp, the TMA and the peer CTA; ring slots and staging buffers reused every row):
    every output stays bit-identical to the first call's.  Stands in for racecheck (closed on this
    pool): a lost hand-over shows as a wrong row or a hang."""
    w = W.workload(3, n_groups=4, group_size=4, n_tok=n_tok, V=V)
    batch = W.make_batch(w, seed=5, device=DEV, ld=ld, masked_frac=0.03)
    call = A.LossCall(batch["logits"], batch["target_ids"], batch["behave_lp"], batch["prox_lp"],
                      batch["step_off"], batch["traj_off"], batch["group_off"], batch["rewards"],
                      want=("err_word", "tok_term", "tok_coef", "token_entropy"),
                      **dict(batch["params"], kernel=kernel, dual_clip_c=3.0))
    call.run()
    torch.cuda.synchronize()
    ref = {k: v.clone() for k, v in call.out.items()}
    for i in range(300):
        call.out["dlogits"].fill_(7.0)
        call.run()
        if i % 50 == 49:
            torch.cuda.synchronize()
            for k, v in ref.items():
                a, b = call.out[k], v
                if k == "dlogits":
                    a, b = a[:, :V], b[:, :V]
                assert torch.equal(a, b), (k, i)


# ------------------------------------------------------------------ edge cases
def test_empty_batch():
    z = torch.empty(0, 1024, dtype=torch.bfloat16, device=DEV)
    i32 = lambda x: torch.tensor(x, dtype=torch.int32, device=DEV)
    f32 = lambda x: torch.tensor(x, dtype=torch.float32, device=DEV)
    out = A.awr_loss_fwd_bwd(z, i32([]), f32([]), f32([]), i32([0]), i32([0]), i32([0]), f32([]))
    torch.cuda.synchronize()
    assert float(out["loss"][0]) == 0.0 and int(out["clip_count"][0]) == 0
    assert int(out["err_word"][0]) == 0


def test_empty_steps_trajectories_groups():
    """A10: empty step counts toward |tau_i|; empty trajectory enters its group's statistics;
    single-member and empty groups give A = 0."""
    V = 2048
    step_off = np.array([0, 3, 3, 10, 10, 10, 25, 40], dtype=np.int32)    # steps 1,3,4 empty
    traj_off = np.array([0, 2, 2, 5, 6, 7], dtype=np.int32)               # traj 1 has no steps
    group_off = np.array([0, 3, 3, 4, 5], dtype=np.int32)                 # group 1 empty, 2/3 single
    rewards = np.array([1, 0, 0.5, 1, 0], dtype=np.float32)
    g = torch.Generator(DEV).manual_seed(3)
    n = 40
    z = (torch.randn(n, V, generator=g, device=DEV) * 3).to(torch.bfloat16)
    y = torch.randint(0, V, (n,), generator=g, device=DEV).to(torch.int32)
    lp = torch.log_softmax(z.float(), 1)[torch.arange(n, device=DEV), y.long()]
    q = lp + 0.1 * torch.randn(n, generator=g, device=DEV)
    b = q + 0.1 * torch.randn(n, generator=g, device=DEV)
    batch = dict(logits=z, target_ids=y, behave_lp=b, prox_lp=q, V=V, ld=V, n_tok=n,
                 step_off=torch.from_numpy(step_off).to(DEV),
                 traj_off=torch.from_numpy(traj_off).to(DEV),
                 group_off=torch.from_numpy(group_off).to(DEV),
                 rewards=torch.from_numpy(rewards).to(DEV),
                 params=dict(k_norm=10.0, clip_eps=0.2, stale_cap=2.0, normalizer=A.NORM_PER_TRAJ,
                             flags=0, loss_scale=0.5))
    gpu, ora = P.full_check(batch)
    assert ora["adv"][3] == 0 and ora["adv"][4] == 0
    P.full_check(batch, normalizer=A.NORM_CONST_K)


def test_error_word_bits():
    w = W.workload(1, n_groups=2, group_size=4, n_tok=120, V=1024, dtype=torch.float32)
    batch = W.make_batch(w, seed=1, device=DEV)
    ids = batch["target_ids"].clone()
    ids[7] = 1024
    ids[9] = 5000
    batch["target_ids"] = ids
    gpu, ora = P.full_check(batch)
    assert int(gpu["err_word"][0]) == A.ERRBIT_TARGET_RANGE
    assert float(gpu["token_lp"][7]) == 0.0 and float(gpu["dlogits"][7].abs().max()) == 0.0
    bad = batch["step_off"].clone()
    bad[3] = bad[2] - 1
    out = A.awr_loss_fwd(batch["logits"], ids, batch["behave_lp"], batch["prox_lp"], bad,
                         batch["traj_off"], batch["group_off"], batch["rewards"])
    torch.cuda.synchronize()
    assert int(out["err_word"][0]) & A.ERRBIT_STEP_OFF
    bad = batch["group_off"].clone()
    bad[-1] += 1
    out = A.awr_loss_fwd(batch["logits"], ids, batch["behave_lp"], batch["prox_lp"],
                         batch["step_off"], batch["traj_off"], bad, batch["rewards"])
    torch.cuda.synchronize()
    assert int(out["err_word"][0]) & A.ERRBIT_GROUP_OFF


def test_status_codes_on_device():
    w = W.workload(1, n_groups=2, group_size=4, n_tok=64, V=1024, dtype=torch.float32)
    batch = W.make_batch(w, seed=1, device=DEV)
    args = (batch["logits"], batch["target_ids"], batch["behave_lp"], batch["prox_lp"],
            batch["step_off"], batch["traj_off"], batch["group_off"], batch["rewards"])
    with pytest.raises(A.AwrError) as e:
        A.awr_loss_fwd_bwd(*args, clip_eps=1.5)
    assert e.value.status == -5
    with pytest.raises(A.AwrError) as e:
        A.awr_loss_fwd_bwd(*args, workspace=torch.empty(256, dtype=torch.uint8, device=DEV))
    assert e.value.status == -6
    with pytest.raises(A.AwrError) as e:
        A.awr_loss_fwd_bwd(*args, kernel=A.KERNEL_CLUSTER)      # fp32 / small V: unsupported
    assert e.value.status == -5
    with pytest.raises(A.AwrError) as e:
        A.awr_loss_fwd_bwd(batch["logits"][:, 1:], *args[1:])  # rows not 16-byte aligned
    assert e.value.status == -4


def test_group_advantage_kernel():
    rng = np.random.default_rng(0)
    sizes = [8, 1, 0, 33, 64, 100, 2, 16]
    off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int32)
    R = rng.normal(size=off[-1]).astype(np.float32)
    R[off[4]:off[5]] = 0.25                                     # an all-equal group
    for flags in (0, A.FLAG_SAMPLE_STD):
        adv = A.awr_group_advantage(torch.from_numpy(R).to(DEV), torch.from_numpy(off).to(DEV),
                                    flags=flags).cpu().numpy()
        ref = O.group_advantage(R, off, flags)
        np.testing.assert_allclose(adv, ref, rtol=0, atol=5e-6)
        assert np.all(adv[off[4]:off[5]] == 0) and adv[off[1]] == 0


def test_graph_capture():
    """The call only enqueues work: it can be captured into a CUDA graph and replayed."""
    w = W.workload(1, n_groups=2, group_size=4, n_tok=200, V=40_000)
    batch = W.make_batch(w, seed=6, device=DEV)
    call = A.LossCall(batch["logits"], batch["target_ids"], batch["behave_lp"], batch["prox_lp"],
                      batch["step_off"], batch["traj_off"], batch["group_off"], batch["rewards"],
                      **batch["params"])
    ref = {k: v.clone() for k, v in call.run().items()}
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):
            call.run(stream=s)
    for v in call.out.values():
        v.zero_()
    g.replay()
    torch.cuda.synchronize()
    for k in ref:
        assert torch.equal(ref[k], call.out[k]), k


def _random_shapes(n, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    out = []
    for _ in range(n):
        V = int(rng.integers(16_384 // 8, 163_840 // 8 + 1)) * 8
        ld = V + 8 * int(rng.integers(0, 3))
        out.append((V, ld, int(rng.integers(1, 260)), int(rng.integers(0, 1 << 30))))
    return out


@pytest.mark.parametrize("V,ld,n_tok,seed", _random_shapes(10, 2024))
def test_register_file_kernels_random_shapes(V, ld, n_tok, seed):
    """Seeded random vocabulary sizes over the whole range the register-file kernels accept
    (every NU from 3 to 20 has its own instantiation), random row strides and row counts
    (fewer rows than clusters included), both cluster shapes, entropy on."""
    w = W.workload(3, n_groups=3, group_size=4, n_tok=max(n_tok, 12), V=V)
    batch = W.make_batch(w, seed=seed % 1000, device=DEV, ld=ld, masked_frac=0.05)
    kernels = [A.KERNEL_CLUSTER_RF, A.KERNEL_CLUSTER_RF4] + (
        [A.KERNEL_CLUSTER_RFS, A.KERNEL_CLUSTER_RFS_LATE] if V <= 153_600 else [])
    for kernel in kernels:
        batch["params"]["kernel"] = kernel
        gpu, ora = P.full_check(batch, dual_clip_c=3.0)
    out = A.awr_loss_fwd(batch["logits"], batch["target_ids"], batch["behave_lp"], batch["prox_lp"],
                         batch["step_off"], batch["traj_off"], batch["group_off"], batch["rewards"],
                         V=V, want=("token_entropy",), **batch["params"])
    torch.cuda.synchronize()
    ref = P.run_oracle(batch, want_dlogits=False, want_entropy=True)
    assert np.abs(out["token_entropy"].cpu().numpy() - ref["token_entropy"]).max() <= 1e-4


@pytest.mark.parametrize("n_tok,V,dtype", [(7000, 40_000, torch.bfloat16), (300, 1024, torch.float32)])
def test_host_buffer_entry(n_tok, V, dtype):
    """awr_loss_fwd_bwd_host (the e2e leg of bench.py): pinned host buffers, row panels over three
    device buffers (7,000 rows of 80 KB = three 256 MB panels).  Same kernels as the device entry,
    so every output must be bit-identical to it, and it is checked against the oracle as well."""
    w = W.workload(3, n_groups=6, group_size=4, n_tok=n_tok, V=V, dtype=dtype)
    batch = W.make_batch(w, seed=81, device=DEV, masked_frac=0.02)
    want = A.OPTIONAL_OUTPUTS + ("token_entropy",)
    dev = A.awr_loss_fwd_bwd(batch["logits"], batch["target_ids"], batch["behave_lp"],
                             batch["prox_lp"], batch["step_off"], batch["traj_off"],
                             batch["group_off"], batch["rewards"], want=want,
                             **dict(batch["params"], dual_clip_c=3.0))
    torch.cuda.synchronize()
    host_in = {k: batch[k].cpu().pin_memory() for k in ("logits", "target_ids", "behave_lp", "prox_lp",
                                                        "step_off", "traj_off", "group_off", "rewards")}
    out = A.awr_loss_fwd_bwd_host(host_in["logits"], host_in["target_ids"], host_in["behave_lp"],
                                  host_in["prox_lp"], host_in["step_off"], host_in["traj_off"],
                                  host_in["group_off"], host_in["rewards"], device=DEV, want=want,
                                  **dict(batch["params"], dual_clip_c=3.0))
    for k in ("loss", "clip_count", "dual_clip_count", "token_lp", "tok_term", "tok_coef", "tok_traj",
              "target_logit", "adv", "token_entropy", "err_word", "dlogits"):
        assert not out[k].is_cuda
        assert torch.equal(out[k], dev[k].cpu()), k
    ora = P.run_oracle(batch, dual_clip_c=3.0, want_entropy=True)
    P.check_scalars({k: v for k, v in out.items() if k != "dlogits"}, ora)
    P.check_dlogits(out["dlogits"].to(DEV), ora, V)
    assert np.abs(out["token_entropy"].numpy() - ora["token_entropy"]).max() <= 1e-4


# ------------------------------------------------------------------ red zones (compute-sanitizer is closed on this pool)
def _guarded(shape, dtype, pattern, pad=4096):
    """A tensor of `shape` carved out of a larger buffer whose head and tail hold a byte pattern."""
    n = int(np.prod(shape))
    esz = torch.empty(0, dtype=dtype).element_size()
    pad_e = pad // esz
    buf = torch.empty(n + 2 * pad_e, dtype=dtype, device=DEV)
    buf.view(torch.uint8).fill_(pattern)
    return buf, buf[pad_e:pad_e + n].view(shape), pad_e


def _zones_intact(buf, pad_e, n, pattern):
    raw = buf.view(torch.uint8)
    esz = buf.element_size()
    return bool((raw[:pad_e * esz] == pattern).all()) and bool((raw[(pad_e + n) * esz:] == pattern).all())


@pytest.mark.parametrize("kernel,backward", [(A.KERNEL_GENERIC, True), (A.KERNEL_CLUSTER, True),
                                             (A.KERNEL_CLUSTER_RF, True), (A.KERNEL_CLUSTER_RF4, True),
                                             (A.KERNEL_CLUSTER_RFS, True), (A.KERNEL_CLUSTER_RFS_LATE, True),
                                             (A.KERNEL_FWD_STREAM, False)])
@pytest.mark.parametrize("V,ld", [(151_936, 151_936), (40_000, 40_008)])
def test_red_zones_row_kernels(kernel, backward, V, ld):
    """No kernel writes outside its outputs or its workspace, and none writes the columns
    >= V of a padded gradient row: every output (and the workspace) sits between two 4 KB zones
    of a byte pattern that must survive; the gradient buffer is pre-filled with the pattern and
    its padding columns must still hold it.  (Stands in for compute-sanitizer memcheck, which
    is closed on this pool: profiles/r2_sanitizer.md.)"""
    w = W.workload(3, n_groups=6, group_size=4, n_tok=333, V=V)
    b = W.make_batch(w, seed=21, device=DEV, ld=ld, masked_frac=0.03)
    n, n_traj = b["n_tok"], b["rewards"].numel()
    PAT = 0xA5
    spec = dict(loss=((1,), torch.float32), token_lp=((n,), torch.float32), clip_count=((1,), torch.int64),
                dual_clip_count=((1,), torch.int64), adv=((n_traj,), torch.float32),
                tok_traj=((n,), torch.int32), target_logit=((n,), torch.float32),
                tok_term=((n,), torch.float32), tok_coef=((n,), torch.float32),
                err_word=((1,), torch.int32), token_entropy=((n,), torch.float32))
    bufs, out = {}, {}
    for k, (shape, dt) in spec.items():
        bufs[k], out[k], _ = _guarded(shape, dt, PAT)
    if backward:
        bufs["dlogits"], out["dlogits"], _ = _guarded((n, ld), torch.bfloat16, PAT)
    need = A.workspace_bytes(n, V, b["step_off"].numel() - 1, n_traj, b["group_off"].numel() - 1)
    need = (need + 255) // 256 * 256
    wsbuf = torch.empty(need + 8192, dtype=torch.uint8, device=DEV)
    off = 4096 + ((-(wsbuf.data_ptr() + 4096)) % 256)       # 256-byte aligned, >= 4 KB in
    wsbuf.fill_(PAT)
    ws = wsbuf[off:off + need]
    call = A.LossCall(b["logits"], b["target_ids"], b["behave_lp"], b["prox_lp"], b["step_off"], b["traj_off"],
                      b["group_off"], b["rewards"], V=V, backward=backward, out=out, workspace=ws,
                      **dict(b["params"], kernel=kernel, dual_clip_c=3.0))
    if kernel == A.KERNEL_CLUSTER:
        call.outs.token_entropy = None                   # not offered by the shared-memory cluster kernel
    call.run()
    torch.cuda.synchronize()
    assert int(out["err_word"][0]) == 0
    for k, (shape, dt) in spec.items():
        pad_e = 4096 // torch.empty(0, dtype=dt).element_size()
        assert _zones_intact(bufs[k], pad_e, int(np.prod(shape)), PAT), k
    assert bool((wsbuf[:off] == PAT).all()) and bool((wsbuf[off + need:] == PAT).all()), "workspace"
    if backward:
        assert _zones_intact(bufs["dlogits"], 2048, n * ld, PAT), "dlogits"
        if ld > V:
            padcols = out["dlogits"][:, V:].contiguous().view(torch.uint8)
            assert bool((padcols == PAT).all()), "columns >= V of the gradient rows were written"
        assert np.isfinite(out["dlogits"][:, :V].float().cpu().numpy()).all()
