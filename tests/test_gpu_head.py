"""GPU parity of the fused LM-head path (a5, BASELINE.json config 4) against the fp64 oracle:
the tcgen05 GEMM engine on its own (every operand-major combination, ragged sizes) and
awr_loss_fwd_bwd_fused_head end to end.  Run on the B200 box: pytest -m gpu.

Bars: token_lp 1e-4 absolute; loss as the logits path; clip_count,
tok_traj exact; dhidden / dw_head: relative Frobenius error <= 5e-3 and max-abs error
<= 1e-2 max|oracle| (proposed for config 4)."""
import numpy as np
import pytest
import torch

import paper_2606_05597_b200 as A
from gen import workloads as W
from oracle import awr_oracle as O
import parity_util as P

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


@pytest.fixture(autouse=True, scope="module")
def _gpu():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (run them with gpurun)")
    assert torch.cuda.get_device_capability(0)[0] == 10, "sm_100 only"
    yield


def _f64(t):
    return t.float().cpu().numpy().astype(np.float64)


HEAD_KERNELS = [A.KERNEL_HEAD_1CTA, A.KERNEL_HEAD_2CTA]
HEAD_PANEL_KERNELS = [A.KERNEL_HEAD_2CTA_STORED, A.KERNEL_HEAD_2CTA_E16,   # keep one row panel of logits / E
                      A.KERNEL_HEAD_2CTA_ROWREF]


# ------------------------------------------------------------------ the GEMM engine alone
@pytest.mark.parametrize("kernel", HEAD_KERNELS)
@pytest.mark.parametrize("a_major,b_major", [(0, 0), (0, 1), (1, 0), (1, 1)])
@pytest.mark.parametrize("M,N,Kc", [(128, 256, 64), (256, 512, 256), (300, 1000, 200),
                                    (131, 264, 72), (1000, 2048, 1096), (2304, 1280, 520)])
def test_gemm_engine_matches_fp64_matmul(a_major, b_major, M, N, Kc, kernel):
    """C = A B for K-major and MN-major operands; sizes span one tile, several tiles, ragged
    row / column / contraction tails (TMA zero fill).  The expected value is the float64
    product of the same bf16 inputs; the result is rounded once to bf16."""
    if a_major == 1 and M % 8:
        M = (M + 7) // 8 * 8          # an MN-major operand needs a 16-byte-aligned row stride
    if Kc % 8:
        Kc = (Kc + 7) // 8 * 8
    g = torch.Generator(DEV).manual_seed(M * 7 + N * 3 + Kc)
    a = torch.randn(M, Kc, generator=g, device=DEV).to(torch.bfloat16)
    b = torch.randn(Kc, N, generator=g, device=DEV).to(torch.bfloat16)
    a_st = a if a_major == 0 else a.t().contiguous()          # stored [Kc, M]
    b_st = b.t().contiguous() if b_major == 0 else b          # stored [N, Kc] / [Kc, N]
    c = A.awr_gemm_bf16(a_st, b_st, a_major, b_major, kernel=kernel)
    torch.cuda.synchronize()
    ref = _f64(a) @ _f64(b)
    got = _f64(c)
    tol = 2.0 ** -8 * np.abs(ref) + 1e-3 * np.sqrt(Kc)
    bad = np.abs(got - ref) > tol
    assert not bad.any(), "%d bad entries, first at %s" % (bad.sum(), np.argwhere(bad)[0])


# ------------------------------------------------------------------ a5 end to end
def _head_batch(n_tok, K, V, seed, n_groups=4, group_size=4, masked_frac=0.0, lp_mode=None):
    over = dict(n_groups=n_groups, group_size=group_size, n_tok=n_tok, V=V, hidden=K)
    if lp_mode is not None:
        over["lp_mode"] = lp_mode
    w = W.workload(4, **over)
    return W.make_batch(w, seed=seed, device=DEV, masked_frac=masked_frac)


def _run_head(batch, w_layout=A.W_K_BY_V, **over):
    params = dict(batch["params"])
    params.update(over)
    wh = batch["w_head"] if w_layout == A.W_K_BY_V else batch["w_head"].t().contiguous()
    out = A.awr_loss_fwd_bwd_fused_head(batch["hidden"], wh, batch["target_ids"],
                                        batch["behave_lp"], batch["prox_lp"], batch["step_off"],
                                        batch["traj_off"], batch["group_off"], batch["rewards"],
                                        w_layout=w_layout, **params)
    torch.cuda.synchronize()
    return out


def _oracle_head(batch, **over):
    host = W.to_host(batch)
    args, kw = W.oracle_args(host)
    kw.update(over)
    kw.pop("kernel", None)
    return O.awr_loss_fwd_bwd_fused_head(*args, **kw)


def _check_head(gpu, ora, w_layout):
    assert int(gpu["err_word"][0]) == 0
    assert np.array_equal(gpu["tok_traj"].cpu().numpy(), ora["tok_traj"].astype(np.int32))
    lp = gpu["token_lp"].cpu().numpy().astype(np.float64)
    assert np.abs(lp - ora["token_lp"]).max() <= P.LP_ATOL
    assert int(gpu["clip_count"][0]) == ora["clip_count"]
    assert int(gpu["dual_clip_count"][0]) == ora["dual_clip_count"]
    P.check_loss(gpu["loss"][0], ora["loss"], ora["term"], "fused head")
    coef = gpu["tok_coef"].cpu().numpy()
    assert np.array_equal(coef == 0, ora["coef"] == 0)
    dh = _f64(gpu["dhidden"])
    dw = _f64(gpu["dw_head"])
    if w_layout == A.W_V_BY_K:
        dw = dw.T
    for name, got, ref in (("dhidden", dh, ora["dhidden"]), ("dw_head", dw, ora["dw_head"])):
        fro = np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-300)
        mx = np.abs(got - ref).max() / max(np.abs(ref).max(), 1e-300)
        assert fro <= 5e-3, "%s relative Frobenius error %.3e" % (name, fro)
        assert mx <= 1e-2, "%s max-abs error %.3e of max|oracle|" % (name, mx)
    # rows with c_t = 0 contribute nothing: their dhidden rows are exactly zero
    zero_rows = ora["coef"] == 0
    if zero_rows.any():
        assert not gpu["dhidden"][torch.from_numpy(zero_rows).to(DEV)].any()


@pytest.mark.parametrize("kernel", HEAD_KERNELS + HEAD_PANEL_KERNELS)
@pytest.mark.parametrize("w_layout", [A.W_K_BY_V, A.W_V_BY_K])
@pytest.mark.parametrize("n_tok,K,V", [(300, 128, 1000), (128, 64, 256), (517, 192, 2056)])
def test_head_vs_oracle(n_tok, K, V, w_layout, kernel):
    """Ragged row tile, ragged vocabulary tile, several contraction blocks; masked tokens; the
    config-3 drift law so that clips and zero-advantage rows occur."""
    batch = _head_batch(n_tok, K, V, seed=11, masked_frac=0.03, lp_mode="drift")
    gpu = _run_head(batch, w_layout, stale_cap=2.0, kernel=kernel)
    ora = _oracle_head(batch, stale_cap=2.0)
    assert ora["clip_count"] > 0
    _check_head(gpu, ora, w_layout)


@pytest.mark.parametrize("kernel,n_tok,panels", [(A.KERNEL_HEAD_1CTA, 9700, 3),
                                                 (A.KERNEL_HEAD_2CTA, 19300, 3),
                                                 (A.KERNEL_HEAD_2CTA_STORED, 19300, 3),
                                                 (A.KERNEL_HEAD_2CTA_E16, 19300, 3),
                                                 (A.KERNEL_HEAD_2CTA_ROWREF, 19300, 3)])
@pytest.mark.parametrize("norm", [A.NORM_CONST_K, A.NORM_PER_TRAJ])
def test_head_several_panels(norm, kernel, n_tok, panels):
    """More rows than one dS panel (4,736 rows, 9,472 for CTA pairs): dw_head accumulates
    across panels in fp32."""
    batch = _head_batch(n_tok, 64, 512, seed=3, n_groups=8, group_size=8)
    gpu = _run_head(batch, A.W_K_BY_V, normalizer=norm, kernel=kernel)
    ora = _oracle_head(batch, normalizer=norm)
    _check_head(gpu, ora, A.W_K_BY_V)
    per_call = 5 * panels if kernel in HEAD_PANEL_KERNELS else 2 + 3 * panels
    if kernel == A.KERNEL_HEAD_2CTA_ROWREF:
        per_call = 6 * panels          # (reference tile, F, scalars, fix-up, dhidden, dw_head) per panel
    assert A.head_launches_per_call(n_tok, 512, 64, kernel) == 3 + per_call
    assert A.head_launches_per_call(n_tok, 512, 64) == A.head_launches_per_call(
        n_tok, 512, 64, A.KERNEL_HEAD_2CTA_ROWREF)          # AUTO resolves to the row-reference mode


def test_head_stored_logits_same_bits_as_recompute():
    """The stored-logits mode keeps the fp32 accumulators of the forward GEMM and applies the
    same dS arithmetic as the recompute epilogue: every output is bit-identical."""
    batch = _head_batch(1111, 128, 3000, seed=21, lp_mode="drift", masked_frac=0.02)
    a = _run_head(batch, kernel=A.KERNEL_HEAD_2CTA, stale_cap=2.0)
    b = _run_head(batch, kernel=A.KERNEL_HEAD_2CTA_STORED, stale_cap=2.0)
    for k in ("loss", "token_lp", "clip_count", "tok_coef", "tok_term", "dhidden", "dw_head"):
        assert torch.equal(a[k], b[k]), k


@pytest.mark.parametrize("loud_id", [7, 700])
def test_head_rowref_peaked_and_unlikely_targets(loud_id):
    """Row-reference mode away from its comfortable case.  The reference of a row is its largest logit
    among the first 256 vocabulary entries.  One "loud" token gets a logit ~40 above all others in
    every row; a third of the rows have it as target (p_y -> 1), the others keep a target 40 nats
    below it.  loud_id = 7: the reference IS the loud logit, every stored e <= 1 and the unlikely
    targets sit at e^-40; loud_id = 700: the reference is an ordinary logit, the loud entry is stored
    as e^40 and the row sums are 1e17.  Both must meet the oracle at the usual bars, nothing flagged."""
    n_tok, K, V = 600, 128, 2056
    batch = _head_batch(n_tok, K, V, seed=61, lp_mode="drift", masked_frac=0.02)
    hid = batch["hidden"].float()
    w = batch["w_head"].float().clone()                       # [K, V]
    ids = batch["target_ids"].clone()
    loud = hid.mean(0)
    loud = loud / loud.norm() * 4.0
    w[:, loud_id] = loud
    batch["w_head"] = w.to(torch.bfloat16)
    hid = hid + 10.0 * loud / loud.norm()                    # every row has a component along it: z_loud ~ 40
    batch["hidden"] = hid.to(torch.bfloat16)
    sel = torch.arange(n_tok, device=DEV) % 3 == 0
    ids[sel & (ids >= 0)] = loud_id
    batch["target_ids"] = ids
    z = batch["hidden"].float() @ batch["w_head"].float()
    lp = torch.log_softmax(z.double(), -1)
    gathered = lp.gather(1, ids.clamp(min=0).long()[:, None])[:, 0].float()
    batch["prox_lp"] = gathered + 0.01 * torch.randn_like(gathered)
    batch["behave_lp"] = batch["prox_lp"] + 0.01 * torch.randn_like(gathered)
    assert float(gathered[(~sel) & (ids >= 0)].min()) < -30.0 and float(gathered[sel & (ids >= 0)].max()) > -1e-3
    ora = _oracle_head(batch)
    for kernel in (A.KERNEL_HEAD_2CTA_ROWREF, A.KERNEL_HEAD_2CTA_E16):
        gpu = _run_head(batch, kernel=kernel)
        _check_head(gpu, ora, A.W_K_BY_V)


@pytest.mark.parametrize("w_layout", [A.W_K_BY_V, A.W_V_BY_K])
def test_head_rowref_overflow_rows_are_redone(w_layout):
    """Rows with a logit more than ~88 nats above their reference (the largest of their first 256
    logits) cannot be represented relative to it: exp overflows, head_scalars_kernel marks the row and
    head_fix_rows_kernel redoes it from hidden and w_head.  Two such rows (one with the loud token as
    its target, one with an ordinary target 140 nats below it), a masked row with the same logits,
    entropy on: every output meets the oracle at the usual bars, nothing is flagged."""
    n_tok, K, V = 300, 64, 1000
    batch = _head_batch(n_tok, K, V, seed=62)
    hid = batch["hidden"].float().clone()
    w = batch["w_head"].float().clone()
    ids = batch["target_ids"].clone()
    loud = 500                                                # beyond the reference tile
    bad = [17, 130, 201]
    d = hid[bad].mean(0)
    w[:, loud] = d / d.norm() * 3.0
    for r in bad:
        hid[r] = 6.0 * (0.2 * hid[r] + d / d.norm() * 8.0)    # z[r, loud] ~ 144, the rest ~ N(0, 1)
    ids[17] = 3 if int(ids[17]) == loud else ids[17]
    ids[130] = loud
    ids[201] = -1
    batch["hidden"] = hid.to(torch.bfloat16)
    batch["w_head"] = w.to(torch.bfloat16)
    batch["target_ids"] = ids
    z = batch["hidden"].float() @ batch["w_head"].float()
    for r in bad:
        assert float(z[r, loud] - z[r, :256].max()) > 100.0
    lp = torch.log_softmax(z.double(), -1).gather(1, ids.clamp(min=0).long()[:, None])[:, 0].float()
    batch["prox_lp"] = lp + 0.01 * torch.randn_like(lp)       # ratios near 1 also for the -140 nat token
    batch["behave_lp"] = batch["prox_lp"] + 0.01 * torch.randn_like(lp)
    params = dict(batch["params"], kernel=A.KERNEL_HEAD_2CTA_ROWREF)
    wh = batch["w_head"] if w_layout == A.W_K_BY_V else batch["w_head"].t().contiguous()
    gpu = A.awr_loss_fwd_bwd_fused_head(batch["hidden"], wh, batch["target_ids"], batch["behave_lp"],
                                        batch["prox_lp"], batch["step_off"], batch["traj_off"],
                                        batch["group_off"], batch["rewards"], w_layout=w_layout,
                                        want=A.api.HEAD_OPTIONAL_OUTPUTS + ("token_entropy",), **params)
    torch.cuda.synchronize()
    ora = _oracle_head(batch, want_entropy=True)
    assert ora["token_lp"][17] < -100.0 and ora["token_lp"][130] > -1e-6
    _check_head(gpu, ora, w_layout)
    H = gpu["token_entropy"].cpu().numpy().astype(np.float64)
    assert np.abs(H - ora["token_entropy"]).max() <= 1e-4
    assert torch.isfinite(gpu["dhidden"].float()).all() and torch.isfinite(gpu["dw_head"].float()).all()


def test_head_shapes_agree_bitwise_on_integers():
    """Both tcgen05 shapes see the same inputs: same integers, values within rounding."""
    batch = _head_batch(700, 128, 1512, seed=8, lp_mode="drift")
    a = _run_head(batch, kernel=A.KERNEL_HEAD_1CTA)
    b = _run_head(batch, kernel=A.KERNEL_HEAD_2CTA)
    assert (a["token_lp"] - b["token_lp"]).abs().max().item() <= 2e-6
    assert int(a["clip_count"][0]) == int(b["clip_count"][0])
    assert torch.equal(a["tok_coef"] == 0, b["tok_coef"] == 0)
    d = (a["dhidden"].float() - b["dhidden"].float()).abs().max().item()
    assert d <= 2.0 ** -7 * a["dhidden"].float().abs().max().item()


def test_head_dual_clip():
    """Eq. (2) through the fused head: same scalars code as the logits path."""
    batch = _head_batch(400, 128, 1000, seed=17, lp_mode="drift")
    q = batch["prox_lp"].clone()
    q[::5] -= 1.5
    batch["prox_lp"] = q
    gpu = _run_head(batch, dual_clip_c=3.0)
    ora = _oracle_head(batch, dual_clip_c=3.0)
    assert ora["dual_clip_count"] > 5
    assert np.abs(np.log(ora["ratio"][ora["ratio"] > 0]) - np.log(3.0)).min() > 1e-4
    _check_head(gpu, ora, A.W_K_BY_V)


def test_head_matches_logits_path():
    """The same batch through the logits entry point (fp32 logits = H W computed in fp32) gives
    the same integers and, within tolerance, the same per-token values."""
    batch = _head_batch(384, 128, 1024, seed=5, lp_mode="drift")
    gpu = _run_head(batch)
    z = (batch["hidden"].float() @ batch["w_head"].float()).contiguous()
    ref = A.awr_loss_fwd_bwd(z, batch["target_ids"], batch["behave_lp"], batch["prox_lp"],
                             batch["step_off"], batch["traj_off"], batch["group_off"],
                             batch["rewards"], **batch["params"])
    torch.cuda.synchronize()
    assert int(gpu["clip_count"][0]) == int(ref["clip_count"][0])
    assert torch.equal(gpu["tok_traj"], ref["tok_traj"])
    assert (gpu["token_lp"] - ref["token_lp"]).abs().max().item() <= 2e-5


def test_head_empty_and_status_codes():
    batch = _head_batch(128, 64, 256, seed=1)
    with pytest.raises(A.AwrError) as ei:        # K not a multiple of 64
        A.awr_loss_fwd_bwd_fused_head(batch["hidden"][:, :40].contiguous(),
                                      batch["w_head"][:40].contiguous(), batch["target_ids"],
                                      batch["behave_lp"], batch["prox_lp"], batch["step_off"],
                                      batch["traj_off"], batch["group_off"], batch["rewards"])
    assert ei.value.status == -2
    z = torch.zeros(0, dtype=torch.float32, device=DEV)
    zi = torch.zeros(0, dtype=torch.int32, device=DEV)
    off = torch.zeros(1, dtype=torch.int32, device=DEV)
    out = A.awr_loss_fwd_bwd_fused_head(torch.zeros(0, 64, dtype=torch.bfloat16, device=DEV),
                                        batch["w_head"], zi, z, z, off, off, off, z)
    torch.cuda.synchronize()
    assert float(out["loss"][0]) == 0.0 and int(out["clip_count"][0]) == 0
    assert not out["dw_head"].any()


def test_head_graph_capture_and_side_stream():
    """The fused-head call (tensor-map encodes on the host, 20+ launches, one memset) only
    enqueues work on the caller's stream: it runs on a side stream and replays from a CUDA graph
    with identical results."""
    batch = _head_batch(600, 128, 2056, seed=9, lp_mode="drift")
    call = A.HeadLossCall(batch["hidden"], batch["w_head"], batch["target_ids"], batch["behave_lp"],
                          batch["prox_lp"], batch["step_off"], batch["traj_off"], batch["group_off"],
                          batch["rewards"], **batch["params"])
    ref = {k: v.clone() for k, v in call.run().items()}
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    for v in call.out.values():
        v.zero_()
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        call.run(stream=s)
    s.synchronize()
    for k in ref:
        assert torch.equal(ref[k], call.out[k]), k
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


def _random_head_shapes(n, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    return [(int(rng.integers(1, 700)), 64 * int(rng.integers(1, 5)), 8 * int(rng.integers(1, 400)),
             int(rng.integers(0, 1000))) for _ in range(n)]


@pytest.mark.parametrize("n_tok,K,V,seed", _random_head_shapes(8, 7))
def test_head_random_shapes(n_tok, K, V, seed):
    """Seeded random (rows, K, V): ragged tiles in every dimension, rank-3 and rank-2 tensor maps
    (V a multiple of 64 or not), all three kernel modes."""
    batch = _head_batch(max(n_tok, 16), K, V, seed=seed, lp_mode="drift", masked_frac=0.02)
    ora = _oracle_head(batch, stale_cap=2.0)
    for kernel in HEAD_KERNELS + HEAD_PANEL_KERNELS:
        gpu = _run_head(batch, kernel=kernel, stale_cap=2.0)
        _check_head(gpu, ora, A.W_K_BY_V)
    gpu = _run_head(batch, A.W_V_BY_K, stale_cap=2.0)
    _check_head(gpu, ora, A.W_V_BY_K)


@pytest.mark.parametrize("kernel", HEAD_KERNELS + HEAD_PANEL_KERNELS)
def test_head_token_entropy(kernel):
    """Per-token entropy from the fused head: a third per-tile partial (sum e^{z-m} z) merged
    across the vocabulary tiles; |dH| <= 1e-4 against the oracle, 0 for masked tokens, and the
    other outputs unchanged by asking for it."""
    batch = _head_batch(700, 128, 3000, seed=33, lp_mode="drift", masked_frac=0.03)
    params = dict(batch["params"], kernel=kernel)
    args = (batch["hidden"], batch["w_head"], batch["target_ids"], batch["behave_lp"],
            batch["prox_lp"], batch["step_off"], batch["traj_off"], batch["group_off"], batch["rewards"])
    out = A.awr_loss_fwd_bwd_fused_head(*args, want=A.api.HEAD_OPTIONAL_OUTPUTS + ("token_entropy",), **params)
    ref = A.awr_loss_fwd_bwd_fused_head(*args, **params)
    torch.cuda.synchronize()
    ora = _oracle_head(batch, want_entropy=True)
    H = out["token_entropy"].cpu().numpy().astype(np.float64)
    assert np.abs(H - ora["token_entropy"]).max() <= 1e-4
    assert np.all(H[batch["target_ids"].cpu().numpy() < 0] == 0.0) and ora["token_entropy"].max() > 1.0
    for k in ("loss", "token_lp", "dhidden", "dw_head"):
        assert torch.equal(out[k], ref[k]), k


@pytest.mark.parametrize("K,n_tok", [(512, 700), (1024, 300)])
def test_head_wide_dhidden_tiles(K, n_tok):
    """K a multiple of 512: the dhidden GEMM of the CTA-pair modes runs on 256 x 512 tiles (one
    undoubled 512-column TMEM accumulator).  Against the oracle, and equal to the one-CTA mode
    within rounding."""
    batch = _head_batch(n_tok, K, 1512, seed=44, lp_mode="drift", masked_frac=0.02)
    ora = _oracle_head(batch, stale_cap=2.0)
    outs = {}
    for kernel in HEAD_KERNELS + HEAD_PANEL_KERNELS:
        outs[kernel] = _run_head(batch, kernel=kernel, stale_cap=2.0)
        _check_head(outs[kernel], ora, A.W_K_BY_V)
    d = (outs[A.KERNEL_HEAD_1CTA]["dhidden"].float() - outs[A.KERNEL_HEAD_2CTA]["dhidden"].float()).abs().max()
    assert float(d) <= 2.0 ** -7 * float(outs[A.KERNEL_HEAD_1CTA]["dhidden"].float().abs().max())


def test_head_two_threads_two_streams():
    """Two host threads call the stored-logits fused head at the same time, each on its own
    stream with its own buffers: side streams and fork / join events come from a pool keyed by
    the caller's stream, so neither call can wait on the other's event record.  Several panels
    per call (so that the fork / join path is exercised repeatedly); every output must be
    bit-identical to a single-threaded run of the same call."""
    import threading
    calls, refs = [], []
    for i in range(2):
        batch = _head_batch(19_300, 64, 512, seed=50 + i, n_groups=8, group_size=8, lp_mode="drift")
        call = A.HeadLossCall(batch["hidden"], batch["w_head"], batch["target_ids"], batch["behave_lp"],
                              batch["prox_lp"], batch["step_off"], batch["traj_off"], batch["group_off"],
                              batch["rewards"], **dict(batch["params"], kernel=A.KERNEL_HEAD_2CTA_STORED))
        refs.append({k: v.clone() for k, v in call.run().items()})
        calls.append(call)
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream() for _ in calls]
    errors = []

    def worker(i):
        try:
            for it in range(6):
                for v in calls[i].out.values():
                    with torch.cuda.stream(streams[i]):
                        v.zero_()
                calls[i].run(stream=streams[i])
                streams[i].synchronize()
                for k, v in refs[i].items():
                    if not torch.equal(v, calls[i].out[k]):
                        errors.append((i, it, k))
        except Exception as e:                      # noqa: BLE001 - reported below
            errors.append((i, repr(e)))

    th = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    torch.cuda.synchronize()
    assert not errors, errors


def test_second_device_if_visible():
    """Function attributes and occupancy answers are cached per device ordinal: a process that
    used cuda:0 must still be able to launch the large-shared-memory kernels on cuda:1."""
    if torch.cuda.device_count() < 2:
        pytest.skip("one GPU visible")
    outs = []
    for dev in ("cuda:0", "cuda:1"):
        with torch.cuda.device(dev):
            w = W.workload(1, n_groups=2, group_size=4, n_tok=200)
            batch = W.make_batch(w, seed=3, device=dev)
            o = A.awr_loss_fwd_bwd(batch["logits"], batch["target_ids"], batch["behave_lp"],
                                   batch["prox_lp"], batch["step_off"], batch["traj_off"],
                                   batch["group_off"], batch["rewards"], **batch["params"])
            hb = W.make_batch(W.workload(4, n_groups=4, group_size=4, n_tok=300, V=1000, hidden=128),
                              seed=3, device=dev)
            h = A.awr_loss_fwd_bwd_fused_head(hb["hidden"], hb["w_head"], hb["target_ids"], hb["behave_lp"],
                                              hb["prox_lp"], hb["step_off"], hb["traj_off"], hb["group_off"],
                                              hb["rewards"], **hb["params"])
            torch.cuda.synchronize(dev)
            outs.append((float(o["loss"][0]), float(h["loss"][0])))
    assert np.isfinite(outs).all()


def test_head_host_buffer_entry():
    """awr_loss_fwd_bwd_fused_head_host (the e2e leg of bench.py --config 4): host buffers in and
    out through the C ABI; same kernels as the device entry, so every output is bit-identical."""
    batch = _head_batch(700, 128, 2056, seed=23, lp_mode="drift", masked_frac=0.02)
    want = A.api.HEAD_OPTIONAL_OUTPUTS + ("token_entropy",)
    dev = A.awr_loss_fwd_bwd_fused_head(batch["hidden"], batch["w_head"], batch["target_ids"],
                                        batch["behave_lp"], batch["prox_lp"], batch["step_off"],
                                        batch["traj_off"], batch["group_off"], batch["rewards"],
                                        want=want, **dict(batch["params"], dual_clip_c=3.0))
    torch.cuda.synchronize()
    hin = [batch[k].cpu().pin_memory() for k in ("hidden", "w_head", "target_ids", "behave_lp", "prox_lp",
                                                 "step_off", "traj_off", "group_off", "rewards")]
    call = A.HostHeadLossCall(*hin, device=DEV, want=want, **dict(batch["params"], dual_clip_c=3.0))
    out = call.run()
    for k in ("loss", "clip_count", "dual_clip_count", "token_lp", "tok_term", "tok_coef", "tok_traj",
              "adv", "token_entropy", "err_word", "dhidden", "dw_head"):
        assert not out[k].is_cuda
        assert torch.equal(out[k], dev[k].cpu()), k
    assert call.h2d_bytes > 2 * (700 * 128 + 128 * 2056) and call.d2h_bytes > 2 * (700 * 128 + 128 * 2056)


def test_head_workspace_is_mode_aware():
    """include/awr.h: the workspace query takes the kernel; AUTO (row reference) and E16 keep 2 bytes
    per logit of one row panel - BASELINE.json configs[4] fits in 5 GB - the stored-fp32 mode needs
    three times that."""
    auto = A.head_workspace_bytes(32_768, 151_936, 2048, 3000, 256, 16)
    rowref = A.head_workspace_bytes(32_768, 151_936, 2048, 3000, 256, 16, A.KERNEL_HEAD_2CTA_ROWREF)
    e16 = A.head_workspace_bytes(32_768, 151_936, 2048, 3000, 256, 16, A.KERNEL_HEAD_2CTA_E16)
    stored = A.head_workspace_bytes(32_768, 151_936, 2048, 3000, 256, 16, A.KERNEL_HEAD_2CTA_STORED)
    assert e16 < auto == rowref <= 5 * 10 ** 9 < stored
    assert A.head_workspace_bytes(32_768, 151_936, 2048, 3000, 256, 16, A.KERNEL_CLUSTER_RF) == 0


@pytest.mark.parametrize("kernel", HEAD_KERNELS + HEAD_PANEL_KERNELS)
def test_red_zones_fused_head(kernel):
    """dhidden, dw_head and the workspace of the fused head between 4 KB zones of a byte pattern
    that must survive the call (stands in for compute-sanitizer memcheck, closed on this pool)."""
    PAT = 0x5A
    batch = _head_batch(600, 128, 2056, seed=19, lp_mode="drift", masked_frac=0.02)
    n_steps, n_traj, n_groups = (batch[k].numel() - 1 for k in ("step_off", "traj_off", "group_off"))
    need = A.head_workspace_bytes(600, 2056, 128, n_steps, n_traj, n_groups, kernel)
    need = (need + 255) // 256 * 256
    wsbuf = torch.empty(need + 8192, dtype=torch.uint8, device=DEV)
    wsbuf.fill_(PAT)
    off = 4096 + ((-(wsbuf.data_ptr() + 4096)) % 256)
    call = A.HeadLossCall(batch["hidden"], batch["w_head"], batch["target_ids"], batch["behave_lp"],
                          batch["prox_lp"], batch["step_off"], batch["traj_off"], batch["group_off"],
                          batch["rewards"], workspace=wsbuf[off:off + need],
                          **dict(batch["params"], kernel=kernel))
    guarded = {}
    for k in ("dhidden", "dw_head", "token_lp"):
        t = call.out[k]
        buf = torch.empty(t.numel() + 4096, dtype=t.dtype, device=DEV)
        buf.view(torch.uint8).fill_(PAT)
        view = buf[2048:2048 + t.numel()].view(t.shape)
        call.out[k] = view
        setattr(call.outs, k, view.data_ptr())
        guarded[k] = (buf, t.numel())
    call.run()
    torch.cuda.synchronize()
    assert int(call.out["err_word"][0]) == 0
    for k, (buf, n) in guarded.items():
        raw = buf.view(torch.uint8)
        esz = buf.element_size()
        assert bool((raw[:2048 * esz] == PAT).all()) and bool((raw[(2048 + n) * esz:] == PAT).all()), k
    assert bool((wsbuf[:off] == PAT).all()) and bool((wsbuf[off + need:] == PAT).all()), "workspace"
    ora = _oracle_head(batch)
    _check_head(call.out, ora, A.W_K_BY_V)
