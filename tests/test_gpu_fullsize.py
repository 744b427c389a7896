"""GPU parity at BASELINE.json's FULL sizes (configs 1-3: 40,960 / 65,536 / 131,072 rows of
V = 151,936 bf16; config 4: the fused head at 32,768 x 2048 x 151,936), in the launch
configuration bench.py times (kernel = AUTO, device buffers).

Per config:
  * ALL rows through the oracle's forward steps (O1..O7, O9: segment expansion, advantage,
    token_logprob on every row in 256-row chunks spread over the host's cores, token_terms, the
    sequential fp64 sum in token order): loss, clip_count, dual_clip_count, err_word, every
    token_lp, target_logit, tok_term, tok_coef (and with it every trigger flag) are compared
    with the GPU outputs at the bars of parity_util.  Only the gradient ROWS (O8, 10^10 fp64
    exps per config) are sampled:
  * sampled rows (first, last, the rows around every cluster-schedule wrap, random ones,
    masked / triggered / zero-advantage ones) go through the oracle's own step functions
    (O2..O8 of oracle/awr_oracle.py, the same ones its awr_loss_fwd_bwd chains) and are compared
    element by element at the usual bars;
  * properties that hold at any size cover every row: tok_traj against the oracle's expansion
    (exact), loss = -(sum of the per-token terms in token order) in fp64, clip_count = number of
    trigger-flagged tokens implied by tok_coef / tok_term, all-bits-zero gradient rows exactly
    where c_t = 0, every non-zero gradient row sums to ~0 (P8), and token_lp against the
    library log-softmax (torch, fp32) on all rows.
"""
import os
import time

import numpy as np
import pytest
import torch

import paper_2606_05597_b200 as A
from gen import workloads as W
from oracle import awr_oracle as O
import parity_util as P

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
N_SAMPLE = 160


@pytest.fixture(autouse=True, scope="module")
def _gpu():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (run them with gpurun)")
    assert torch.cuda.get_device_capability(0)[0] == 10, "sm_100 only"
    yield


def _sample_rows(n_tok, extra, rng):
    edge = [0, 1, n_tok - 2, n_tok - 1]
    for c in (74, 148):                      # row schedule wraps of the persistent kernels
        edge += [c - 1, c, c + 1, n_tok - c, n_tok - c - 1]
    rows = np.unique(np.clip(np.concatenate([
        np.asarray(edge), np.asarray(extra, dtype=np.int64),
        rng.integers(0, n_tok, size=N_SAMPLE)]), 0, n_tok - 1))
    return rows


def _oracle_on_rows(batch, rows, params):
    """Chain the oracle's step functions on a subset of rows (offsets are the full ones)."""
    so, to, go = (batch[k].cpu().numpy() for k in ("step_off", "traj_off", "group_off"))
    rewards = batch["rewards"].cpu().numpy()
    seg = O.segment_expand(so, to, go)
    adv = O.group_advantage(rewards, go, params.get("flags", 0))
    scale = O.traj_scale(so, to, go, params["k_norm"], params["normalizer"],
                         params.get("loss_scale", 1.0))
    idx = torch.as_tensor(rows, device=DEV)
    V = batch["V"]
    z = batch["logits"][idx][:, :V].float().cpu().numpy()          # exact widening of bf16
    y = batch["target_ids"][idx].cpu().numpy().astype(np.int64)
    q = batch["prox_lp"][idx].cpu().numpy()
    b = batch["behave_lp"][idx].cpu().numpy()
    tt = seg["tok_traj"][rows]
    valid = (y >= 0) & (y < V)
    lse, lp, zy = O.token_logprob(z, y)
    term, coef, trig, r, w, dual = O.token_terms(lp, q, b, adv[tt], scale[tt], params["clip_eps"],
                                                 params["stale_cap"], valid,
                                                 params.get("dual_clip_c", 0.0), want_dual=True)
    g = O.dlogits_rows(z, y, lse, coef)
    return dict(seg=seg, adv=adv, lp=lp, zy=zy, term=term, coef=coef, trig=trig | dual, dlogits=g,
                grad_rows=np.arange(rows.size), y=y)


def _logits_rows_fn(batch):
    V = batch["V"]
    z = batch["logits"]
    return lambda lo, hi: z[lo:hi, :V].float().cpu().numpy()       # exact widening of bf16


# config 2: "both normalizers, separate runs" (BASELINE.json configs[2])
@pytest.mark.parametrize("cfg,in_place,norm", [(1, False, None), (2, False, A.NORM_CONST_K),
                                               (2, False, A.NORM_PER_TRAJ), (3, True, None)])
def test_full_size_sampled(cfg, in_place, norm):
    w = W.workload(cfg)
    batch = W.make_batch(w, seed=100 + cfg, device=DEV, masked_frac=0.001 if cfg == 3 else 0.0)
    n_tok, V = batch["n_tok"], batch["V"]
    assert n_tok == w.n_tok and V == 151_936
    params = dict(batch["params"])
    if norm is not None:
        params["normalizer"] = norm
    if cfg == 3:
        params["dual_clip_c"] = 3.0                     # Eq. (2) as in the paper's GRPO runs (:461)
    rng = np.random.Generator(np.random.PCG64(cfg))
    masked = torch.nonzero(batch["target_ids"] < 0).flatten().cpu().numpy()[:8]
    rows = _sample_rows(n_tok, masked, rng)
    # the oracle reads the logits BEFORE the call: config 3 runs in place
    ora = _oracle_on_rows(batch, rows, params)
    t0 = time.perf_counter()
    ora_all = P.oracle_terms_all_rows(
        P.oracle_forward_all_rows(batch, params, _logits_rows_fn(batch)), batch, params)
    print("config %d: oracle forward over all %d rows in %.1f s on %d host cores" % (
        cfg, n_tok, time.perf_counter() - t0, len(os.sched_getaffinity(0))))

    assert A.select_kernel(V, batch["ld"], torch.bfloat16) == A.KERNEL_CLUSTER_RFS
    kw = dict(dlogits=batch["logits"]) if in_place else {}
    if in_place:
        ref_lp = None
    out = A.awr_loss_fwd_bwd(batch["logits"], batch["target_ids"], batch["behave_lp"],
                             batch["prox_lp"], batch["step_off"], batch["traj_off"],
                             batch["group_off"], batch["rewards"], V=V, **params, **kw)
    torch.cuda.synchronize()
    assert int(out["err_word"][0]) == 0
    dl = out["dlogits"]

    # ---- all rows against the oracle: loss, counts, every per-token scalar and trigger flag
    P.check_scalars(out, ora_all, label="full size config %d norm %d" % (cfg, params["normalizer"]))
    flags_all = (out["tok_coef"].cpu().numpy() == 0) & (out["tok_term"].cpu().numpy() != 0)
    assert np.array_equal(flags_all, ora_all["trig"] | ora_all["dual"]), "trigger flags, all rows"
    if cfg == 3:
        assert ora_all["clip_count"] > 0.1 * n_tok and ora_all["dual_clip_count"] >= 0

    # ---- all rows: integers and properties
    assert np.array_equal(out["tok_traj"].cpu().numpy(), ora["seg"]["tok_traj"].astype(np.int32))
    np.testing.assert_allclose(out["adv"].cpu().numpy(), ora["adv"], rtol=0, atol=4e-6)
    term_all = out["tok_term"].double().cpu().numpy()
    coef_all = out["tok_coef"].cpu().numpy()
    loss_seq = 0.0
    for t in term_all:                                   # token order, fp64 (O7)
        loss_seq -= t
    assert abs(float(out["loss"][0]) - loss_seq) <= 1e-6 * abs(loss_seq) + 1e-7 * np.abs(term_all).sum()
    # a triggered token has a non-zero term and a zero coefficient (A5); masked and
    # zero-advantage tokens have both zero
    trig_all = (coef_all == 0) & (term_all != 0)
    assert int(out["clip_count"][0]) + int(out["dual_clip_count"][0]) == int(trig_all.sum())
    if cfg == 3:
        rate = trig_all.mean()
        assert 0.10 < rate < 0.30, "config 3 should drive a clip-trigger rate of ~20 %%, got %g" % rate
    zero_rows = torch.as_tensor(coef_all == 0, device=DEV)
    for lo in range(0, n_tok, 4096):
        blk = dl[lo:lo + 4096, :V]
        nz = (blk.view(torch.int16) != 0).any(dim=1)
        assert torch.equal(nz, ~zero_rows[lo:lo + 4096]), "zero pattern of the gradient rows"
        s = blk.float().sum(dim=1)
        mx = blk.float().abs().amax(dim=1)
        assert bool((s.abs() <= 0.05 * mx + 1e-30).all()), "a gradient row does not sum to ~0 (P8)"

    # ---- sampled rows against the oracle, element by element
    sel = rows
    lp_gpu = out["token_lp"].cpu().numpy()[sel].astype(np.float64)
    assert np.abs(lp_gpu - ora["lp"]).max() <= P.LP_ATOL
    assert np.array_equal(out["target_logit"].cpu().numpy()[sel], ora["zy"].astype(np.float32))
    assert np.array_equal(coef_all[sel] == 0, ora["coef"] == 0)
    cs = np.abs(ora["coef"]).max()
    np.testing.assert_allclose(coef_all[sel], ora["coef"], rtol=2e-4, atol=1e-6 * cs + 1e-30)
    ts = np.abs(ora["term"]).max()
    np.testing.assert_allclose(term_all[sel], ora["term"], rtol=2e-4, atol=1e-6 * ts + 1e-30)
    flags_gpu = (coef_all[sel] == 0) & (term_all[sel] != 0)
    assert np.array_equal(flags_gpu, ora["trig"])
    sub = dl[torch.as_tensor(sel, device=DEV)]
    P.check_dlogits(sub, dict(dlogits=ora["dlogits"], grad_rows=ora["grad_rows"],
                              coef=ora["coef"]), V, y=ora["y"])

    # ---- all rows: token_lp against the library log-softmax (not possible after in-place)
    if not in_place:
        worst = 0.0
        for lo in range(0, n_tok, 2048):
            zf = batch["logits"][lo:lo + 2048, :V].float()
            y = batch["target_ids"][lo:lo + 2048].long()
            ok = y >= 0
            lp = torch.log_softmax(zf, dim=1).gather(1, y.clamp(min=0)[:, None])[:, 0]
            d = torch.where(ok, (lp - out["token_lp"][lo:lo + 2048]).abs(), torch.zeros_like(lp))
            worst = max(worst, float(d.max()))
        assert worst <= P.LP_ATOL


def test_full_size_fused_head_config4():
    """BASELINE.json configs[4] at full size (32,768 x 2048 x 151,936) in the launch configuration
    bench.py times (AUTO = CTA pairs, stored logits panel, 4 row panels).

    * sampled rows against the fp64 oracle: the oracle's own steps on H[rows] W (exact fp64
      product of the bf16 inputs): token_lp, coefficient zero pattern, and the dhidden rows
      dS_row W^T;
    * every row / every element against a library computation that shares nothing with the
      kernels (torch fp32 matmul with TF32 off + log_softmax, in row chunks): token_lp on all
      rows, dhidden and dw_head in full (relative Frobenius error <= 5e-3, DESIGN.md tolerances);
    * properties: loss = -(sum of per-token terms), clip_count from the per-token outputs."""
    w = W.workload(4)
    batch = W.make_batch(w, seed=104, device=DEV)
    n_tok, V, K = batch["n_tok"], batch["V"], w.hidden
    assert (n_tok, V, K) == (32_768, 151_936, 2048)
    params = dict(batch["params"])
    out = A.awr_loss_fwd_bwd_fused_head(batch["hidden"], batch["w_head"], batch["target_ids"],
                                        batch["behave_lp"], batch["prox_lp"], batch["step_off"],
                                        batch["traj_off"], batch["group_off"], batch["rewards"],
                                        **params)
    torch.cuda.synchronize()
    assert int(out["err_word"][0]) == 0
    H, Wh = batch["hidden"], batch["w_head"]

    # ---- all rows against the oracle's forward steps on the exact fp64 product H W (A17):
    # loss, clip_count, every token_lp / term / coefficient / trigger flag
    Hd = H.float().cpu().numpy().astype(np.float64)
    Wd = Wh.float().cpu().numpy().astype(np.float64)
    t0 = time.perf_counter()
    ora_all = P.oracle_terms_all_rows(
        P.oracle_forward_all_rows(batch, params, lambda lo, hi: Hd[lo:hi] @ Wd, n_threads=4,
                                  chunk=512), batch, params)
    print("config 4: oracle forward (fp64 GEMM + log-softmax) over all %d rows in %.1f s" % (
        n_tok, time.perf_counter() - t0))
    gp = {k: v for k, v in out.items() if k not in ("dhidden", "dw_head")}
    del ora_all["target_logit"]                        # not an output of the fused-head entry
    P.check_scalars(gp, ora_all, label="full size config 4")
    del Hd, Wd

    # ---- properties on all rows
    so, to, go = (batch[k].cpu().numpy() for k in ("step_off", "traj_off", "group_off"))
    seg = O.segment_expand(so, to, go)
    assert np.array_equal(out["tok_traj"].cpu().numpy(), seg["tok_traj"].astype(np.int32))
    term = out["tok_term"].double().cpu().numpy()
    coef = out["tok_coef"].cpu().numpy()
    assert abs(float(out["loss"][0]) + term.sum()) <= 1e-6 * abs(term.sum()) + 1e-7 * np.abs(term).sum()
    assert int(out["clip_count"][0]) == int(((coef == 0) & (term != 0)).sum())

    # ---- library reference on all rows (fp32, TF32 off)
    prev = torch.backends.cuda.matmul.allow_tf32
    torch.backends.cuda.matmul.allow_tf32 = False
    try:
        Wf = Wh.float()
        dW_ref = torch.zeros(K, V, dtype=torch.float32, device=DEV)
        dH_ref = torch.empty(n_tok, K, dtype=torch.float32, device=DEV)
        worst_lp = 0.0
        for lo in range(0, n_tok, 2048):
            hi = min(n_tok, lo + 2048)
            Hf = H[lo:hi].float()
            z = Hf @ Wf
            lsm = torch.log_softmax(z, dim=1)
            y = batch["target_ids"][lo:hi].long()
            lp = lsm.gather(1, y[:, None])[:, 0]
            worst_lp = max(worst_lp, float((lp - out["token_lp"][lo:hi]).abs().max()))
            dS = torch.exp(lsm)
            dS[torch.arange(hi - lo, device=DEV), y] -= 1.0
            dS *= out["tok_coef"][lo:hi, None]
            dH_ref[lo:hi] = dS @ Wf.t()
            dW_ref += Hf.t() @ dS
            del z, lsm, dS
    finally:
        torch.backends.cuda.matmul.allow_tf32 = prev
    assert worst_lp <= P.LP_ATOL
    for name, got, ref in (("dhidden", out["dhidden"].float(), dH_ref),
                           ("dw_head", out["dw_head"].float(), dW_ref)):
        fro = float((got - ref).norm() / ref.norm())
        mx = float((got - ref).abs().max() / ref.abs().max())
        assert fro <= 5e-3, "%s relative Frobenius error %.3e" % (name, fro)
        assert mx <= 1e-2, "%s max-abs error %.3e of max|ref|" % (name, mx)
    del dW_ref, Wf

    # ---- sampled rows against the oracle
    rng = np.random.Generator(np.random.PCG64(4))
    rows = np.unique(np.concatenate([[0, 1, 255, 256, 9471, 9472, 9473, 28415, 28416, n_tok - 1],
                                     rng.integers(0, n_tok, size=38)]))
    idx = torch.as_tensor(rows, device=DEV)
    Hs = H[idx].float().cpu().numpy().astype(np.float64)
    Ws = Wh.float().cpu().numpy().astype(np.float64)
    z = Hs @ Ws                                        # exact widening, fp64 product (A17)
    y = batch["target_ids"][idx].cpu().numpy().astype(np.int64)
    adv = O.group_advantage(batch["rewards"].cpu().numpy(), go, params.get("flags", 0))
    scale = O.traj_scale(so, to, go, params["k_norm"], params["normalizer"], params.get("loss_scale", 1.0))
    tt = seg["tok_traj"][rows]
    lse, lp, zy = O.token_logprob(z, y)
    t_, c_, trig, r_, w_ = O.token_terms(lp, batch["prox_lp"][idx].cpu().numpy(),
                                         batch["behave_lp"][idx].cpu().numpy(), adv[tt], scale[tt],
                                         params["clip_eps"], params["stale_cap"], np.ones(rows.size, bool))
    assert np.abs(out["token_lp"][idx].cpu().numpy().astype(np.float64) - lp).max() <= P.LP_ATOL
    assert np.array_equal(coef[rows] == 0, c_ == 0)
    np.testing.assert_allclose(coef[rows], c_, rtol=2e-4, atol=1e-6 * np.abs(c_).max() + 1e-30)
    dS = O.dlogits_rows(z, y, lse, c_)
    dH = dS @ Ws.T
    got = out["dhidden"][idx].float().cpu().numpy().astype(np.float64)
    fro = np.linalg.norm(got - dH) / max(np.linalg.norm(dH), 1e-300)
    assert fro <= 5e-3, "sampled dhidden rows: relative Frobenius error %.3e" % fro
