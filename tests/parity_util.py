"""Shared comparison code of the GPU parity tests: runs the CUDA path through the binding
(C ABI) and the fp64 oracle on the same seeded bytes and compares element by element.

Bars (BASELINE.json north_star):
  bit-exact   tok_traj, target_logit, clip_count, dual_clip_count, err_word, the zero pattern of c_t
  token_lp    |d| <= 1e-4 absolute
  loss        |d| <= 1e-5 |loss| + 1e-6 sum_t |term_t|   (second term: conditioning floor, the
              advantages sum to zero per group so the loss is a difference of large sums)
  dlogits     bf16: |d| <= max(2 ulp_bf16(oracle), 1e-3 max_v |oracle row|); rows with c_t = 0
              must be all-bits-zero.  fp32: |d| <= 2e-5 |oracle| + 1e-5 rowmax.
              Supplementary for bf16 (the 1e-3 rowmax floor hides most non-target entries at
              V = 151,936): the sum of the NON-TARGET entries of every row against the oracle's
              c_t (1 - p_y) within 8 sigma of independent bf16 roundings (catches a zeroed or
              mis-scaled part of a row); tests also compare the cluster kernels with the generic
              kernel element by element and run a peaked-logits workload.

Every loss comparison is logged (LOSS_LOG: conditioning sum|term| / |sum term|, and whether the
1e-5 |loss| term alone would have passed) and printed in pytest's terminal summary (conftest.py).
"""
from __future__ import annotations

import numpy as np
import torch

import paper_2606_05597_b200 as A
from gen import workloads as W
from oracle import awr_oracle as O

LP_ATOL = 1e-4
LOSS_RTOL = 1e-5
LOSS_COND_FLOOR = 1e-6
LOSS_COND_MIN = 100.0  # the floor applies only to sums at least this ill-conditioned
LOSS_LOG = []          # (label, |loss|, cond, |diff|, rel-only tolerance, passed on the rel term alone)


def check_loss(got, ora_loss, ora_term, label=""):
    """north_star: 1e-5 relative.  DESIGN.md section 3 adds the conditioning floor
    1e-6 sum|term_t| ONLY for batches whose advantages cancel almost exactly - conditioning
    sum|term| / |sum term| >= 100 (P3: config 0 at ratio 1 sums to 0 exactly; config 0 as drawn
    has conditioning 1,238).  Measured over the 156 loss comparisons of the GPU suite (round 2):
    151 pass on the 1e-5 term alone; the 5 that need the floor have conditioning 570 ... 3.8e9."""
    abs_sum = float(np.abs(ora_term).sum())
    diff = abs(float(got) - float(ora_loss))
    rel_tol = LOSS_RTOL * abs(float(ora_loss))
    cond = abs_sum / abs(float(ora_loss)) if ora_loss != 0 else float("inf")
    LOSS_LOG.append((label, abs(float(ora_loss)), cond, diff, rel_tol, diff <= rel_tol))
    tol = rel_tol + (LOSS_COND_FLOOR * abs_sum if cond >= LOSS_COND_MIN else 0.0)
    assert diff <= tol + 1e-30, "loss %r vs oracle %r (tol %g, conditioning %g)" % (
        float(got), float(ora_loss), tol, cond)


def bf16_ulp(x):
    """Spacing of bfloat16 (8 significand bits) at |x|, float64 array."""
    ax = np.abs(x)
    e = np.floor(np.log2(np.maximum(ax, 2.0 ** -126)))
    return 2.0 ** (e - 7)


def run_gpu(batch, backward=True, **over):
    params = dict(batch["params"])
    params.update(over)
    fn = A.awr_loss_fwd_bwd if backward else A.awr_loss_fwd
    out = fn(batch["logits"], batch["target_ids"], batch["behave_lp"], batch["prox_lp"],
             batch["step_off"], batch["traj_off"], batch["group_off"], batch["rewards"],
             V=batch["V"], **params)
    torch.cuda.synchronize()
    return out


def run_oracle(batch, grad_rows=None, want_dlogits=True, **over):
    host = W.to_host(batch)
    args, kw = W.oracle_args(host)
    kw.update(over)
    kw.pop("kernel", None)            # which row kernel runs is not the oracle's business
    return O.awr_loss_fwd_bwd(*args, want_dlogits=want_dlogits, grad_rows=grad_rows, **kw)


def check_scalars(gpu, ora, rows=None, label=""):
    """Everything except dlogits.  rows: compare per-token arrays on these rows only."""
    sel = slice(None) if rows is None else np.asarray(rows)
    g = {k: v.cpu().numpy() for k, v in gpu.items() if k != "dlogits"}
    if "tok_traj" in g:
        assert np.array_equal(g["tok_traj"][sel], ora["tok_traj"][sel].astype(np.int32))
    if "adv" in g:
        np.testing.assert_allclose(g["adv"], ora["adv"], rtol=0, atol=4e-6)
    if "target_logit" in g:
        assert np.array_equal(g["target_logit"][sel],
                              ora["target_logit"][sel].astype(np.float32))
    d_lp = np.abs(g["token_lp"][sel].astype(np.float64) - ora["token_lp"][sel])
    assert d_lp.max(initial=0.0) <= LP_ATOL, "token_lp off by %g" % d_lp.max()
    if "tok_term" in g:
        scale = np.abs(ora["term"][sel]).max(initial=0.0)
        np.testing.assert_allclose(g["tok_term"][sel], ora["term"][sel], rtol=2e-4,
                                   atol=1e-6 * scale + 1e-30)
    if "tok_coef" in g:
        assert np.array_equal(g["tok_coef"][sel] == 0, ora["coef"][sel] == 0), \
            "zero pattern of c_t (clip triggers / masked / zero advantage) differs"
        scale = np.abs(ora["coef"][sel]).max(initial=0.0)
        np.testing.assert_allclose(g["tok_coef"][sel], ora["coef"][sel], rtol=2e-4,
                                   atol=1e-6 * scale + 1e-30)
    if rows is None:
        assert int(g["clip_count"][0]) == ora["clip_count"], \
            "clip_count %d != oracle %d" % (int(g["clip_count"][0]), ora["clip_count"])
        if "err_word" in g:
            assert int(g["err_word"][0]) == ora["err_word"]
        if "dual_clip_count" in g:
            assert int(g["dual_clip_count"][0]) == ora["dual_clip_count"], \
                "dual_clip_count %d != oracle %d" % (int(g["dual_clip_count"][0]),
                                                     ora["dual_clip_count"])
        check_loss(g["loss"][0], ora["loss"], ora["term"], label)


def check_dlogits(dl_gpu, ora, V, rows=None, y=None):
    """dl_gpu: torch tensor [n_tok, ld]; ora['dlogits'] holds ora['grad_rows'] rows.
    y: target ids of ALL rows (numpy); enables the non-target row-sum check for bf16."""
    grows = ora["grad_rows"]
    G = ora["dlogits"]
    is_bf16 = dl_gpu.dtype == torch.bfloat16
    step = max(1, (1 << 25) // V)
    for lo in range(0, grows.size, step):
        idx = grows[lo:lo + step]
        got_t = dl_gpu[torch.as_tensor(idx, device=dl_gpu.device)][:, :V]
        ref = G[lo:lo + step]
        zero_rows = ora["coef"][idx] == 0
        if zero_rows.any():
            raw = got_t[torch.as_tensor(zero_rows, device=got_t.device)]
            bits = raw.view(torch.int16 if is_bf16 else torch.int32)
            assert int(bits.count_nonzero()) == 0, "a c_t = 0 row is not all-bits-zero"
        got = got_t.float().cpu().numpy().astype(np.float64)
        rowmax = np.abs(ref).max(axis=1, keepdims=True)
        if is_bf16:
            tol = np.maximum(2.0 * bf16_ulp(ref), 1e-3 * rowmax)
        else:
            tol = 2e-5 * np.abs(ref) + 1e-5 * rowmax
        bad = np.abs(got - ref) > tol
        if bad.any():
            r, c = np.argwhere(bad)[0]
            raise AssertionError("dlogits[%d, %d] = %r, oracle %r, tol %g (%d bad)" % (
                idx[r], c, got[r, c], ref[r, c], tol[r, c] if tol.ndim == 2 else tol, bad.sum()))
        # P8 holds for the GPU result too: rows sum to ~0 relative to their size
        if not is_bf16:
            assert np.all(np.abs(got.sum(axis=1)) <= 1e-4 * rowmax[:, 0] + 1e-30)
        elif y is not None:
            # bf16: every entry is the oracle's value rounded at most twice (e, then e * F), i.e.
            # an independent error of std <= sqrt(2) ulp / sqrt(12) with ulp <= 2^-7 |entry|.
            # The non-target entries therefore sum to the oracle's c_t (1 - p_y) within
            # 8 sigma = 8 sqrt(2) 2^-7 / sqrt(12) ||non-target row||_2 (+ 1e-6 for the lse).
            yy = np.asarray(y)[idx].astype(np.int64)
            ok = (yy >= 0) & (yy < V)
            r = np.arange(idx.size)
            g_nt, r_nt = got.copy(), ref.copy()
            g_nt[r[ok], yy[ok]] = 0.0
            r_nt[r[ok], yy[ok]] = 0.0
            bound = 8.0 * np.sqrt(2.0 / 12.0) * 2.0 ** -7 * np.sqrt((r_nt ** 2).sum(axis=1)) \
                + 1e-6 * np.abs(r_nt).sum(axis=1) + 1e-30
            d = np.abs(g_nt.sum(axis=1) - r_nt.sum(axis=1))
            assert np.all(d <= bound), "non-target row sum off: row %d, |d| %g > %g" % (
                idx[int(np.argmax(d / bound))], d.max(), bound[int(np.argmax(d / bound))])


def full_check(batch, backward=True, **over):
    gpu = run_gpu(batch, backward=backward, **over)
    ora = run_oracle(batch, want_dlogits=backward, **over)
    check_scalars(gpu, ora, label=batch.get("name", ""))
    if backward:
        check_dlogits(gpu["dlogits"], ora, batch["V"], y=batch["target_ids"].cpu().numpy())
    return gpu, ora


def oracle_forward_all_rows(batch, params, rows_fn, n_threads=None, chunk=256):
    """The oracle's forward steps over ALL rows of a full-size batch: O.token_logprob on row
    chunks (rows_fn(lo, hi) -> exact float32 / float64 logits of rows [lo, hi)), then one
    O.token_terms call over all tokens and the sequential fp64 sum in token order (O7).  Row
    chunks only bound memory and let the host's cores work side by side (numpy releases the GIL
    inside exp / sum); every row goes through the unchanged oracle functions."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    so, to, go = (batch[k].cpu().numpy() for k in ("step_off", "traj_off", "group_off"))
    rewards = batch["rewards"].cpu().numpy()
    n_tok, V = batch["n_tok"], batch["V"]
    flags = params.get("flags", 0)
    seg = O.segment_expand(so, to, go)
    adv = O.group_advantage(rewards, go, flags)
    scale = O.traj_scale(so, to, go, params["k_norm"], params["normalizer"],
                         params.get("loss_scale", 1.0), rewards, flags)
    y = batch["target_ids"].cpu().numpy().astype(np.int64)
    lse = np.empty(n_tok)
    lp = np.empty(n_tok)
    zy = np.empty(n_tok)

    def work(lo):
        hi = min(n_tok, lo + chunk)
        lse[lo:hi], lp[lo:hi], zy[lo:hi] = O.token_logprob(rows_fn(lo, hi), y[lo:hi])

    n_threads = n_threads or max(1, min(32, len(os.sched_getaffinity(0))))
    with ThreadPoolExecutor(n_threads) as ex:
        list(ex.map(work, range(0, n_tok, chunk)))
    return dict(seg=seg, adv=adv, scale=scale, lse=lse, token_lp=lp, target_logit=zy, y=y,
                tok_traj=seg["tok_traj"], err_word=O.check_offsets(so, to, go, n_tok))


def oracle_terms_all_rows(fw, batch, params):
    """O4..O7, O9 on the result of oracle_forward_all_rows for one parameter set."""
    y, V = fw["y"], batch["V"]
    q = batch["prox_lp"].cpu().numpy()
    b = batch["behave_lp"].cpu().numpy()
    if params.get("flags", 0) & O.FLAG_COUPLED:
        q = b
    tt = fw["tok_traj"]
    valid = (y >= 0) & (y < V)
    term, coef, trig, r, w, dual = O.token_terms(fw["token_lp"], q, b, fw["adv"][tt], fw["scale"][tt],
                                                 params["clip_eps"], params["stale_cap"], valid,
                                                 params.get("dual_clip_c", 0.0), want_dual=True)
    loss = 0.0
    for t in range(term.size):                                   # O7: token order, fp64
        loss -= term[t]
    return dict(fw, term=term, coef=coef, trig=trig, ratio=r, stale_w=w, dual=dual, loss=loss,
                clip_count=int(trig.sum()), dual_clip_count=int(dual.sum()))
