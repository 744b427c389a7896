"""Shared comparison code of the GPU parity tests: runs the CUDA path through the binding
(C ABI) and the fp64 oracle on the same seeded bytes and compares element by element.

Bars (BASELINE.json north_star):
  bit-exact   tok_traj, target_logit, clip_count, dual_clip_count, err_word, the zero pattern of c_t
  token_lp    |d| <= 1e-4 absolute
  loss        |d| <= 1e-5 |loss| + 1e-6 sum_t |term_t|   (second term: conditioning floor, the
              advantages sum to zero per group so the loss is a difference of large sums)
  dlogits     bf16: |d| <= max(2 ulp_bf16(oracle), 1e-3 max_v |oracle row|); rows with c_t = 0
              must be all-bits-zero.  fp32: |d| <= 2e-5 |oracle| + 1e-5 rowmax.
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


def check_scalars(gpu, ora, rows=None):
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
        tol = LOSS_RTOL * abs(ora["loss"]) + LOSS_COND_FLOOR * np.abs(ora["term"]).sum()
        assert abs(float(g["loss"][0]) - ora["loss"]) <= tol + 1e-30, \
            "loss %r vs oracle %r (tol %g)" % (float(g["loss"][0]), ora["loss"], tol)


def check_dlogits(dl_gpu, ora, V, rows=None):
    """dl_gpu: torch tensor [n_tok, ld]; ora['dlogits'] holds ora['grad_rows'] rows."""
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


def full_check(batch, backward=True, **over):
    gpu = run_gpu(batch, backward=backward, **over)
    ora = run_oracle(batch, want_dlogits=backward, **over)
    check_scalars(gpu, ora)
    if backward:
        check_dlogits(gpu["dlogits"], ora, batch["V"])
    return gpu, ora
