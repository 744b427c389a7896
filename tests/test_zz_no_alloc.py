"""awr_loss_fwd_bwd_static (include/awr.h): the entry point that allocates nothing - its workspace
is a fixed 1 MiB device array inside libawr.so - against the existing awr_loss_fwd_bwd with a
caller workspace, on the same seeded inputs, two calls in a row (the array keeps the previous
call's contents).  Collected last on purpose (pytest -x).  pytest -m gpu."""
import pytest
import torch

import paper_2606_05597_b200 as A
from gen import workloads as W
import parity_util as P

pytestmark = pytest.mark.gpu
DEV = "cuda:0"

FIELDS = ("token_lp", "adv", "tok_traj", "target_logit", "tok_term", "tok_coef")


def _args(batch):
    return [batch[k] for k in ("logits", "target_ids", "behave_lp", "prox_lp", "step_off", "traj_off",
                               "group_off", "rewards")]


def _compare(got, ref, V, label):
    """The tolerances of the parity tests (parity_util): 1e-4 on log-probs, 1e-5 relative on the
    loss, integers exact, gradient within 2 bf16 ulp / 1e-3 of the row max.  Both sides run the
    same deterministic kernels, so they are in fact expected to agree far inside those bars."""
    assert int(got["err_word"][0]) == int(ref["err_word"][0]) == 0, label
    assert int(got["clip_count"][0]) == int(ref["clip_count"][0]), label
    assert torch.equal(got["tok_traj"], ref["tok_traj"]), label
    for k in ("token_lp", "target_logit"):
        assert float((got[k] - ref[k]).abs().max()) <= P.LP_ATOL, (label, k)
    for k in ("adv", "tok_term", "tok_coef"):
        d = float((got[k] - ref[k]).abs().max())
        assert d <= P.LOSS_RTOL * max(1.0, float(ref[k].abs().max())), (label, k, d)
    lg, lr = float(got["loss"][0]), float(ref["loss"][0])
    assert abs(lg - lr) <= P.LOSS_RTOL * abs(lr) + P.LOSS_COND_FLOOR * float(ref["tok_term"].abs().sum()), label
    g = got["dlogits"][:, :V].double()
    r = ref["dlogits"][:, :V].double()
    tol = 1e-3 * r.abs().amax(dim=1, keepdim=True)
    if got["dlogits"].dtype == torch.bfloat16:      # 2 bf16 ulp at |r| (parity_util.bf16_ulp, in torch)
        ulp = torch.exp2(torch.floor(torch.log2(r.abs().clamp_min(2.0 ** -126))) - 7)
        tol = torch.maximum(tol.expand_as(r), 2.0 * ulp)
    assert bool(((g - r).abs() <= tol).all()), label


def _both(batch, label):
    V = batch["V"]
    ref = A.awr_loss_fwd_bwd(*_args(batch), V=V, **batch["params"])
    ref = {k: v.clone() for k, v in ref.items()}
    got = A.awr_loss_fwd_bwd_static(*_args(batch), V=V, **batch["params"])
    torch.cuda.synchronize()
    _compare(got, ref, V, label)
    return got


def test_static_entry_two_calls_in_a_row():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (run them with gpurun)")
    # call 1: the register-file cluster kernel (V = 151,936 bf16), 600 rows, padded row stride;
    # call 2: a SMALLER fp32 batch (config 0, generic kernel) right behind it on the same stream, so
    # that everything it reads from the shared array beyond its own prefix is call 1's leftovers
    w1 = W.workload(1, n_groups=3, n_tok=600)
    b1 = W.make_batch(w1, seed=4242, device=DEV, ld=w1.V + 64)
    w0 = W.workload(0)
    b0 = W.make_batch(w0, seed=7, device=DEV)
    g1 = _both(b1, "call 1 (config-1 laws, 600 rows)")
    g0 = _both(b0, "call 2 (config 0)")
    # and once more in the other order, prepared calls: nothing but enqueues inside run()
    c0 = A.StaticLossCall(*_args(b0), V=b0["V"], **b0["params"])
    c1 = A.StaticLossCall(*_args(b1), V=b1["V"], **b1["params"])
    torch.cuda.synchronize()
    a0 = torch.cuda.memory_allocated()
    for _ in range(2):
        o0 = {k: v.clone() for k, v in c0.run().items()}
        o1 = c1.run()
    torch.cuda.synchronize()
    for k in FIELDS + ("loss", "clip_count"):
        assert torch.equal(o0[k], g0[k]), k
        assert torch.equal(o1[k], g1[k]), k
    # (the padding columns >= V of a gradient row are never written: compare the V columns)
    assert torch.equal(o0["dlogits"][:, :b0["V"]], g0["dlogits"][:, :b0["V"]])
    assert torch.equal(o1["dlogits"][:, :b1["V"]], g1["dlogits"][:, :b1["V"]])
    del o0
    assert torch.cuda.memory_allocated() <= a0                   # run() allocated nothing that stayed


def test_static_entry_rejects_large_batches():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (run them with gpurun)")
    # 9 bytes per token: 120,000 tokens need more than 1 MiB; nothing may be launched or written
    assert A.workspace_bytes(120_000, 1024, 1, 1, 1) > A.STATIC_WS_BYTES
    n_tok, V = 120_000, 16
    logits = torch.zeros(n_tok, V, dtype=torch.bfloat16, device=DEV)
    zi = torch.zeros(n_tok, dtype=torch.int32, device=DEV)
    zf = torch.zeros(n_tok, dtype=torch.float32, device=DEV)
    off = torch.tensor([0, n_tok], dtype=torch.int32, device=DEV)
    one = torch.tensor([0, 1], dtype=torch.int32, device=DEV)
    rew = torch.ones(1, dtype=torch.float32, device=DEV)
    dl = torch.full_like(logits, 7.0)
    with pytest.raises(A.AwrError) as ei:
        A.awr_loss_fwd_bwd_static(logits, zi, zf, zf, off, one, one, rew, dlogits=dl)
    assert ei.value.status == -9 and "AWR_STATIC_WS_BYTES" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((dl == 7.0).all())
    # the workspace path takes the same batch
    out = A.awr_loss_fwd_bwd(logits, zi, zf, zf, off, one, one, rew)
    torch.cuda.synchronize()
    assert int(out["err_word"][0]) == 0
