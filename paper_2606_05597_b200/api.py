"""Python binding of libawr.so: the same entry points as include/awr.h, taking torch tensors.

Only marshals arguments (pointers, sizes, output / workspace allocation through torch's
allocator, the current CUDA stream).  Every step of the path - segment expansion, group
advantage, log-sum-exp + gather, decoupled ratio / clip / normalizer (Eq. 1,
PAPER.md:57-:59), the gradient write - runs in the CUDA kernels.
"""
from __future__ import annotations

import ctypes as C

import torch

from . import _abi
from ._abi import (DTYPE_BF16, DTYPE_F32, KERNEL_AUTO, NORM_CONST_K, awr_batch, awr_head_batch,
                   awr_head_outputs, awr_outputs, awr_params, check, load)

OPTIONAL_OUTPUTS = ("adv", "tok_traj", "target_logit", "tok_term", "tok_coef", "err_word")


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream_ptr(stream, device):
    s = torch.cuda.current_stream(device) if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _dtype_code(t):
    if t.dtype == torch.bfloat16:
        return DTYPE_BF16
    if t.dtype == torch.float32:
        return DTYPE_F32
    raise TypeError("logits must be bfloat16 or float32, got %s" % t.dtype)


def _req(t, dtype, name, cuda=True):
    if not torch.is_tensor(t) or t.dtype != dtype or not t.is_contiguous():
        raise TypeError("%s must be a contiguous %s tensor" % (name, dtype))
    if cuda and not t.is_cuda:
        raise TypeError("%s must live on the GPU (there is no CPU path)" % name)
    return t


def make_params(k_norm=10.0, clip_eps=0.2, stale_cap=0.0, normalizer=NORM_CONST_K, flags=0,
                loss_scale=1.0, kernel=KERNEL_AUTO, dual_clip_c=0.0) -> awr_params:
    return awr_params(float(k_norm), float(clip_eps), float(stale_cap), float(loss_scale),
                      float(dual_clip_c), int(normalizer), int(flags), int(kernel))


def workspace_bytes(n_tok, V, n_steps, n_traj, n_groups) -> int:
    return int(load().awr_workspace_bytes(n_tok, V, n_steps, n_traj, n_groups))


def alloc_outputs(n_tok, n_traj, device, like_logits=None, want=OPTIONAL_OUTPUTS):
    """Output tensors of awr_loss_fwd_bwd (dlogits only if like_logits is given)."""
    o = dict(loss=torch.empty(1, dtype=torch.float32, device=device),
             token_lp=torch.empty(n_tok, dtype=torch.float32, device=device),
             clip_count=torch.empty(1, dtype=torch.int64, device=device),
             dual_clip_count=torch.empty(1, dtype=torch.int64, device=device))
    if like_logits is not None:
        o["dlogits"] = torch.empty_like(like_logits)
    spec = dict(adv=(n_traj, torch.float32), tok_traj=(n_tok, torch.int32),
                target_logit=(n_tok, torch.float32), tok_term=(n_tok, torch.float32),
                tok_coef=(n_tok, torch.float32), err_word=(1, torch.int32),
                token_entropy=(n_tok, torch.float32))
    for k in want:
        n, dt = spec[k]
        o[k] = torch.empty(n, dtype=dt, device=device)
    return o


def _batch_struct(logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off, rewards,
                  V, cuda=True):
    if logits.dim() != 2 or logits.stride(1) != 1:
        raise TypeError("logits must be [n_tok, ld] with unit column stride")
    n_tok = logits.shape[0]
    ld = logits.stride(0) if n_tok > 1 else logits.shape[1]
    V = logits.shape[1] if V is None else int(V)
    if cuda and not logits.is_cuda:
        raise TypeError("logits must live on the GPU (there is no CPU path)")
    _req(target_ids, torch.int32, "target_ids", cuda)
    _req(behave_lp, torch.float32, "behave_lp", cuda)
    if prox_lp is not None:              # may be None with FLAG_COUPLED (not read)
        _req(prox_lp, torch.float32, "prox_lp", cuda)
    _req(step_off, torch.int32, "step_off", cuda)
    _req(traj_off, torch.int32, "traj_off", cuda)
    _req(group_off, torch.int32, "group_off", cuda)
    _req(rewards, torch.float32, "rewards", cuda)
    for t, name in ((target_ids, "target_ids"), (behave_lp, "behave_lp"), (prox_lp, "prox_lp")):
        if t is not None and t.numel() != n_tok:
            raise ValueError("%s must have n_tok = %d entries" % (name, n_tok))
    if traj_off.numel() != rewards.numel() + 1:
        raise ValueError("traj_off must have n_traj + 1 entries")
    b = awr_batch(n_tok, V, ld, _ptr(logits), _ptr(target_ids), _ptr(behave_lp), _ptr(prox_lp),
                  _ptr(step_off), _ptr(traj_off), _ptr(group_off), _ptr(rewards),
                  step_off.numel() - 1, traj_off.numel() - 1, group_off.numel() - 1,
                  _dtype_code(logits))
    return b


def _out_struct(o):
    g = o.get
    return awr_outputs(_ptr(g("loss")), _ptr(g("dlogits")), _ptr(g("token_lp")),
                       _ptr(g("clip_count")), _ptr(g("adv")), _ptr(g("tok_traj")),
                       _ptr(g("target_logit")), _ptr(g("tok_term")), _ptr(g("tok_coef")),
                       _ptr(g("err_word")), _ptr(g("dual_clip_count")), _ptr(g("token_entropy")),
                       None, None)


class LossCall:
    """One prepared awr_loss_fwd_bwd / awr_loss_fwd call: structs, outputs and workspace are
    built once, ``run()`` only enqueues the library call on the current stream (what bench.py
    times; CUDA-graph capturable)."""

    def __init__(self, logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                 rewards, *, V=None, backward=True, dlogits=None, out=None, workspace=None,
                 want=OPTIONAL_OUTPUTS, **params):
        self.lib = load()
        self.batch = _batch_struct(logits, target_ids, behave_lp, prox_lp, step_off, traj_off,
                                   group_off, rewards, V)
        self.params = make_params(**params)
        dev = logits.device
        self.device = dev
        self.backward = backward
        n_tok, n_traj = self.batch.n_tok, self.batch.n_traj
        self.out = out if out is not None else alloc_outputs(n_tok, n_traj, dev, None, want)
        if backward:
            if dlogits is not None:
                if dlogits.dtype != logits.dtype or dlogits.stride() != logits.stride():
                    raise TypeError("dlogits must match logits in dtype and strides")
                self.out["dlogits"] = dlogits
            elif "dlogits" not in self.out:
                self.out["dlogits"] = torch.empty_strided(logits.shape, logits.stride(),
                                                          dtype=logits.dtype, device=dev)
        need = workspace_bytes(n_tok, self.batch.V, self.batch.n_steps, n_traj,
                               self.batch.n_groups)
        self.workspace = workspace if workspace is not None else torch.empty(
            max(need, 256), dtype=torch.uint8, device=dev)
        self.ws_bytes = self.workspace.numel() * self.workspace.element_size()
        self.outs = _out_struct(self.out)
        self._keep = (logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                      rewards)
        self._fn = self.lib.awr_loss_fwd_bwd if backward else self.lib.awr_loss_fwd
        self._name = "awr_loss_fwd_bwd" if backward else "awr_loss_fwd"

    def run(self, stream=None, row_events=None):
        """``row_events``: optional pair of ``torch.cuda.Event(enable_timing=True)`` that have been
        recorded once (so that their handles exist); this call records them on its stream right
        around the row kernel (``awr_outputs.ev_row_begin / ev_row_end``)."""
        if row_events is not None:
            self.outs.ev_row_begin = row_events[0].cuda_event
            self.outs.ev_row_end = row_events[1].cuda_event
        try:
            rc = self._fn(C.byref(self.batch), C.byref(self.params), C.byref(self.outs),
                          _ptr(self.workspace), self.ws_bytes, _stream_ptr(stream, self.device))
        finally:
            if row_events is not None:
                self.outs.ev_row_begin = None
                self.outs.ev_row_end = None
        check(rc, self._name)
        return self.out


def awr_loss_fwd_bwd(logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                     rewards, **kw):
    """include/awr.h awr_loss_fwd_bwd.  Returns a dict of device tensors: loss [1], dlogits,
    token_lp, clip_count [1] and the optional per-token outputs (``want=``)."""
    return LossCall(logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                    rewards, backward=True, **kw).run()


class StaticLossCall:
    """include/awr.h awr_loss_fwd_bwd_static: awr_loss_fwd_bwd with the library's fixed 1 MiB
    device array as workspace (``STATIC_WS_BYTES``), for callers that cannot allocate.  Outputs
    are the caller's (``out=`` / ``dlogits=``; allocated here, once, if not given); ``run()``
    allocates nothing.  Every call on a GPU shares the array: calls that overlap on the GPU race."""

    def __init__(self, logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                 rewards, *, V=None, dlogits=None, out=None, want=OPTIONAL_OUTPUTS, **params):
        self.lib = load()
        self.batch = _batch_struct(logits, target_ids, behave_lp, prox_lp, step_off, traj_off,
                                   group_off, rewards, V)
        self.params = make_params(**params)
        self.device = logits.device
        n_tok, n_traj = self.batch.n_tok, self.batch.n_traj
        self.out = out if out is not None else alloc_outputs(n_tok, n_traj, self.device, None, want)
        if dlogits is not None:
            if dlogits.dtype != logits.dtype or dlogits.stride() != logits.stride():
                raise TypeError("dlogits must match logits in dtype and strides")
            self.out["dlogits"] = dlogits
        elif "dlogits" not in self.out:
            self.out["dlogits"] = torch.empty_strided(logits.shape, logits.stride(),
                                                      dtype=logits.dtype, device=self.device)
        self.outs = _out_struct(self.out)
        self._keep = (logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                      rewards)

    def run(self, stream=None):
        check(self.lib.awr_loss_fwd_bwd_static(C.byref(self.batch), C.byref(self.params),
                                               C.byref(self.outs), _stream_ptr(stream, self.device)),
              "awr_loss_fwd_bwd_static")
        return self.out


def awr_loss_fwd_bwd_static(logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                            rewards, **kw):
    """include/awr.h awr_loss_fwd_bwd_static (no workspace argument, no allocation in the call)."""
    return StaticLossCall(logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                          rewards, **kw).run()


def awr_loss_fwd(logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off, rewards,
                 **kw):
    """include/awr.h awr_loss_fwd (no gradient; each row is read once)."""
    return LossCall(logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                    rewards, backward=False, **kw).run()


def awr_group_advantage(rewards, group_off, flags=0, stream=None):
    """include/awr.h awr_group_advantage, kernel 1 alone."""
    _req(rewards, torch.float32, "rewards")
    _req(group_off, torch.int32, "group_off")
    adv = torch.empty_like(rewards)
    rc = load().awr_group_advantage(_ptr(rewards), _ptr(group_off), group_off.numel() - 1,
                                    rewards.numel(), int(flags), _ptr(adv),
                                    _stream_ptr(stream, rewards.device))
    check(rc, "awr_group_advantage")
    return adv


def select_kernel(V, ld, dtype) -> int:
    code = DTYPE_BF16 if dtype == torch.bfloat16 else DTYPE_F32
    return int(load().awr_select_kernel(V, ld, code))


def launches_per_call() -> int:
    return int(load().awr_launches_per_call())


# ------------------------------------------------------------------ host-buffer entry point
def host_workspace_bytes(n_tok, V, ld, dtype, n_steps, n_traj, n_groups) -> int:
    code = DTYPE_BF16 if dtype == torch.bfloat16 else DTYPE_F32
    return int(load().awr_host_workspace_bytes(n_tok, V, ld, code, n_steps, n_traj, n_groups))


class HostLossCall:
    """awr_loss_fwd_bwd_host: every tensor is a HOST tensor (pinned for full PCIe speed); the
    library stages row panels through ``dev_workspace`` and returns once the results are in
    the host buffers.  ``h2d_bytes`` / ``d2h_bytes`` are the bytes one call copies."""

    def __init__(self, logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                 rewards, *, device, V=None, dlogits=None, pin=True, want=("err_word",),
                 **params):
        self.lib = load()
        for t in (logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off, rewards):
            if t is not None and t.is_cuda:
                raise TypeError("awr_loss_fwd_bwd_host takes host tensors")
        self.batch = _batch_struct(logits, target_ids, behave_lp, prox_lp, step_off, traj_off,
                                   group_off, rewards, V, cuda=False)
        self.params = make_params(**params)
        self.device = torch.device(device)
        n_tok, n_traj = self.batch.n_tok, self.batch.n_traj
        self.out = alloc_outputs(n_tok, n_traj, "cpu", None, want)
        if pin:                           # small arrays: a pinned copy is cheap
            self.out = {k: v.pin_memory() for k, v in self.out.items()}
        self.out["dlogits"] = dlogits if dlogits is not None else torch.empty_strided(
            logits.shape, logits.stride(), dtype=logits.dtype, pin_memory=pin)
        self.outs = _out_struct(self.out)
        need = host_workspace_bytes(n_tok, self.batch.V, self.batch.ld, logits.dtype,
                                    self.batch.n_steps, n_traj, self.batch.n_groups)
        self.workspace = torch.empty(max(need, 256), dtype=torch.uint8, device=self.device)
        self._keep = (logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                      rewards)
        esz = logits.element_size()
        small_in = 12 * n_tok + 4 * (self.batch.n_steps + self.batch.n_traj +
                                     self.batch.n_groups + 3) + 4 * n_traj
        self.h2d_bytes = n_tok * self.batch.ld * esz + small_in
        small_out = 4 * n_tok + 20 + sum(self.out[k].numel() * self.out[k].element_size()
                                         for k in want)
        self.d2h_bytes = n_tok * self.batch.ld * esz + small_out

    def run(self, stream=None):
        with torch.cuda.device(self.device):
            rc = self.lib.awr_loss_fwd_bwd_host(
                C.byref(self.batch), C.byref(self.params), C.byref(self.outs),
                _ptr(self.workspace), self.workspace.numel(),
                _stream_ptr(stream, self.device))
        check(rc, "awr_loss_fwd_bwd_host")
        return self.out


def awr_loss_fwd_bwd_host(logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                          rewards, **kw):
    return HostLossCall(logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                        rewards, **kw).run()


# ---------------------------------------------------------------------------- a5: fused LM head
HEAD_OPTIONAL_OUTPUTS = ("adv", "tok_traj", "tok_term", "tok_coef", "err_word")


def head_workspace_bytes(n_tok, V, K, n_steps, n_traj, n_groups, kernel=KERNEL_AUTO) -> int:
    return int(load().awr_head_workspace_bytes(n_tok, V, K, n_steps, n_traj, n_groups, int(kernel)))


def head_launches_per_call(n_tok, V, K, kernel=KERNEL_AUTO) -> int:
    return int(load().awr_head_launches_per_call(n_tok, V, K, int(kernel)))


class HeadLossCall:
    """One prepared awr_loss_fwd_bwd_fused_head call (hidden states + W_head instead of logits;
    the logits live only in tensor memory).  ``run()`` enqueues it on the current stream."""

    def __init__(self, hidden, w_head, target_ids, behave_lp, prox_lp, step_off, traj_off,
                 group_off, rewards, *, w_layout=_abi.W_K_BY_V, want=HEAD_OPTIONAL_OUTPUTS,
                 workspace=None, **params):
        self.lib = load()
        _req(hidden, torch.bfloat16, "hidden")
        _req(w_head, torch.bfloat16, "w_head")
        if hidden.dim() != 2 or w_head.dim() != 2:
            raise TypeError("hidden must be [n_tok, K] and w_head [K, V] or [V, K]")
        n_tok, K = hidden.shape
        if w_layout == _abi.W_K_BY_V:
            if w_head.shape[0] != K:
                raise ValueError("w_head must be [K, V] for W_K_BY_V")
            V = w_head.shape[1]
        else:
            if w_head.shape[1] != K:
                raise ValueError("w_head must be [V, K] for W_V_BY_K")
            V = w_head.shape[0]
        for t, dt, name in ((target_ids, torch.int32, "target_ids"),
                            (behave_lp, torch.float32, "behave_lp"),
                            (prox_lp, torch.float32, "prox_lp"), (step_off, torch.int32, "step_off"),
                            (traj_off, torch.int32, "traj_off"), (group_off, torch.int32, "group_off"),
                            (rewards, torch.float32, "rewards")):
            _req(t, dt, name)
        if target_ids.numel() != n_tok or behave_lp.numel() != n_tok or prox_lp.numel() != n_tok:
            raise ValueError("per-token arrays must have n_tok = %d entries" % n_tok)
        dev = hidden.device
        self.device = dev
        n_steps, n_traj, n_groups = step_off.numel() - 1, traj_off.numel() - 1, group_off.numel() - 1
        self.batch = awr_head_batch(n_tok, V, K, _ptr(hidden), _ptr(w_head), _ptr(target_ids),
                                    _ptr(behave_lp), _ptr(prox_lp), _ptr(step_off), _ptr(traj_off),
                                    _ptr(group_off), _ptr(rewards), n_steps, n_traj, n_groups,
                                    int(w_layout))
        self.params = make_params(**params)
        o = dict(loss=torch.empty(1, dtype=torch.float32, device=dev),
                 dhidden=torch.empty_like(hidden), dw_head=torch.empty_like(w_head),
                 token_lp=torch.empty(n_tok, dtype=torch.float32, device=dev),
                 clip_count=torch.empty(1, dtype=torch.int64, device=dev),
                 dual_clip_count=torch.empty(1, dtype=torch.int64, device=dev))
        spec = dict(adv=(n_traj, torch.float32), tok_traj=(n_tok, torch.int32),
                    tok_term=(n_tok, torch.float32), tok_coef=(n_tok, torch.float32),
                    err_word=(1, torch.int32), token_entropy=(n_tok, torch.float32))
        for k in want:
            n, dt = spec[k]
            o[k] = torch.empty(n, dtype=dt, device=dev)
        self.out = o
        g = o.get
        self.outs = awr_head_outputs(_ptr(g("loss")), _ptr(g("dhidden")), _ptr(g("dw_head")),
                                     _ptr(g("token_lp")), _ptr(g("clip_count")), _ptr(g("adv")),
                                     _ptr(g("tok_traj")), _ptr(g("tok_term")), _ptr(g("tok_coef")),
                                     _ptr(g("err_word")), _ptr(g("dual_clip_count")),
                                     _ptr(g("token_entropy")))
        need = head_workspace_bytes(n_tok, V, K, n_steps, n_traj, n_groups, self.params.kernel)
        self.workspace = workspace if workspace is not None else torch.empty(
            max(need, 256), dtype=torch.uint8, device=dev)
        self.ws_bytes = self.workspace.numel()
        self.launches = head_launches_per_call(n_tok, V, K, self.params.kernel)
        self._keep = (hidden, w_head, target_ids, behave_lp, prox_lp, step_off, traj_off,
                      group_off, rewards)

    def run(self, stream=None):
        rc = self.lib.awr_loss_fwd_bwd_fused_head(
            C.byref(self.batch), C.byref(self.params), C.byref(self.outs), _ptr(self.workspace),
            self.ws_bytes, _stream_ptr(stream, self.device))
        check(rc, "awr_loss_fwd_bwd_fused_head")
        return self.out


def awr_loss_fwd_bwd_fused_head(hidden, w_head, target_ids, behave_lp, prox_lp, step_off, traj_off,
                                group_off, rewards, stream=None, **kw):
    """loss, dhidden, dw_head, token_lp, clip_count (+ optional per-token outputs) as a dict."""
    return HeadLossCall(hidden, w_head, target_ids, behave_lp, prox_lp, step_off, traj_off,
                        group_off, rewards, **kw).run(stream)


def head_host_workspace_bytes(n_tok, V, K, n_steps, n_traj, n_groups, kernel=KERNEL_AUTO) -> int:
    return int(load().awr_head_host_workspace_bytes(n_tok, V, K, n_steps, n_traj, n_groups, int(kernel)))


class HostHeadLossCall:
    """awr_loss_fwd_bwd_fused_head_host: every tensor is a HOST tensor (pinned for full PCIe
    speed); the library copies them into ``workspace`` on the device, runs the fused head there
    and returns once dhidden, dw_head, loss, token_lp (+ optional outputs) are in the host
    buffers.  ``h2d_bytes`` / ``d2h_bytes`` are the bytes one call copies."""

    def __init__(self, hidden, w_head, target_ids, behave_lp, prox_lp, step_off, traj_off,
                 group_off, rewards, *, device, w_layout=_abi.W_K_BY_V, want=("err_word",),
                 workspace=None, pin=True, **params):
        self.lib = load()
        host = (hidden, w_head, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off, rewards)
        for t in host:
            if t is not None and t.is_cuda:
                raise TypeError("awr_loss_fwd_bwd_fused_head_host takes host tensors")
        _req(hidden, torch.bfloat16, "hidden", cuda=False)
        _req(w_head, torch.bfloat16, "w_head", cuda=False)
        n_tok, K = hidden.shape
        V = w_head.shape[1] if w_layout == _abi.W_K_BY_V else w_head.shape[0]
        n_steps, n_traj, n_groups = step_off.numel() - 1, traj_off.numel() - 1, group_off.numel() - 1
        self.device = torch.device(device)
        self.batch = awr_head_batch(n_tok, V, K, _ptr(hidden), _ptr(w_head), _ptr(target_ids),
                                    _ptr(behave_lp), _ptr(prox_lp), _ptr(step_off), _ptr(traj_off),
                                    _ptr(group_off), _ptr(rewards), n_steps, n_traj, n_groups,
                                    int(w_layout))
        self.params = make_params(**params)
        mk = (lambda *a, **k: torch.empty(*a, **k).pin_memory()) if pin else torch.empty
        o = dict(loss=mk(1, dtype=torch.float32), dhidden=mk(hidden.shape, dtype=torch.bfloat16),
                 dw_head=mk(w_head.shape, dtype=torch.bfloat16), token_lp=mk(n_tok, dtype=torch.float32),
                 clip_count=mk(1, dtype=torch.int64), dual_clip_count=mk(1, dtype=torch.int64))
        spec = dict(adv=(n_traj, torch.float32), tok_traj=(n_tok, torch.int32),
                    tok_term=(n_tok, torch.float32), tok_coef=(n_tok, torch.float32),
                    err_word=(1, torch.int32), token_entropy=(n_tok, torch.float32))
        for k in want:
            nn, dt = spec[k]
            o[k] = mk(nn, dtype=dt)
        self.out = o
        g = o.get
        self.outs = awr_head_outputs(_ptr(g("loss")), _ptr(g("dhidden")), _ptr(g("dw_head")),
                                     _ptr(g("token_lp")), _ptr(g("clip_count")), _ptr(g("adv")),
                                     _ptr(g("tok_traj")), _ptr(g("tok_term")), _ptr(g("tok_coef")),
                                     _ptr(g("err_word")), _ptr(g("dual_clip_count")),
                                     _ptr(g("token_entropy")))
        need = head_host_workspace_bytes(n_tok, V, K, n_steps, n_traj, n_groups, self.params.kernel)
        if workspace is not None and workspace.numel() >= need:
            self.workspace = workspace
        else:
            self.workspace = torch.empty(max(need, 256), dtype=torch.uint8, device=self.device)
        self._keep = host
        small_in = 12 * n_tok + 4 * (n_steps + n_traj + n_groups + 3) + 4 * n_traj
        self.h2d_bytes = 2 * (n_tok * K + K * V) + small_in
        self.d2h_bytes = 2 * (n_tok * K + K * V) + 4 * n_tok + 20 + sum(
            o[k].numel() * o[k].element_size() for k in want)

    def run(self, stream=None):
        with torch.cuda.device(self.device):
            rc = self.lib.awr_loss_fwd_bwd_fused_head_host(
                C.byref(self.batch), C.byref(self.params), C.byref(self.outs), _ptr(self.workspace),
                self.workspace.numel(), _stream_ptr(stream, self.device))
        check(rc, "awr_loss_fwd_bwd_fused_head_host")
        return self.out


def awr_gemm_bf16(a, b, a_major=0, b_major=0, kernel=KERNEL_AUTO, stream=None):
    """C = A B on the tcgen05 engine of the fused head.  `a` is stored [M, Kc] (a_major 0) or
    [Kc, M] (a_major 1); `b` is stored [N, Kc] (b_major 0) or [Kc, N] (b_major 1)."""
    _req(a, torch.bfloat16, "a")
    _req(b, torch.bfloat16, "b")
    M, Kc = (a.shape[0], a.shape[1]) if a_major == 0 else (a.shape[1], a.shape[0])
    N, Kb = (b.shape[0], b.shape[1]) if b_major == 0 else (b.shape[1], b.shape[0])
    if Kc != Kb:
        raise ValueError("contraction lengths differ: %d vs %d" % (Kc, Kb))
    c = torch.empty((M, N), dtype=torch.bfloat16, device=a.device)
    rc = load().awr_gemm_bf16(_ptr(a), a_major, a.stride(0), _ptr(b), b_major, b.stride(0), M, N, Kc,
                              _ptr(c), c.stride(0), int(kernel), _stream_ptr(stream, a.device))
    check(rc, "awr_gemm_bf16")
    return c
