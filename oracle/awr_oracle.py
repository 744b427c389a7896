"""fp64 CPU oracle for the AsyncWebRL token loss and its gradient over the vocabulary.

TEST INFRASTRUCTURE ONLY.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this file.
The product path (``paper_2606_05597_b200``) never imports it, shares no code, table
or constant with it, and has no CPU fallback.

What it computes is the *plain definition*, evaluated in float64 with numpy, one
statement per step of SURVEY.md section 8(c) (O1..O9), in the paper's notation:

  PAPER.md:57  Eq. (1)  J = E[ 1/(G k) sum_i sum_j sum_t min( (pi_theta/pi_behave) A_i ,
                              (pi_prox/pi_behave) clip(pi_theta/pi_prox, 1-eps, 1+eps) A_i ) ]
  PAPER.md:59           constant 1/k in place of 1/|tau_i|   (selectable here)
  PAPER.md:61           A_i = (r_i - mean(r)) / std(r), one value per trajectory
  PAPER.md:53, :63      pi_prox/pi_behave is an unclipped staleness weight; the clip is
                        centred on pi_prox

Symbols: z_t logits row, y_t target id, l_t = log pi_theta(y_t), q_t = log pi_prox(y_t),
b_t = log pi_behave(y_t), r_t = exp(l_t - q_t), w_t = exp(q_t - b_t).

Readings of silent / ambiguous points that
this file fixes: A1 (mean over groups: kappa_g = 1/(NG G_g)), A2 (population std, no eps
in the denominator, zero-variance group -> A = 0 exactly; sample std by flag), A3
(k_norm is its own scalar), A4 (stale_cap truncates w_t; <= 0 or inf = off), A5/A6
(trigger = clipped branch strictly smaller), A10 (empty steps count toward |tau_i|),
A13 (negative target id = masked token), A14 (thresholds are 1 -/+ float64(float32(eps))),
A7 (Eq. (2), is dimensionally garbled - "max[f(rho), c A]" with f a ratio;
read as the dual clip of Ye et al. 2020 that the text cites: with s_t the inner min of Eq. (1)
and rho = r_t, a token with A < 0 contributes max(s_t, c A); a *dual-clip hit* is c A > s_t
strictly, i.e. A < 0 and r_t > c; its gradient is zero.  c <= 1 = off = Eq. (1)).

Pins (tests/test_oracle_pins.py, ``-m "not gpu"``): P1..P12 of SURVEY.md 8(c) - closed
forms, a library softmax-cross-entropy gradient, finite differences, a literal
pure-Python loop, invariants.  The paper's *empirical* rates (0.3 % clip rate, "about 2x
when coupled") are **parity unpinned**: they need the paper's data.

No blocking, fusion or reordering: every function below is a direct transcription of the
formula it cites.  ``rows=`` arguments only *select* tokens (each row's result depends on
that row and per-token scalars alone), they do not change the arithmetic.
"""
from __future__ import annotations

import numpy as np

NORM_CONST_K = 0      # n_i = 1 / k_norm           (the paper's fix)
NORM_PER_TRAJ = 1     # n_i = 1 / |tau_i| (steps)  (standard multi-step GRPO)

FLAG_SAMPLE_STD = 1   # A2: divide by (G-1) instead of G
FLAG_SUCCESS_FILTER = 2  # RAFT++ baseline: A_i = 1[R_i > 0], group normalisation off
FLAG_SKIP_UNIFORM = 8  # dynamic sampling (DAPO): all-success / all-failure groups are
                       # skipped - zero advantage AND left out of the mean over groups
FLAG_COUPLED = 4      # coupled-ratio ablation: one pi_theta/pi_behave ratio, clip
                      # centred on it, no staleness weight (= Eq. (1) with pi_prox := pi_behave)

ERR_STEP_OFF = 1      # step_off not starting at 0 / decreasing / not ending at n_tok
ERR_TRAJ_OFF = 2      # traj_off  ... n_steps
ERR_GROUP_OFF = 4     # group_off ... n_traj
ERR_TARGET_RANGE = 8  # some target id >= V


# ----------------------------------------------------------------------------- O1
def check_offsets(step_off, traj_off, group_off, n_tok):
    """O1 (PAPER.md:61 hierarchy token -> step -> trajectory -> group).

    Each array must start at 0, be non-decreasing and end at the count of the level
    below.  Returns the error word (0 = fine)."""
    step_off = np.asarray(step_off, dtype=np.int64)
    traj_off = np.asarray(traj_off, dtype=np.int64)
    group_off = np.asarray(group_off, dtype=np.int64)
    n_steps = step_off.size - 1
    n_traj = traj_off.size - 1
    err = 0
    for arr, last, bit in ((step_off, n_tok, ERR_STEP_OFF),
                           (traj_off, n_steps, ERR_TRAJ_OFF),
                           (group_off, n_traj, ERR_GROUP_OFF)):
        bad = arr[0] != 0 or arr[-1] != last or np.any(np.diff(arr) < 0)
        if bad:
            err |= bit
    return err


def segment_expand(step_off, traj_off, group_off):
    """a0: token -> step -> trajectory -> group indices, |tau_i| and G_g."""
    step_off = np.asarray(step_off, dtype=np.int64)
    traj_off = np.asarray(traj_off, dtype=np.int64)
    group_off = np.asarray(group_off, dtype=np.int64)
    n_steps = step_off.size - 1
    n_traj = traj_off.size - 1
    n_groups = group_off.size - 1
    tok_step = np.repeat(np.arange(n_steps, dtype=np.int64), np.diff(step_off))
    step_traj = np.repeat(np.arange(n_traj, dtype=np.int64), np.diff(traj_off))
    traj_group = np.repeat(np.arange(n_groups, dtype=np.int64), np.diff(group_off))
    tok_traj = step_traj[tok_step]
    traj_steps = np.diff(traj_off)        # |tau_i| : steps, not tokens (PAPER.md:37 footnote 1)
    group_size = np.diff(group_off)       # G_g
    return dict(tok_step=tok_step, tok_traj=tok_traj, traj_group=traj_group,
                traj_steps=traj_steps, group_size=group_size)


def mixed_groups(rewards, group_off):
    """PAPER.md:63 dynamic sampling: a group is *mixed* if its rewards are not all equal
    (neither all-success nor all-failure); single-member and empty groups are not."""
    R = np.asarray(rewards)
    go = np.asarray(group_off)
    return np.array([bool(np.any(R[int(go[g]):int(go[g + 1])] != R[int(go[g])]))
                     if go[g + 1] > go[g] else False for g in range(go.size - 1)], dtype=bool)


# ----------------------------------------------------------------------------- O2
def group_advantage(rewards, group_off, flags=0):
    """O2: A_i = (r_i - mean(r)) / std(r) within each task group.

    Reading A2: population std; if every reward of the group has the same value (tested
    on the values, -0 == +0) or the group has one member, A_i = 0 exactly; no eps.
    FLAG_SUCCESS_FILTER (RAFT++): "group normalization disabled and the
    group-relative advantage replaced by a success filter (r > 0)": A_i = 1 if R_i > 0 else 0."""
    if flags & FLAG_SUCCESS_FILTER:
        adv = (np.asarray(rewards, dtype=np.float64) > 0.0).astype(np.float64)
        if flags & FLAG_SKIP_UNIFORM:
            mixed = mixed_groups(rewards, group_off)
            for g in range(np.asarray(group_off).size - 1):
                if not mixed[g]:
                    adv[int(group_off[g]):int(group_off[g + 1])] = 0.0
        return adv
    rewards = np.asarray(rewards, dtype=np.float64)
    group_off = np.asarray(group_off, dtype=np.int64)
    adv = np.zeros(rewards.size, dtype=np.float64)
    for g in range(group_off.size - 1):
        lo, hi = int(group_off[g]), int(group_off[g + 1])
        G = hi - lo
        if G <= 1:
            continue
        R = rewards[lo:hi]
        if np.all(R == R[0]):
            continue
        mu = R.sum() / G
        denom = (G - 1) if (flags & FLAG_SAMPLE_STD) else G
        sigma = np.sqrt(((R - mu) ** 2).sum() / denom)
        adv[lo:hi] = (R - mu) / sigma
    return adv


# ----------------------------------------------------------------------------- O3
def row_logsumexp(logits_rows):
    """O3: m = max_v z_v ; lse = m + log sum_v exp(z_v - m), per row, float64."""
    z = np.asarray(logits_rows, dtype=np.float64)
    m = z.max(axis=1)
    return m + np.log(np.exp(z - m[:, None]).sum(axis=1))


def token_logprob(logits_rows, target_ids):
    """O3 (PAPER.md:435 token-level IS): l_t = z[y_t] - lse.  Masked / out-of-range
    targets give (lse, 0, 0).  Returns lse, l_t, z[y_t]."""
    z = np.asarray(logits_rows, dtype=np.float64)
    y = np.asarray(target_ids, dtype=np.int64)
    V = z.shape[1]
    lse = row_logsumexp(z)
    ok = (y >= 0) & (y < V)
    zy = np.where(ok, z[np.arange(z.shape[0]), np.where(ok, y, 0)], 0.0)
    lp = np.where(ok, zy - lse, 0.0)
    return lse, lp, zy


def token_entropy(logits_rows):
    """Per-token entropy of the policy over the vocabulary, the paper's training diagnostic
    ("per-token entropy"): H_t = -sum_v p_v log p_v with p = softmax(z_t),
    evaluated as lse - sum_v p_v z_v; entries with z_v = -inf have p_v = 0 and contribute 0
    (the limit of p log p).  SURVEY.md 8(f) rank 2."""
    z = np.asarray(logits_rows, dtype=np.float64)
    lse = row_logsumexp(z)
    p = np.exp(z - lse[:, None])
    zp = np.where(p > 0.0, z, 0.0)
    return lse - (p * zp).sum(axis=1)


# ----------------------------------------------------------------------------- O4..O6, O8 scalar part
def token_terms(lp, prox_lp, behave_lp, adv_tok, scale_tok, clip_eps, stale_cap, valid,
                dual_clip_c=0.0, want_dual=False):
    """O4, O5 and the scalar part of O7/O8 for a set of tokens.

    lp = l_t, prox_lp = q_t, behave_lp = b_t, adv_tok = A_i of the token's trajectory,
    scale_tok = loss_scale * kappa_g * n_i (O6), valid = token is neither masked nor out of
    range.  Returns (term_t, c_t, trig_t, r_t, w_t) with
       term_t = scale * w_t * min(r_t A, clip(r_t) A)
       c_t    = scale * w_t * r_t * A   if the unclipped branch is active, else 0
       trig_t = clipped branch strictly smaller (A5, A6).
    dual_clip_c > 1 (Eq. (2), reading A7): for A < 0 the inner min s_t is
    capped from below, s_t <- max(s_t, c A); dual_t = (c A > s_t) strictly; such a token's
    term is constant in theta, so c_t = 0.  ``want_dual`` appends dual_t to the result."""
    lp = np.asarray(lp, dtype=np.float64)
    q = np.asarray(prox_lp, dtype=np.float64)
    b = np.asarray(behave_lp, dtype=np.float64)
    A = np.asarray(adv_tok, dtype=np.float64)
    scale = np.asarray(scale_tok, dtype=np.float64)
    eps = float(np.float32(clip_eps))                       # A14: the f32 eps, widened
    r = np.exp(lp - q)                                      # O4  pi_theta / pi_prox
    w = np.exp(q - b)                                       # O4  pi_prox / pi_behave
    cap = float(np.float32(stale_cap))
    if 0.0 < cap < np.inf:                                  # A4
        w = np.minimum(w, cap)
    u = r * A                                               # O5  unclipped branch (times w below)
    v = np.minimum(np.maximum(r, 1.0 - eps), 1.0 + eps) * A  # O5  clipped branch
    s = np.minimum(u, v)
    trig = v < u                                            # A5 / A6: strict
    dual = np.zeros(s.shape, dtype=bool)
    cdual = float(np.float32(dual_clip_c))
    if cdual > 1.0:                                         # Eq. (2), A7
        floor = cdual * A
        dual = (A < 0.0) & (floor > s)
        s = np.where(A < 0.0, np.maximum(s, floor), s)
    term = scale * w * s
    coef = np.where(trig | dual, 0.0, scale * w * r * A)    # O8
    valid = np.asarray(valid, dtype=bool)
    term = np.where(valid, term, 0.0)
    coef = np.where(valid, coef, 0.0)
    trig = trig & valid
    dual = dual & valid
    if want_dual:
        return term, coef, trig, r, w, dual
    return term, coef, trig, r, w


# ----------------------------------------------------------------------------- O8 row part
def dlogits_rows(logits_rows, target_ids, lse, coef):
    """O8: dlogits[t, v] = c_t * (exp(z_v - lse_t) - [v = y_t]).

    Derivative of O7: d(r_t A)/d l_t = r_t A, d l_t / d z_v = [v = y_t] - softmax_v, the
    clipped branch is constant in theta.  Rows with c_t = 0 are exactly zero."""
    z = np.asarray(logits_rows, dtype=np.float64)
    y = np.asarray(target_ids, dtype=np.int64)
    lse = np.asarray(lse, dtype=np.float64)
    coef = np.asarray(coef, dtype=np.float64)
    p = np.exp(z - lse[:, None])
    ok = (y >= 0) & (y < z.shape[1]) & (coef != 0.0)
    rows = np.nonzero(ok)[0]
    p[rows, y[rows]] -= 1.0
    g = coef[:, None] * p
    g[coef == 0.0, :] = 0.0
    return g


# ----------------------------------------------------------------------------- the whole path
def traj_scale(step_off, traj_off, group_off, k_norm, normalizer, loss_scale, rewards=None,
               flags=0):
    """O6: scale_i = loss_scale * kappa_g * n_i with kappa_g = 1/(NG G_g) (A1) and
    n_i = 1/k_norm or 1/|tau_i|."""
    seg = segment_expand(step_off, traj_off, group_off)
    n_groups = np.asarray(group_off).size - 1
    G = seg["group_size"][seg["traj_group"]].astype(np.float64)
    if flags & FLAG_SKIP_UNIFORM:             # the batch is the mixed groups only
        n_groups = int(mixed_groups(rewards, group_off).sum())
        if n_groups == 0:
            return np.zeros(G.size, dtype=np.float64)
    kappa = 1.0 / (n_groups * G)
    if normalizer == NORM_CONST_K:
        n_i = np.full(G.size, 1.0 / float(np.float32(k_norm)))
    elif normalizer == NORM_PER_TRAJ:
        steps = seg["traj_steps"].astype(np.float64)
        n_i = np.where(steps > 0, 1.0 / np.maximum(steps, 1.0), 0.0)
    else:
        raise ValueError("normalizer")
    return float(np.float32(loss_scale)) * kappa * n_i


def awr_loss_fwd_bwd(logits, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                     rewards, *, k_norm, clip_eps, stale_cap, normalizer, flags=0,
                     loss_scale=1.0, dual_clip_c=0.0, want_dlogits=True, grad_rows=None,
                     want_entropy=False):
    """The whole hot path a0..a4 for one batch.

    logits: [n_tok, V] array of the *exact* input values (bf16 widened exactly by the
    caller).  grad_rows: optional index array; if given, dlogits is returned for those rows
    only (shape [len(grad_rows), V]).  loss = -sum_t term_t, summed in token order (O7);
    ``term`` in the result is the per-token contribution to J (so loss = -term.sum())."""
    z = np.asarray(logits)
    n_tok, V = z.shape
    y = np.asarray(target_ids, dtype=np.int64)
    err = check_offsets(step_off, traj_off, group_off, n_tok)                     # O1
    if np.any(y >= V):
        err |= ERR_TARGET_RANGE
    seg = segment_expand(step_off, traj_off, group_off)                          # a0
    adv = group_advantage(rewards, group_off, flags)                              # O2
    scale = traj_scale(step_off, traj_off, group_off, k_norm, normalizer, loss_scale,
                       rewards, flags)                                            # O6
    tok_traj = seg["tok_traj"]
    valid = (y >= 0) & (y < V)
    lse = np.empty(n_tok, dtype=np.float64)
    lp = np.empty(n_tok, dtype=np.float64)
    zy = np.empty(n_tok, dtype=np.float64)
    ent = np.zeros(n_tok, dtype=np.float64)
    step = max(1, (1 << 24) // max(V, 1))             # row panels: memory only, same arithmetic
    for lo in range(0, n_tok, step):
        hi = min(n_tok, lo + step)
        lse[lo:hi], lp[lo:hi], zy[lo:hi] = token_logprob(z[lo:hi], y[lo:hi])    # O3
        if want_entropy:
            ent[lo:hi] = np.where(valid[lo:hi], token_entropy(z[lo:hi]), 0.0)    # 0 for masked tokens
    if flags & FLAG_COUPLED:                  # the single ratio pi_theta / pi_behave
        prox_lp = behave_lp
    term, coef, trig, r, w, dual = token_terms(lp, prox_lp, behave_lp, adv[tok_traj],
                                               scale[tok_traj], clip_eps, stale_cap, valid,
                                               dual_clip_c, want_dual=True)       # O4..O6, Eq. (2)
    loss = 0.0
    for t in range(n_tok):                                                        # O7: token order
        loss -= term[t]
    out = dict(loss=loss, token_lp=lp, clip_count=int(trig.sum()), adv=adv,       # O9
               tok_traj=tok_traj, target_logit=zy, lse=lse, term=term, coef=coef,
               trig=trig, ratio=r, stale_w=w, err_word=err, traj_scale=scale,
               dual=dual, dual_clip_count=int(dual.sum()))
    if want_entropy:
        out["token_entropy"] = ent
    if want_dlogits:
        rows = np.arange(n_tok) if grad_rows is None else np.asarray(grad_rows, dtype=np.int64)
        g = np.empty((rows.size, V), dtype=np.float64)
        for lo in range(0, rows.size, step):
            sel = rows[lo:lo + step]
            g[lo:lo + step] = dlogits_rows(z[sel], y[sel], lse[sel], coef[sel])  # O8
        out["dlogits"] = g
        out["grad_rows"] = rows
    return out


# ----------------------------------------------------------------------------- fused LM head (a5)
def awr_loss_fwd_bwd_fused_head(hidden, w_head, target_ids, behave_lp, prox_lp, step_off,
                                traj_off, group_off, rewards, **params):
    """a5 (BASELINE.json config 4; the paper is silent on the LM head): logits are the
    exact float64 product of the (bf16-valued) hidden [n_tok, K] and W [K, V] (reading
    A17: no bf16 round trip), then the token oracle; dH = dS W^T, dW = H^T dS with
    dS = dlogits.  The contraction uses the library float64 GEMM (numpy.matmul)."""
    H = np.asarray(hidden, dtype=np.float64)
    W = np.asarray(w_head, dtype=np.float64)
    z = H @ W
    out = awr_loss_fwd_bwd(z, target_ids, behave_lp, prox_lp, step_off, traj_off, group_off,
                           rewards, **params)
    dS = out.pop("dlogits")
    out["dhidden"] = dS @ W.T
    out["dw_head"] = H.T @ dS
    out["logits"] = z
    return out
