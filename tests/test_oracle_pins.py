"""Pins for the fp64 oracle: each test checks oracle/awr_oracle.py
against something other than itself - a closed form, a paper statement, a library routine,
finite differences, a literal pure-Python loop or an invariant.  CPU only."""
import math
import os

import numpy as np
import pytest
import torch

from gen import workloads as W
from oracle import awr_oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")


def golden():
    vals = {}
    for line in open(GOLDEN):
        line = line.split("#")[0].split()
        if len(line) == 2:
            vals[line[0]] = float(line[1])
    return vals


def small_batch(seed=0, V=48, cfg=1, **over):
    kw = dict(n_groups=3, group_size=4, n_tok=90, V=V, dtype=torch.float32)
    kw.update(over)
    w = W.workload(cfg, **kw)
    return W.to_host(W.make_batch(w, seed))


def run(host, **over):
    args, kw = W.oracle_args(host)
    kw.update(over)
    return O.awr_loss_fwd_bwd(*args, **kw)


# ------------------------------------------------------------------------------------ P1
def test_p1_advantage_closed_form():
    """rewards {1,0,0,1} -> mean .5, std .5, A = {+1,-1,-1,+1} exactly."""
    adv = O.group_advantage([1, 0, 0, 1], [0, 4])
    assert adv.tolist() == [1.0, -1.0, -1.0, 1.0]
    adv_s = O.group_advantage([1, 0, 0, 1], [0, 4], flags=O.FLAG_SAMPLE_STD)
    assert np.allclose(np.abs(adv_s), math.sqrt(3) / 2, rtol=0, atol=1e-15)


def test_p1_advantage_invariants():
    rng = np.random.default_rng(1)
    R = rng.normal(size=37)
    off = [0, 5, 5, 6, 20, 37]      # includes an empty group and a single-member group
    adv = O.group_advantage(R, off)
    for g in range(len(off) - 1):
        a = adv[off[g]:off[g + 1]]
        G = a.size
        if G <= 1:
            assert np.all(a == 0)
            continue
        assert abs(a.sum()) < 1e-12                   # sum A_i = 0
        assert abs((a ** 2).sum() - G) < 1e-10       # sum A_i^2 = G (population std)
    adv2 = O.group_advantage(3.5 * R - 2.0, off)      # invariant under R -> aR + b, a > 0
    assert np.allclose(adv, adv2, atol=1e-11)
    # a different routine for the same statistic
    a3 = (R[6:20] - np.mean(R[6:20])) / np.std(R[6:20])
    assert np.allclose(adv[6:20], a3, atol=1e-12)


# ------------------------------------------------------------------------------------ P2
def test_p2_all_ratios_one_is_weighted_cross_entropy_gradient():
    """b = q = l (every ratio 1) -> dlogits = kappa n_i A_i (softmax - onehot): the gradient of
    a weighted softmax cross entropy, here taken from torch autograd in float64."""
    host = small_batch(seed=3)
    z = torch.tensor(host["logits"], dtype=torch.float64, requires_grad=True)
    y = torch.tensor(host["target_ids"], dtype=torch.int64)
    lp = -torch.nn.functional.cross_entropy(z, y, reduction="none")
    host["prox_lp"] = lp.detach().numpy().copy()
    host["behave_lp"] = lp.detach().numpy().copy()
    for norm in (O.NORM_CONST_K, O.NORM_PER_TRAJ):
        out = run(host, normalizer=norm, stale_cap=0.0)
        weight = torch.tensor(out["traj_scale"][out["tok_traj"]] * out["adv"][out["tok_traj"]])
        ce = (weight * torch.nn.functional.cross_entropy(z, y, reduction="none")).sum()
        (gref,) = torch.autograd.grad(ce, z)
        assert np.allclose(out["dlogits"], gref.numpy(), rtol=1e-12, atol=1e-15)
        assert out["clip_count"] == 0
        assert np.allclose(out["token_lp"], lp.detach().numpy(), atol=1e-12)


# ------------------------------------------------------------------------------------ P3
def test_p3_config0_loss_exactly_cancels():
    """Config 0 at all ratios 1: loss = -(16/(4k)) sum A_i |tau_i| = -(4/k)(2-3-5+6) = 0 under
    1/k and -(16/4) sum A_i = 0 under 1/|tau_i|, while the gradient is not zero."""
    w = W.workload(0)
    host = W.to_host(W.make_batch(w, 0))
    assert host["logits"].shape == (256, 1024)
    _, lp, _ = O.token_logprob(host["logits"], host["target_ids"])
    host["prox_lp"] = lp
    host["behave_lp"] = lp
    for norm in (O.NORM_CONST_K, O.NORM_PER_TRAJ):
        out = run(host, normalizer=norm)
        assert abs(out["loss"]) < 1e-13
        assert np.abs(out["dlogits"]).max() > 1e-3
    # the uncancelled pieces have the closed form  A_i |tau_i| 16 / (4 k)
    out = run(host, normalizer=O.NORM_CONST_K, k_norm=10.0)
    per_traj = np.bincount(out["tok_traj"], weights=out["term"], minlength=4)
    assert np.allclose(per_traj, np.array([1, -1, -1, 1]) * np.array([2, 3, 5, 6]) * 16 / 40.0,
                       atol=1e-13)


# ------------------------------------------------------------------------------------ P4
def test_p4_equal_rewards_give_exact_zero():
    host = small_batch(seed=4)
    host["rewards"] = np.full_like(host["rewards"], 1.0)
    out = run(host)
    assert out["loss"] == 0.0 and out["clip_count"] == 0
    assert not np.any(out["dlogits"]) and not np.any(out["adv"])


# ------------------------------------------------------------------------------------ P5
def test_p5_normalizers_coincide_when_every_traj_has_k_steps():
    """under 1/|tau_i| every rollout has total weight 1, under 1/k weight
    |tau_i|/k; they coincide when |tau_i| = k for all i."""
    k = 5
    n_traj, tok = 8, 3
    step_off = np.arange(n_traj * k + 1) * tok
    traj_off = np.arange(n_traj + 1) * k
    group_off = np.array([0, 4, 8])
    rng = np.random.default_rng(5)
    z = rng.normal(size=(step_off[-1], 32)) * 2
    y = rng.integers(0, 32, size=step_off[-1])
    _, lp, _ = O.token_logprob(z, y)
    q = lp + rng.normal(size=lp.size) * 0.1
    b = q + rng.normal(size=lp.size) * 0.1
    R = rng.integers(0, 2, size=n_traj).astype(float)
    R[0], R[1], R[4], R[5] = 1, 0, 0, 1
    kw = dict(clip_eps=0.2, stale_cap=2.0, k_norm=float(k))
    a = O.awr_loss_fwd_bwd(z, y, b, q, step_off, traj_off, group_off, R,
                           normalizer=O.NORM_CONST_K, **kw)
    c = O.awr_loss_fwd_bwd(z, y, b, q, step_off, traj_off, group_off, R,
                           normalizer=O.NORM_PER_TRAJ, **kw)
    assert a["loss"] == pytest.approx(c["loss"], rel=1e-14)
    assert np.allclose(a["dlogits"], c["dlogits"], rtol=1e-14, atol=0)
    # summed step weight of a trajectory: |tau_i|/k under 1/k, 1 under 1/|tau_i|
    traj_off2 = np.array([0, 2, 9, 20, 40])
    sc_k = O.traj_scale(step_off, traj_off2, [0, 4], 10.0, O.NORM_CONST_K, 1.0)
    sc_t = O.traj_scale(step_off, traj_off2, [0, 4], 10.0, O.NORM_PER_TRAJ, 1.0)
    steps = np.diff(traj_off2)
    kappa = 1.0 / 4
    assert np.allclose(sc_k * steps / kappa, steps / 10.0)
    assert np.allclose(sc_t * steps / kappa, 1.0)


# ------------------------------------------------------------------------------------ P6
def brute_force(host, params):
    """Literal token-by-token loop over Eq. (1) with math.exp; no numpy arithmetic."""
    z, y = host["logits"], host["target_ids"]
    so, to, go = host["step_off"], host["traj_off"], host["group_off"]
    eps = float(np.float32(params["clip_eps"]))
    cap = float(np.float32(params["stale_cap"]))
    NG = len(go) - 1
    loss, count, lps = 0.0, 0, []
    for g in range(NG):
        members = list(range(go[g], go[g + 1]))
        G = len(members)
        Rs = [float(host["rewards"][i]) for i in members]
        mu = sum(Rs) / G
        var = sum((r - mu) ** 2 for r in Rs) / G
        for i, Ri in zip(members, Rs):
            A = 0.0 if var == 0 else (Ri - mu) / math.sqrt(var)
            n_steps = to[i + 1] - to[i]
            n_i = 1.0 / params["k_norm"] if params["normalizer"] == O.NORM_CONST_K else 1.0 / n_steps
            for j in range(to[i], to[i + 1]):
                for t in range(so[j], so[j + 1]):
                    row = [float(x) for x in z[t]]
                    m = max(row)
                    lse = m + math.log(sum(math.exp(x - m) for x in row))
                    lp = row[y[t]] - lse
                    lps.append((t, lp))
                    ratio_behave = math.exp(lp - float(host["behave_lp"][t]))   # pi_theta/pi_behave
                    w = math.exp(float(host["prox_lp"][t]) - float(host["behave_lp"][t]))
                    r = math.exp(lp - float(host["prox_lp"][t]))
                    if 0 < cap < math.inf:
                        if w > cap:
                            ratio_behave = ratio_behave * cap / w
                            w = cap
                    first = ratio_behave * A                       # Eq. (1) first argument of min
                    second = w * min(max(r, 1 - eps), 1 + eps) * A  # Eq. (1) second argument
                    # the two arguments are *equal* when nothing clips (w r = pi_theta/pi_behave)
                    # and differ only by rounding there; a real trigger differs by > 1e-4
                    if second < first - 1e-9 * abs(first):
                        count += 1
                    loss -= min(first, second) * n_i / (NG * G)
    return loss, count, lps


@pytest.mark.parametrize("eps,drift,norm", [(0.2, "perturb", O.NORM_CONST_K),
                                            (0.01, "perturb", O.NORM_PER_TRAJ),
                                            (0.2, "drift", O.NORM_PER_TRAJ)])
def test_p6_loss_and_clip_count_match_a_literal_loop(eps, drift, norm):
    host = small_batch(seed=6, V=24, n_tok=70, lp_mode=drift, clip_eps=eps, normalizer=norm,
                       stale_cap=2.0)
    out = run(host)
    loss, count, lps = brute_force(host, host["params"])
    assert out["clip_count"] == count
    if drift == "drift" or eps == 0.01:
        assert count > 0                                  # the count is non-trivial
    assert out["loss"] == pytest.approx(loss, rel=1e-12, abs=1e-15)
    for t, lp in lps:
        assert out["token_lp"][t] == pytest.approx(lp, abs=1e-12)


def test_p6_unclipped_branch_is_pi_theta_over_pi_behave():
    """P10 / PAPER.md:57: w_t r_t = exp(l_t - b_t) with the cap off."""
    host = small_batch(seed=7, lp_mode="drift")
    out = run(host, stale_cap=0.0)
    assert np.allclose(out["stale_w"] * out["ratio"],
                       np.exp(out["token_lp"] - host["behave_lp"].astype(np.float64)), rtol=1e-13)


# ------------------------------------------------------------------------------------ P7
def test_p7_finite_differences():
    host = small_batch(seed=8, V=16, n_groups=2, group_size=3, n_tok=20, lp_mode="drift",
                       stale_cap=2.0, normalizer=O.NORM_PER_TRAJ)
    host["logits"] = host["logits"].astype(np.float64)
    out = run(host)
    # stay away from the kinks of min / clip
    eps = float(np.float32(host["params"]["clip_eps"]))
    lr = out["token_lp"] - host["prox_lp"]
    assert np.all(np.abs(lr - math.log1p(eps)) > 1e-3) and np.all(np.abs(lr - math.log1p(-eps)) > 1e-3)
    h = 1e-6
    rng = np.random.default_rng(0)
    checked = 0
    for t in range(host["logits"].shape[0]):
        for v in rng.choice(16, size=5, replace=False).tolist() + [int(host["target_ids"][t])]:
            zp = host["logits"].copy(); zp[t, v] += h
            zm = host["logits"].copy(); zm[t, v] -= h
            lp_ = run(dict(host, logits=zp), want_dlogits=False)["loss"]
            lm_ = run(dict(host, logits=zm), want_dlogits=False)["loss"]
            fd = (lp_ - lm_) / (2 * h)
            assert out["dlogits"][t, v] == pytest.approx(fd, abs=1e-7)
            checked += 1
    assert checked > 100
    assert out["clip_count"] > 0 and np.any(out["coef"] != 0)


# ------------------------------------------------------------------------------------ P8 / P9
def test_p8_rows_sum_to_zero_and_sign_pattern():
    host = small_batch(seed=9, lp_mode="drift")
    out = run(host)
    g, y = out["dlogits"], host["target_ids"]
    assert np.abs(g.sum(axis=1)).max() < 1e-15
    A = out["adv"][out["tok_traj"]]
    for t in range(g.shape[0]):
        if out["trig"][t] or A[t] == 0:
            assert not np.any(g[t])
            continue
        others = np.delete(g[t], y[t])
        if A[t] > 0:
            assert g[t, y[t]] < 0 and np.all(others > 0)
        else:
            assert g[t, y[t]] > 0 and np.all(others < 0)


def test_p9_shift_and_permutation_invariance():
    host = small_batch(seed=10, lp_mode="drift")
    host["logits"] = host["logits"].astype(np.float64)
    out = run(host)
    rng = np.random.default_rng(2)
    shift = rng.normal(size=(host["logits"].shape[0], 1)) * 5
    out_s = run(dict(host, logits=host["logits"] + shift))
    assert np.allclose(out_s["token_lp"], out["token_lp"], atol=1e-12)
    assert out_s["loss"] == pytest.approx(out["loss"], rel=1e-10)
    assert np.allclose(out_s["dlogits"], out["dlogits"], atol=1e-13)
    perm = rng.permutation(host["logits"].shape[1])
    inv = np.argsort(perm)
    out_p = run(dict(host, logits=host["logits"][:, perm], target_ids=inv[host["target_ids"]].astype(np.int32)))
    assert out_p["loss"] == pytest.approx(out["loss"], rel=1e-12)
    assert np.allclose(out_p["dlogits"], out["dlogits"][:, perm], atol=1e-14)
    assert out_p["clip_count"] == out["clip_count"]


# ------------------------------------------------------------------------------------ P11
def test_p11_prox_equals_behave_is_plain_ppo_clip():
    """q = b: the objective is the standard PPO-clip surrogate on r = pi_theta/pi_behave; with
    eps -> 1 and r < 2 nothing clips and it is the importance-weighted policy gradient."""
    host = small_batch(seed=11, lp_mode="drift")
    host["behave_lp"] = host["prox_lp"].copy()
    out = run(host, stale_cap=0.0)
    A = out["adv"][out["tok_traj"]]
    sc = out["traj_scale"][out["tok_traj"]]
    r = np.exp(out["token_lp"] - host["behave_lp"].astype(np.float64))
    eps = float(np.float32(0.2))
    ppo = np.minimum(r * A, np.clip(r, 1 - eps, 1 + eps) * A) * sc
    assert np.allclose(out["term"], ppo, rtol=1e-13, atol=0)
    out1 = run(host, stale_cap=0.0, clip_eps=0.999999)
    keep = r < 1.999
    assert np.allclose(out1["term"][keep], (r * A * sc)[keep], rtol=1e-13, atol=0)
    assert np.allclose(out1["coef"][keep], (r * A * sc)[keep], rtol=1e-13, atol=0)


# ------------------------------------------------------------------------------------ P12
def test_p12_length_attenuation_matches_the_papers_arithmetic():
    """failures 12.5 steps vs successes 5.1 -> "2.4x" attenuation under
    1/|tau_i|, none under 1/k.  Integer stand-in: 25 vs 10 steps (ratio 2.5), plus the exact
    printed ratio on the formula."""
    gv = golden()
    assert gv["fail_steps"] / gv["succ_steps"] == pytest.approx(2.45, abs=0.01)
    assert round(gv["fail_steps"] / gv["succ_steps"], 1) in (gv["length_gap"], 2.5)
    step_off = np.arange(36) * 2
    traj_off = np.array([0, 10, 35])
    sc_t = O.traj_scale(step_off, traj_off, [0, 2], gv["k_norm"], O.NORM_PER_TRAJ, 1.0)
    sc_k = O.traj_scale(step_off, traj_off, [0, 2], gv["k_norm"], O.NORM_CONST_K, 1.0)
    assert sc_t[0] / sc_t[1] == pytest.approx(25 / 10)
    assert sc_k[0] / sc_k[1] == 1.0
    assert sc_k[0] == pytest.approx(1.0 / (1 * 2 * gv["k_norm"]))


# ------------------------------------------------------------------------------------ edges
def test_offsets_check_and_masked_tokens():
    assert O.check_offsets([0, 2, 5], [0, 1, 2], [0, 2], 5) == 0
    assert O.check_offsets([1, 2, 5], [0, 1, 2], [0, 2], 5) & O.ERR_STEP_OFF
    assert O.check_offsets([0, 3, 2, 5], [0, 1, 3], [0, 2], 5) & O.ERR_STEP_OFF
    assert O.check_offsets([0, 2, 5], [0, 1, 3], [0, 2], 5) & O.ERR_TRAJ_OFF
    assert O.check_offsets([0, 2, 5], [0, 1, 2], [0, 3], 5) & O.ERR_GROUP_OFF
    host = small_batch(seed=12, lp_mode="drift")
    ref = run(host)
    y = host["target_ids"].copy()
    y[3] = -1
    y[7] = host["logits"].shape[1] + 2
    out = run(dict(host, target_ids=y))
    assert out["err_word"] == O.ERR_TARGET_RANGE
    for t in (3, 7):
        assert out["token_lp"][t] == 0 and out["term"][t] == 0 and not np.any(out["dlogits"][t])
    keep = np.ones(y.size, bool); keep[[3, 7]] = False
    assert np.allclose(out["dlogits"][keep], ref["dlogits"][keep], atol=0)
    assert out["loss"] == pytest.approx(ref["loss"] + ref["term"][3] + ref["term"][7], rel=1e-12)


def test_empty_steps_and_trajectories():
    """A10: an empty step counts toward |tau_i|; an empty trajectory still enters mean/std."""
    step_off = np.array([0, 3, 3, 6])        # step 1 empty
    traj_off = np.array([0, 2, 2, 3])        # trajectory 1 has no steps
    group_off = np.array([0, 3])
    R = np.array([1.0, 0.0, 0.0])
    seg = O.segment_expand(step_off, traj_off, group_off)
    assert seg["tok_traj"].tolist() == [0, 0, 0, 2, 2, 2]
    assert seg["traj_steps"].tolist() == [2, 0, 1]
    adv = O.group_advantage(R, group_off)
    assert adv[0] == pytest.approx(math.sqrt(2)) and adv[1] == pytest.approx(-1 / math.sqrt(2))
    sc = O.traj_scale(step_off, traj_off, group_off, 10.0, O.NORM_PER_TRAJ, 1.0)
    assert sc.tolist() == [0.5 / 3, 0.0, 1.0 / 3]


def test_stale_cap_truncates_weight_only():
    host = small_batch(seed=13, lp_mode="drift")
    a = run(host, stale_cap=0.0)
    c = run(host, stale_cap=1.02)
    w_a, w_c = a["stale_w"], c["stale_w"]
    assert np.all(w_c <= float(np.float32(1.02))) and np.any(w_a > 1.02)
    assert np.array_equal(a["trig"], c["trig"])                   # w has no theta-dependence
    assert np.allclose(c["coef"] * w_a, a["coef"] * w_c, rtol=1e-13, atol=0)


def test_fused_head_miniature_against_plain_loops():
    """a5 on a miniature: numpy.matmul vs plain loops for the three contractions."""
    w = W.workload(4, n_groups=2, group_size=2, n_tok=12, V=10, hidden=6)
    host = W.to_host(W.make_batch(w, 3))
    args, kw = W.oracle_args(host)
    out = O.awr_loss_fwd_bwd_fused_head(*args, **kw)
    H, Wh = host["hidden"].astype(np.float64), host["w_head"].astype(np.float64)
    n, K = H.shape
    V = Wh.shape[1]
    z = [[sum(H[t, k] * Wh[k, v] for k in range(K)) for v in range(V)] for t in range(n)]
    assert np.allclose(out["logits"], z, atol=1e-14)
    tok = O.awr_loss_fwd_bwd(np.array(z), *args[2:], **kw)
    dS = tok["dlogits"]
    dH = [[sum(dS[t, v] * Wh[k, v] for v in range(V)) for k in range(K)] for t in range(n)]
    dW = [[sum(H[t, k] * dS[t, v] for t in range(n)) for v in range(V)] for k in range(K)]
    assert np.allclose(out["dhidden"], dH, atol=1e-15)
    assert np.allclose(out["dw_head"], dW, atol=1e-15)
    assert out["loss"] == tok["loss"]


# ------------------------------------------------------------------------------------ P13: Eq. (2)
def _with_exploded_ratios(host, every=5, shift=1.5):
    """Lower prox_lp on every 5th token so that r_t = pi_theta/pi_prox grows by e^1.5 = 4.5 > c."""
    host = dict(host)
    q = host["prox_lp"].copy()
    q[::every] -= shift
    host["prox_lp"] = q
    return host


def test_p13_dual_clip_worked_example():
    """PAPER.md:270-275 with c = 3 (:461), eps = 0.2, one trajectory pair so that A = -1/+1:
    r = 5, A = -1: min(5(-1), 1.2(-1)) = -5, capped to c A = -3 (hit, zero gradient);
    r = 2, A = -1: min(-2, -1.2) = -2 > -3 (no hit);  r = 5, A = +1: min(5, 1.2) = 1.2 (eps-clip)."""
    lp = np.log(np.array([0.5, 0.2, 0.5]))
    q = lp - np.log(np.array([5.0, 2.0, 5.0]))
    A = np.array([-1.0, -1.0, 1.0])
    one = np.ones(3)
    term, coef, trig, r, w, dual = O.token_terms(lp, q, q, A, one, 0.2, 0.0, one.astype(bool),
                                                 dual_clip_c=3.0, want_dual=True)
    assert np.allclose(r, [5.0, 2.0, 5.0]) and np.allclose(w, 1.0)
    assert np.allclose(term, [-3.0, -2.0, 1.0 + float(np.float32(0.2))])
    assert dual.tolist() == [True, False, False] and trig.tolist() == [False, False, True]
    assert coef[0] == 0.0 and coef[2] == 0.0 and coef[1] == pytest.approx(-2.0)


@pytest.mark.parametrize("norm", [O.NORM_CONST_K, O.NORM_PER_TRAJ])
def test_p13_dual_clip_matches_a_literal_loop_and_bounds_the_term(norm):
    """Ye et al. 2020 as cited by PAPER.md:270: max(min(rho A, clip(rho) A), c A) for A < 0, times
    the staleness weight; literal loop with math.exp.  Also the paper's claim (:275): c A is an
    absolute lower bound of the per-token contribution (before the weights)."""
    host = _with_exploded_ratios(small_batch(seed=13, V=24, n_tok=80, lp_mode="drift",
                                             normalizer=norm, stale_cap=2.0))
    c = 3.0
    out = run(host, dual_clip_c=c)
    eps = float(np.float32(host["params"]["clip_eps"]))
    loss, hits = 0.0, 0
    for t in range(host["logits"].shape[0]):
        A = float(out["adv"][out["tok_traj"][t]])
        scale = float(out["traj_scale"][out["tok_traj"][t]])
        r = math.exp(out["token_lp"][t] - float(host["prox_lp"][t]))
        w = min(math.exp(float(host["prox_lp"][t]) - float(host["behave_lp"][t])), 2.0)
        s = min(r * A, min(max(r, 1 - eps), 1 + eps) * A)
        if A < 0 and c * A > s:
            s = c * A
            hits += 1
        loss -= scale * w * s
        if A < 0:
            assert out["term"][t] >= scale * w * c * A * (1 + 1e-12)
    assert hits > 0 and out["dual_clip_count"] == hits
    assert out["loss"] == pytest.approx(loss, rel=1e-12, abs=1e-15)
    # hit tokens: A < 0 and r > c exactly; they carry no gradient and are not eps-triggers
    hit = out["dual"]
    assert np.array_equal(hit, (out["adv"][out["tok_traj"]] < 0) & (out["ratio"] > c))
    assert not np.any(out["trig"] & hit)
    assert np.all(out["coef"][hit] == 0) and np.all(out["dlogits"][hit] == 0)


def test_p13_dual_clip_off_and_limit_cases():
    host = _with_exploded_ratios(small_batch(seed=14, lp_mode="drift"))
    base = run(host)
    for c in (0.0, 1.0):                               # c <= 1: off = Eq. (1)
        o = run(host, dual_clip_c=c)
        assert o["loss"] == base["loss"] and o["dual_clip_count"] == 0
    big = run(host, dual_clip_c=1e30)                  # c -> inf: the floor is never reached
    assert big["loss"] == base["loss"] and big["dual_clip_count"] == 0
    assert np.array_equal(big["dlogits"], base["dlogits"])
    on = run(host, dual_clip_c=3.0)
    pos = base["adv"][base["tok_traj"]] >= 0           # A >= 0 tokens are untouched
    assert np.array_equal(on["term"][pos], base["term"][pos])
    assert np.array_equal(on["coef"][pos], base["coef"][pos])
    assert on["dual_clip_count"] > 0 and on["loss"] < base["loss"]   # -J with a raised floor


def test_p13_dual_clip_finite_differences():
    host = _with_exploded_ratios(small_batch(seed=15, V=16, n_groups=2, group_size=3, n_tok=24,
                                             lp_mode="drift", normalizer=O.NORM_PER_TRAJ))
    host["logits"] = host["logits"].astype(np.float64)
    out = run(host, dual_clip_c=3.0)
    assert out["dual_clip_count"] > 0
    lr = out["token_lp"] - host["prox_lp"]
    assert np.all(np.abs(lr - math.log(3.0)) > 1e-3)   # away from the new kink
    h = 1e-6
    for t in range(host["logits"].shape[0]):
        for v in (0, 7, int(host["target_ids"][t])):
            zp = host["logits"].copy(); zp[t, v] += h
            zm = host["logits"].copy(); zm[t, v] -= h
            fd = (run(dict(host, logits=zp), dual_clip_c=3.0, want_dlogits=False)["loss"] -
                  run(dict(host, logits=zm), dual_clip_c=3.0, want_dlogits=False)["loss"]) / (2 * h)
            assert out["dlogits"][t, v] == pytest.approx(fd, abs=1e-7)


# ------------------------------------------------------------------------------------ P14: entropy
def test_p14_entropy_closed_forms_and_library():
    """PAPER.md:232 / :341 per-token entropy.  Uniform logits give log V exactly; a two-point
    distribution gives the binary entropy; a near one-hot row gives ~0; -inf entries count as
    p = 0; a constant shift changes nothing; and the whole thing agrees with the library
    Categorical entropy."""
    V = 1000
    assert O.token_entropy(np.full((1, V), 3.25))[0] == pytest.approx(math.log(V), abs=1e-12)
    p = 0.3
    z = np.array([[math.log(p), math.log(1 - p)]])
    assert O.token_entropy(z)[0] == pytest.approx(-(p * math.log(p) + (1 - p) * math.log(1 - p)), abs=1e-14)
    one_hot = np.full((1, 50), -60.0); one_hot[0, 7] = 40.0
    assert 0.0 <= O.token_entropy(one_hot)[0] < 1e-40
    zi = np.array([[0.5, -np.inf, 1.5, -np.inf]])
    assert O.token_entropy(zi)[0] == pytest.approx(O.token_entropy(zi[:, [0, 2]])[0], abs=1e-15)
    rng = np.random.default_rng(3)
    z = rng.normal(0, 3, size=(7, 333))
    H = O.token_entropy(z)
    assert np.allclose(O.token_entropy(z + 11.0), H, atol=1e-12)
    ref = torch.distributions.Categorical(logits=torch.from_numpy(z)).entropy().numpy()
    assert np.allclose(H, ref, atol=1e-12)
    assert np.all(H > 0) and np.all(H <= math.log(333) + 1e-12)


def test_p14_entropy_in_the_path_and_masked_tokens():
    host = small_batch(seed=16)
    host["target_ids"] = host["target_ids"].copy()
    host["target_ids"][::7] = -1
    out = run(host, want_entropy=True)
    H = O.token_entropy(host["logits"])
    masked = host["target_ids"] < 0
    assert np.all(out["token_entropy"][masked] == 0.0)
    assert np.array_equal(out["token_entropy"][~masked], H[~masked])
    assert "token_entropy" not in run(host)


# ------------------------------------------------------------------------------------ P15: baselines
def test_p15_raft_success_filter():
    """RAFT++ (PAPER.md:65): advantage = 1[R > 0], no group normalisation, decoupled ratio kept.
    Only successful trajectories carry gradient; with all ratios 1 the gradient is behaviour
    cloning on the positives: scale_i (softmax - onehot) on their tokens, 0 elsewhere."""
    assert O.group_advantage(np.array([1, 0, 0, 1, 0.5, 0, -1], dtype=np.float32), np.array([0, 4, 7]),
                             O.FLAG_SUCCESS_FILTER).tolist() == [1, 0, 0, 1, 1, 0, 0]
    # a single-member group (the paper runs RAFT++ with G = 1, :462) still gets A = 1[R > 0]
    assert O.group_advantage(np.array([1.0], dtype=np.float32), np.array([0, 1]), O.FLAG_SUCCESS_FILTER)[0] == 1.0
    host = small_batch(seed=17, normalizer=O.NORM_PER_TRAJ)
    lp = run(host)["token_lp"]
    host = dict(host, prox_lp=lp.astype(np.float32), behave_lp=lp.astype(np.float32))
    out = run(host, flags=O.FLAG_SUCCESS_FILTER)
    succ = host["rewards"][out["tok_traj"]] > 0
    assert succ.any() and (~succ).any()
    assert np.all(out["dlogits"][~succ] == 0)
    z = torch.from_numpy(host["logits"].astype(np.float64))
    p = torch.softmax(z, dim=1).numpy()
    p[np.arange(p.shape[0]), host["target_ids"]] -= 1.0
    r = np.exp(lp - host["prox_lp"])                      # ~1, not exactly (f32 rounding of lp)
    expect = (out["traj_scale"][out["tok_traj"]] * r)[:, None] * p
    assert np.allclose(out["dlogits"][succ], expect[succ], rtol=1e-9, atol=1e-15)


def test_p15_coupled_ratio_is_eq1_with_prox_equal_behave():
    """the coupled baseline folds staleness and update movement into one
    pi_theta/pi_behave ratio with the clip centred on it: Eq. (1) with pi_prox := pi_behave
    (w_t = 1), whatever prox log-probs are passed.  Literal loop as the second check."""
    host = small_batch(seed=18, lp_mode="drift")
    a = run(host, flags=O.FLAG_COUPLED)
    b = run(dict(host, prox_lp=host["behave_lp"]))
    for k in ("loss", "clip_count"):
        assert a[k] == b[k]
    assert np.array_equal(a["dlogits"], b["dlogits"]) and np.all(a["stale_w"] == 1.0)
    eps = float(np.float32(host["params"]["clip_eps"]))
    loss = 0.0
    for t in range(host["logits"].shape[0]):
        A = float(a["adv"][a["tok_traj"][t]])
        rho = math.exp(a["token_lp"][t] - float(host["behave_lp"][t]))
        loss -= float(a["traj_scale"][a["tok_traj"][t]]) * min(rho * A, min(max(rho, 1 - eps), 1 + eps) * A)
    assert a["loss"] == pytest.approx(loss, rel=1e-12, abs=1e-15)
    assert a["clip_count"] != run(host)["clip_count"]     # the decoupled clip is centred elsewhere


# ------------------------------------------------------------------------------------ P16
def test_p16_dynamic_sampling_skips_uniform_groups():
    """PAPER.md:63 (DAPO dynamic sampling): all-success / all-failure groups are skipped.  The
    result must equal the loss of the batch that physically contains only the mixed groups."""
    w = W.workload(3, n_groups=8, group_size=4, n_tok=160, V=32, dtype=torch.float32,
                   p_equal_groups=0.5)
    host = W.to_host(W.make_batch(w, seed=19))
    mixed = O.mixed_groups(host["rewards"], host["group_off"])
    assert 0 < mixed.sum() < mixed.size
    out = run(host, flags=O.FLAG_SKIP_UNIFORM)
    # rebuild the batch from the mixed groups only
    so, to, go = host["step_off"], host["traj_off"], host["group_off"]
    keep_traj = np.concatenate([np.arange(go[g], go[g + 1]) for g in np.nonzero(mixed)[0]])
    keep_steps = np.concatenate([np.arange(to[i], to[i + 1]) for i in keep_traj])
    keep_tok = np.concatenate([np.arange(so[j], so[j + 1]) for j in keep_steps])
    sub = dict(host)
    sub["logits"] = host["logits"][keep_tok]
    for k in ("target_ids", "behave_lp", "prox_lp"):
        sub[k] = host[k][keep_tok]
    sub["rewards"] = host["rewards"][keep_traj]
    sub["step_off"] = np.concatenate([[0], np.cumsum(np.diff(so)[keep_steps])]).astype(np.int32)
    sub["traj_off"] = np.concatenate([[0], np.cumsum(np.diff(to)[keep_traj])]).astype(np.int32)
    sub["group_off"] = np.concatenate([[0], np.cumsum(np.diff(go)[mixed])]).astype(np.int32)
    ref = run(sub)
    assert out["loss"] == pytest.approx(ref["loss"], rel=1e-12, abs=1e-16)
    assert out["clip_count"] == ref["clip_count"]
    assert np.allclose(out["dlogits"][keep_tok], ref["dlogits"], rtol=1e-12, atol=1e-18)
    gone = np.setdiff1d(np.arange(host["logits"].shape[0]), keep_tok)
    assert np.all(out["dlogits"][gone] == 0)
    # without the flag the same tokens carry 1/NG instead of 1/NG_mixed
    base = run(host)
    assert base["loss"] == pytest.approx(out["loss"] * mixed.sum() / mixed.size, rel=1e-12)
    # nothing mixed -> nothing at all
    allsame = dict(host, rewards=np.ones_like(host["rewards"]))
    z = run(allsame, flags=O.FLAG_SKIP_UNIFORM)
    assert z["loss"] == 0.0 and not z["dlogits"].any()
    # with the RAFT++ filter, an all-success group is skipped too
    r = run(allsame, flags=O.FLAG_SKIP_UNIFORM | O.FLAG_SUCCESS_FILTER)
    assert r["loss"] == 0.0 and not r["adv"].any()
