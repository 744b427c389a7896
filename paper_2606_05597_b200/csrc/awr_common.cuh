// Shared device helpers for the AsyncWebRL token-loss kernels (sm_100a only).
// Notation follows include/awr.h: z logits row, y target id, lse log-sum-exp, l_t token
// log-prob, q/b prox/behave log-probs, A advantage, c_t gradient coefficient.
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/awr.h"

namespace awr {

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr unsigned kFull = 0xffffffffu;

// per-token flag byte written by the row kernels, read by the final reduction
constexpr uint8_t kFlagTrig = 1;
constexpr uint8_t kFlagDual = 2;   // Eq. (2) dual-clip hit

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ float lg2_approx(float x) {
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// exp / log on the special-function unit (2 ulp ex2 / lg2 + one rounding of the scaled argument):
// a3 runs redundantly in every thread between the passes of a row, so its latency is on the
// critical path of every row; libm's expf / logf / log1pf cost ~1.2 k clocks there (measured).
__device__ __forceinline__ float fast_exp(float x) { return ex2_approx(x * kLog2e); }
__device__ __forceinline__ float fast_log(float x) { return lg2_approx(x) * kLn2; }
// log(1 + e) for e in [0, 1]: the series below 2^-12 (where 1 + e would round e away)
__device__ __forceinline__ float fast_log1p01(float e) {
    return e < 2.44140625e-4f ? e * (1.0f - 0.5f * e) : fast_log(1.0f + e);
}

// (max, sum of exp(x - max)) pairs: the online log-sum-exp state.  m = -inf, s = 0 is the
// identity.  Combination is written so that the identity never produces NaN.
struct MaxSum {
    float m, s;
};

__device__ __forceinline__ MaxSum combine(MaxSum a, MaxSum b) {
    float M = fmaxf(a.m, b.m);
    if (M == -INFINITY) return MaxSum{M, 0.f};
    float sa = a.s * ex2_approx((a.m - M) * kLog2e);
    float sb = b.s * ex2_approx((b.m - M) * kLog2e);
    return MaxSum{M, sa + sb};
}

__device__ __forceinline__ MaxSum warp_combine(MaxSum v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        MaxSum other{__shfl_xor_sync(kFull, v.m, o), __shfl_xor_sync(kFull, v.s, o)};
        v = combine(v, other);
    }
    return v;
}

// Entropy of the row from the state of its non-target entries: sz_rest = sum_{v != y} e^{z_v - m}
// max(z_v, -FLT_MAX) relative to the same m as lse_rest's sum (entries at -inf contribute 0).
//   H = lse - sum_v p_v z_v = lse - (sz_rest e^{m - lse} + p_y z_y)
__device__ __forceinline__ float row_entropy(float lse, float m_rest, float sz_rest, float lp,
                                             float zy) {
    const float rest = (m_rest == -INFINITY) ? 0.f : sz_rest * ex2_approx((m_rest - lse) * kLog2e);
    const float py = ex2_approx(lp * kLog2e);
    return lse - (rest + (py > 0.f ? py * zy : 0.f));
}
constexpr float kZFloor = -3.0e38f;     // stands in for -inf in e * z (e is 0 there)

// Everything the path needs to know about a row besides the row itself.
struct RowHeader {
    int y;        // target id (already range-checked: valid <=> 0 <= y < V)
    float zy;     // z[y] widened to f32 (0 if invalid)
    float q, b;   // prox / behave log-probs
    float A;      // advantage of the token's trajectory
    float scale;  // loss_scale * kappa_g * n_i
};

struct TokenScalars {
    float lp;    // l_t
    float lse;   // log-sum-exp of the whole row (= zy - l_t for a valid token)
    float term;  // contribution to J
    float coef;  // c_t
    float gy;    // c_t (p_y - 1): the target entry of the gradient row
    bool trig;
    bool dual;   // Eq. (2): A < 0 and the floor c A is the active term
};

// a3: ratio, clip, normalizer (Eq. 1), fp32.
//
// dual_c > 1 adds Eq. (2) (reading A7): for A < 0 the inner min is
// capped from below by dual_c * A; a hit (floor strictly larger) has zero gradient.
//
// lse_rest is the log-sum-exp of the row WITHOUT its target entry (of the whole row when the
// token is not valid).  With d = lse_rest - z_y:  l_t = -softplus(d),  1 - p_y = sigmoid(d).
// Both stay accurate to f32 rounding when p_y -> 1, where z_y - lse and exp(l_t) - 1 cancel
// (DESIGN.md "Numerics").
__device__ __forceinline__ TokenScalars token_scalars(const RowHeader& h, float lse_rest,
                                                      bool valid, float clip_eps,
                                                      float stale_cap, float dual_c) {
    TokenScalars t;
    t.dual = false;
    if (!valid) {
        t.lp = 0.f; t.lse = lse_rest; t.term = 0.f; t.coef = 0.f; t.gy = 0.f; t.trig = false;
        return t;
    }
    const float d = lse_rest - h.zy;                  // -inf if the row has no other entry
    const float e = fast_exp(-fabsf(d));              // in [0, 1]
    const float sp = fmaxf(d, 0.f) + fast_log1p01(e); // softplus(d) = -l_t
    const float one_minus_p = (d >= 0.f ? 1.0f : e) / (1.0f + e);   // sigmoid(d) = 1 - p_y
    t.lp = -sp;
    t.lse = h.zy + sp;
    float r = fast_exp(t.lp - h.q);                   // pi_theta / pi_prox
    float w = fast_exp(h.q - h.b);                    // pi_prox / pi_behave (staleness weight)
    if (stale_cap > 0.f && stale_cap < INFINITY) w = fminf(w, stale_cap);
    float u = r * h.A;
    float v = fminf(fmaxf(r, 1.0f - clip_eps), 1.0f + clip_eps) * h.A;
    t.trig = v < u;
    float sw = h.scale * w;
    float s = fminf(u, v);
    if (dual_c > 1.0f && h.A < 0.f) {
        const float floor_ = dual_c * h.A;
        t.dual = floor_ > s;
        s = fmaxf(s, floor_);
    }
    t.term = sw * s;
    t.coef = (t.trig || t.dual) ? 0.f : sw * u;
    t.gy = -t.coef * one_minus_p;
    return t;
}

__device__ __forceinline__ float bf16_lo(uint32_t p) { return __uint_as_float(p << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t p) { return __uint_as_float(p & 0xffff0000u); }

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}

// the same, an overflowing or infinite input giving the largest finite bf16
__device__ __forceinline__ uint32_t pack_bf16x2_sat(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.satfinite.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}

__device__ __forceinline__ uint32_t max_bf16x2(uint32_t a, uint32_t b) {
    uint32_t r;
    asm("max.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
    return r;
}

// Arguments shared by both row kernels.
struct RowArgs {
    const void* logits;
    void* dlogits;  // nullptr = forward only
    int64_t n_tok, V, ld;
    const int32_t* target_ids;
    const float* behave_lp;
    const float* prox_lp;
    const int32_t* tok_traj;
    const float* adv;
    const float* traj_scale;
    float* token_lp;
    float* tok_term;
    float* tok_coef;      // nullable
    float* target_logit;  // nullable
    float* token_entropy; // nullable: H_t = lse - sum_v p_v z_v (0 for masked tokens)
    uint8_t* tok_flag;
    uint32_t* err_word;
    float clip_eps, stale_cap;
    float dual_c;         // Eq. (2) constant; <= 1 = off
};

// Loads the row header for token t (one thread).  Sets the error bit for y >= V.
__device__ __forceinline__ RowHeader load_row_header(const RowArgs& a, int64_t t, bool& valid,
                                                     bool is_bf16) {
    RowHeader h;
    int y = a.target_ids[t];
    valid = (y >= 0) && (y < a.V);
    if (y >= a.V) atomicOr(a.err_word, AWR_ERRBIT_TARGET_RANGE);
    int traj = a.tok_traj[t];
    h.y = y;
    h.q = a.prox_lp[t];
    h.b = a.behave_lp[t];
    h.A = traj >= 0 ? a.adv[traj] : 0.f;
    h.scale = traj >= 0 ? a.traj_scale[traj] : 0.f;
    h.zy = 0.f;
    if (valid) {
        if (is_bf16) {
            h.zy = __bfloat162float(
                reinterpret_cast<const __nv_bfloat16*>(a.logits)[t * a.ld + y]);
        } else {
            h.zy = reinterpret_cast<const float*>(a.logits)[t * a.ld + y];
        }
    }
    return h;
}

// One thread: per-token outputs of a3.
__device__ __forceinline__ void store_token_outputs(const RowArgs& a, int64_t t,
                                                    const RowHeader& h, const TokenScalars& ts,
                                                    bool valid) {
    a.token_lp[t] = ts.lp;
    a.tok_term[t] = ts.term;
    a.tok_flag[t] = (ts.trig ? kFlagTrig : 0) | (ts.dual ? kFlagDual : 0);
    if (a.tok_coef) a.tok_coef[t] = ts.coef;
    if (a.target_logit) a.target_logit[t] = valid ? h.zy : 0.f;
}

}  // namespace awr
