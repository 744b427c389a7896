// a0 segment expansion, a1 group advantage (kernel 1) and the final fixed-order reduction of a3.
// PAPER.md:61 (hierarchy, advantage), :57-:59 (outer factors).  All three are tiny kernels:
// the arrays they touch are a few hundred KB at most.
#include "awr_common.cuh"
#include "awr_kernels.h"

namespace awr {

// largest i in [0, n) with off[i] <= x, or -1; off has n entries.
__device__ __forceinline__ int last_le(const int32_t* __restrict__ off, int n, int x) {
    int lo = 0, hi = n;  // first index with off[idx] > x
    while (lo < hi) {
        int mid = (lo + hi) >> 1;
        if (off[mid] <= x) lo = mid + 1; else hi = mid;
    }
    return lo - 1;
}

__device__ __forceinline__ void check_offsets(const int32_t* __restrict__ off, int count,
                                              int64_t last, uint32_t bit, uint32_t* err,
                                              int64_t tid, int64_t nthreads) {
    // off has count + 1 entries
    bool bad = false;
    for (int64_t i = tid; i <= count; i += nthreads) {
        int v = off[i];
        if (i == 0 && v != 0) bad = true;
        if (i == count && v != last) bad = true;
        if (i > 0 && v < off[i - 1]) bad = true;
    }
    if (bad) atomicOr(err, bit);
}

// a0: tok_traj[t] = trajectory of token t (-1 if the offsets do not cover it); O1 validation.
__global__ void __launch_bounds__(256)
segment_expand_kernel(const int32_t* __restrict__ step_off, const int32_t* __restrict__ traj_off,
                      const int32_t* __restrict__ group_off, int64_t n_tok, int n_steps,
                      int n_traj, int n_groups, int32_t* __restrict__ tok_traj,
                      uint32_t* __restrict__ err) {
    int64_t tid = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int64_t nthreads = (int64_t)gridDim.x * blockDim.x;
    check_offsets(step_off, n_steps, n_tok, AWR_ERRBIT_STEP_OFF, err, tid, nthreads);
    check_offsets(traj_off, n_traj, n_steps, AWR_ERRBIT_TRAJ_OFF, err, tid, nthreads);
    check_offsets(group_off, n_groups, n_traj, AWR_ERRBIT_GROUP_OFF, err, tid, nthreads);
    for (int64_t t = tid; t < n_tok; t += nthreads) {
        int s = last_le(step_off, n_steps + 1, (int)t);
        int i = -1;
        if (s >= 0 && s < n_steps) {
            i = last_le(traj_off, n_traj + 1, s);
            if (i >= n_traj) i = -1;
        }
        tok_traj[t] = i;
    }
}

// a1 (kernel 1): one warp per group, lanes stride over the group's trajectories, warp-shuffle
// reductions in a fixed order.  Also O6: traj_scale_i = loss_scale / (NG G_g) * n_i.
__global__ void __launch_bounds__(128)
group_advantage_kernel(const float* __restrict__ rewards, const int32_t* __restrict__ group_off,
                       const int32_t* __restrict__ traj_off, int n_groups, int n_traj,
                       uint32_t flags, int normalizer, float k_norm, float loss_scale,
                       float* __restrict__ adv, float* __restrict__ traj_scale,
                       const uint32_t* __restrict__ n_mixed) {
    int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (warp >= n_groups) return;
    int lo = min(max(group_off[warp], 0), n_traj);
    int hi = min(max(group_off[warp + 1], lo), n_traj);
    int G = hi - lo;
    if (G <= 0) return;
    float first = rewards[lo];
    float sum = 0.f;
    bool differs = false;
    for (int i = lo + lane; i < hi; i += 32) {
        float r = rewards[i];
        sum += r;
        differs |= (r != first);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(kFull, sum, o);
    differs = __any_sync(kFull, differs);
    float mu = sum / (float)G;
    float ss = 0.f;
    for (int i = lo + lane; i < hi; i += 32) {
        float d = rewards[i] - mu;
        ss += d * d;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(kFull, ss, o);
    const bool filter = (flags & AWR_FLAG_SUCCESS_FILTER) != 0;   // RAFT++ (:65): A = 1[R > 0]
    bool zero = !differs || G == 1;                       // A2: exact zero, no eps
    float denom = (flags & AWR_FLAG_SAMPLE_STD) ? (float)(G - 1) : (float)G;
    float inv_sigma = zero ? 0.f : 1.0f / sqrtf(ss / denom);
    // A1: mean over groups; with dynamic sampling (:63) over the mixed groups only, and a
    // uniform group contributes nothing at all
    const bool skip = (flags & AWR_FLAG_SKIP_UNIFORM) != 0;
    const bool dropped = skip && !differs;
    const float ng = (skip && n_mixed) ? (float)(*n_mixed) : (float)n_groups;
    float kappa = (ng > 0.f && !dropped) ? 1.0f / (ng * (float)G) : 0.f;
    for (int i = lo + lane; i < hi; i += 32) {
        adv[i] = dropped ? 0.f
                         : (filter ? (rewards[i] > 0.f ? 1.f : 0.f) : (zero ? 0.f : (rewards[i] - mu) * inv_sigma));
        if (traj_scale) {
            float n_i;
            if (normalizer == AWR_NORM_CONST_K) {
                n_i = 1.0f / k_norm;
            } else {
                int steps = traj_off[i + 1] - traj_off[i];
                n_i = steps > 0 ? 1.0f / (float)steps : 0.f;
            }
            traj_scale[i] = loss_scale * kappa * n_i;
        }
    }
}

// a3, last stage: loss = -sum_t term_t in a fixed order (thread-strided partial sums in fp64,
// then a fixed tree), clip_count = number of trigger flags.  One block: n_tok <= a few 10^5.
__global__ void __launch_bounds__(1024)
final_reduce_kernel(const float* __restrict__ tok_term, const uint8_t* __restrict__ tok_flag,
                    int64_t n_tok, float* __restrict__ loss, int64_t* __restrict__ clip_count,
                    int64_t* __restrict__ dual_count) {
    __shared__ double s_sum[1024];
    __shared__ unsigned long long s_cnt[1024];   // trigger count in the low, dual hits in the high 32 bits
    double acc = 0.0;
    unsigned long long cnt = 0;
    for (int64_t t = threadIdx.x; t < n_tok; t += 1024) {
        acc += (double)tok_term[t];
        const uint8_t f = tok_flag[t];
        cnt += ((f & kFlagTrig) ? 1ull : 0ull) + ((f & kFlagDual) ? (1ull << 32) : 0ull);
    }
    s_sum[threadIdx.x] = acc;
    s_cnt[threadIdx.x] = cnt;
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
            s_sum[threadIdx.x] += s_sum[threadIdx.x + o];
            s_cnt[threadIdx.x] += s_cnt[threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        *loss = (float)(-s_sum[0]);
        *clip_count = (int64_t)(s_cnt[0] & 0xffffffffull);
        if (dual_count) *dual_count = (int64_t)(s_cnt[0] >> 32);
    }
}

cudaError_t launch_segment_expand(const int32_t* step_off, const int32_t* traj_off,
                                  const int32_t* group_off, int64_t n_tok, int n_steps,
                                  int n_traj, int n_groups, int32_t* tok_traj, uint32_t* err,
                                  int num_sms, cudaStream_t st) {
    int64_t work = n_tok > n_steps + 1 ? n_tok : n_steps + 1;
    int blocks = (int)((work + 255) / 256);
    if (blocks < 1) blocks = 1;
    if (blocks > num_sms * 8) blocks = num_sms * 8;   // 8 CTAs of 256 threads per SM: one wave
    segment_expand_kernel<<<blocks, 256, 0, st>>>(step_off, traj_off, group_off, n_tok, n_steps,
                                                  n_traj, n_groups, tok_traj, err);
    return cudaGetLastError();
}

// Dynamic sampling: number of groups whose rewards are not all equal.  One warp per
// group, an integer atomic (order-independent, so the result is deterministic).
__global__ void __launch_bounds__(128)
count_mixed_groups_kernel(const float* __restrict__ rewards, const int32_t* __restrict__ group_off,
                          int n_groups, int n_traj, uint32_t* __restrict__ n_mixed) {
    int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (warp >= n_groups) return;
    int lo = min(max(group_off[warp], 0), n_traj);
    int hi = min(max(group_off[warp + 1], lo), n_traj);
    if (hi <= lo) return;
    const float first = rewards[lo];
    bool differs = false;
    for (int i = lo + lane; i < hi; i += 32) differs |= (rewards[i] != first);
    differs = __any_sync(kFull, differs);
    if (lane == 0 && differs) atomicAdd(n_mixed, 1u);
}

cudaError_t launch_group_advantage(const float* rewards, const int32_t* group_off,
                                   const int32_t* traj_off, int n_groups, int n_traj,
                                   uint32_t flags, int normalizer, float k_norm,
                                   float loss_scale, float* adv, float* traj_scale,
                                   uint32_t* n_mixed, cudaStream_t st) {
    if (n_groups <= 0) return cudaSuccess;
    int blocks = (n_groups + 3) / 4;
    if ((flags & AWR_FLAG_SKIP_UNIFORM) && n_mixed) {       // *n_mixed was zeroed by the caller
        count_mixed_groups_kernel<<<blocks, 128, 0, st>>>(rewards, group_off, n_groups, n_traj, n_mixed);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    group_advantage_kernel<<<blocks, 128, 0, st>>>(rewards, group_off, traj_off, n_groups, n_traj,
                                                   flags, normalizer, k_norm, loss_scale, adv,
                                                   traj_scale, n_mixed);
    return cudaGetLastError();
}

cudaError_t launch_final_reduce(const float* tok_term, const uint8_t* tok_flag, int64_t n_tok,
                                float* loss, int64_t* clip_count, int64_t* dual_count,
                                cudaStream_t st) {
    final_reduce_kernel<<<1, 1024, 0, st>>>(tok_term, tok_flag, n_tok, loss, clip_count, dual_count);
    return cudaGetLastError();
}

}  // namespace awr
