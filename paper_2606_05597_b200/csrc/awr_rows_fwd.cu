// Forward-only streaming row kernel: a2 (one-pass log-sum-exp + target gather) and a3 (ratio /
// clip / normalizer) with NO gradient, for bf16 vocabularies.  This is awr_loss_fwd's kernel: the
// proximal log-prob recomputation of PAPER.md:436 and the per-token entropy diagnostic (:232,
// :341).  Each logit is read from HBM exactly once and nothing is written but a few bytes per row.
//
// Nothing has to stay on chip between passes, so - unlike the fwd+bwd kernels - a row is not
// split over a cluster and is never resident: one persistent CTA per SM streams whole rows
// through a ring of 32 KB shared-memory stages filled by ONE producer thread with 1-D TMA bulk
// copies (cp.async.bulk + mbarrier complete_tx; a copy instruction holds its issuing thread for a
// few hundred clocks whatever its size, so stages are large and one thread is enough), six
// stages = 192 KB in flight per SM (Little: 6.5 TB/s x ~1.5 us / 148 SMs = 66 KB).  16 consumer
// warps drain a stage together: every thread takes 4 coalesced 16-byte units (32 logits), moves
// them to registers, takes their max with packed bf16x2 max, rescales its running (max, sum)
// state ONCE per stage and then issues 32 independent ex2 - one MUFU per logit, the secondary
// bound of the pass (16 / clk / SM: 1,024 clocks per stage against ~1,400 at the HBM rate).
// At the end of a row every warp publishes its partial state in a shared-memory slot and goes
// straight on to the next row; a 17th warp merges the 16 states and evaluates a3 a row behind
// (mbarrier hand-shakes, no block-wide barrier anywhere in the row loop).
// Rows are dealt round-robin to CTAs: a static schedule, so results are bit-reproducible.
#include "awr_common.cuh"
#include "awr_kernels.h"
#include "awr_ptx.cuh"

namespace awr {

constexpr int kFwdWarps = 16;                       // consumer warps
constexpr int kFwdConsumers = kFwdWarps * 32;
constexpr int kFwdThreads = kFwdConsumers + 64;     // + the producer warp + the a3 warp
constexpr int kFwdRounds = 4;                       // 16-byte units per thread per stage
constexpr int kFwdStageUnits = kFwdConsumers * kFwdRounds;
constexpr int kFwdStageBytes = kFwdStageUnits * 16; // 32 KB
constexpr int kFwdStages = 6;
constexpr int kFwdSlots = 8;                        // per-row state slots in flight (> kFwdStages)
constexpr int kFwdCtrlBytes = 2048;
constexpr int kFwdSmemBytes = kFwdCtrlBytes + kFwdStages * kFwdStageBytes;
constexpr uint32_t kFwdNegInf2 = 0xff80ff80u;       // bf16x2 (-inf, -inf)
static_assert(kFwdSmemBytes <= 232448, "227 KB of dynamic shared memory per CTA");

struct FwdCtrl {
    uint64_t full[kFwdStages];
    uint64_t empty[kFwdStages];
    uint64_t done[kFwdSlots];                // all 16 consumer warps have published the row's state
    uint64_t freed[kFwdSlots];               // the a3 warp has read the slot
    float2 stats[kFwdSlots][kFwdWarps];      // [slot][warp] (max, sum) of the warp's share of the row
    float statz[kFwdSlots][kFwdWarps];       // [slot][warp] sum e z (entropy output only)
};
static_assert(sizeof(FwdCtrl) <= kFwdCtrlBytes, "control block");

// Three roles, no block-wide barrier after the prologue:
//   warps 0..15  consumers: ring stage -> registers -> (max, sum) state; publish it per row
//   warp 16      producer: lane 0 issues one 32 KB bulk copy per stage
//   warp 17      a3: merges the 16 published states of a row and evaluates the token scalars,
//                with the row's header loads issued a row ahead; consumers never wait for it
//                (only for a free state slot, 8 rows later)
template <bool ENT>
__global__ void __launch_bounds__(kFwdThreads, 1)
rows_fwd_kernel(RowArgs a, int units_per_row) {
    using namespace ptx;
    extern __shared__ __align__(128) uint8_t smem[];
    FwdCtrl* ctrl = reinterpret_cast<FwdCtrl*>(smem);
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    const uint32_t ring = smem_u32(smem + kFwdCtrlBytes);
    const uint32_t full0 = smem_u32(&ctrl->full[0]);
    const uint32_t empty0 = smem_u32(&ctrl->empty[0]);
    const uint32_t done0 = smem_u32(&ctrl->done[0]);
    const uint32_t freed0 = smem_u32(&ctrl->freed[0]);
    const int nch = (units_per_row + kFwdStageUnits - 1) / kFwdStageUnits;   // stages per row
    const int64_t row_bytes = a.ld * 2;

    if (tid == 0) {
        for (int s = 0; s < kFwdStages; ++s) { mbar_init(full0 + 8u * s, 1); mbar_init(empty0 + 8u * s, kFwdWarps); }
        for (int s = 0; s < kFwdSlots; ++s) { mbar_init(done0 + 8u * s, kFwdWarps); mbar_init(freed0 + 8u * s, 1); }
        fence_mbar_init();
    }
    __syncthreads();

    if (warp == kFwdWarps) {
        // ===================== producer: one thread, one bulk copy per stage
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int64_t row = blockIdx.x; row < a.n_tok; row += gridDim.x) {
                const uint8_t* src = reinterpret_cast<const uint8_t*>(a.logits) + row * row_bytes;
                for (int c = 0; c < nch; ++c) {
                    const int u0 = c * kFwdStageUnits;
                    const uint32_t bytes = (uint32_t)min(kFwdStageUnits, units_per_row - u0) * 16u;
                    mbar_wait(empty0 + 8u * stage, phase ^ 1u);
                    mbar_expect_tx(full0 + 8u * stage, bytes);
                    bulk_load(ring + (uint32_t)stage * kFwdStageBytes, src + (int64_t)u0 * 16, bytes,
                              full0 + 8u * stage);
                    if (++stage == kFwdStages) { stage = 0; phase ^= 1u; }
                }
            }
        }
        return;
    }

    if (warp == kFwdWarps + 1) {
        // ===================== a3: one warp, a row behind the consumers
        int slot = 0;
        uint32_t sphase = 0;
        RowHeader h, hn;
        bool valid = false, validn = false;
        if (lane == 0 && blockIdx.x < a.n_tok) hn = load_row_header(a, blockIdx.x, validn, true);
        for (int64_t row = blockIdx.x; row < a.n_tok; row += gridDim.x) {
            h = hn; valid = validn;
            {   // the next row's header: its loads are in flight while this row is waited for
                const int64_t nrow = row + gridDim.x;
                if (lane == 0 && nrow < a.n_tok) hn = load_row_header(a, nrow, validn, true);
            }
            mbar_wait(done0 + 8u * slot, sphase);
            const bool mine = lane < kFwdWarps;
            const float2 st = ctrl->stats[slot][lane & (kFwdWarps - 1)];
            const float stz = ENT ? ctrl->statz[slot][lane & (kFwdWarps - 1)] : 0.f;
            __syncwarp();
            if (lane == 0) mbar_arrive(freed0 + 8u * slot);
            float M = mine ? st.x : -INFINITY;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(kFull, M, o));
            const float rs = (!mine || st.x == -INFINITY) ? 0.f : ex2_approx((st.x - M) * kLog2e);
            float S = st.y * rs;
            float SZ = stz * rs;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                S += __shfl_xor_sync(kFull, S, o);
                if (ENT) SZ += __shfl_xor_sync(kFull, SZ, o);
            }
            if (lane == 0) {
                const float lse_rest = M + logf(S);                      // -inf: nothing but the target
                const TokenScalars ts = token_scalars(h, lse_rest, valid, a.clip_eps, a.stale_cap, a.dual_c);
                store_token_outputs(a, row, h, ts, valid);
                if (ENT) a.token_entropy[row] = valid ? row_entropy(ts.lse, M, SZ, ts.lp, h.zy) : 0.f;
            }
            if (++slot == kFwdSlots) { slot = 0; sphase ^= 1u; }
        }
        return;
    }

    // ===================== consumers
    int stage = 0;
    uint32_t phase = 0;
    int slot = 0;
    uint32_t sphase = 0;
    int y_next = -1;
    if (blockIdx.x < a.n_tok) y_next = a.target_ids[blockIdx.x];
    for (int64_t row = blockIdx.x; row < a.n_tok; row += gridDim.x) {
        const int y = y_next;
        {
            const int64_t nrow = row + gridDim.x;
            if (nrow < a.n_tok) y_next = a.target_ids[nrow];
        }
        const bool valid = (y >= 0) && (y < a.V);
        // the target entry is left out of the (max, sum) state (token_scalars works from lse_rest)
        const int y_unit = valid ? (y >> 3) : -1;
        const int y_word = (y & 7) >> 1;
        const uint32_t y_keep = (y & 1) ? 0x0000ffffu : 0xffff0000u;    // the OTHER half of the word

        float m = -INFINITY, s = 0.f, sz = 0.f;
        for (int c = 0; c < nch; ++c) {
            const int u0 = c * kFwdStageUnits;
            const int left = units_per_row - u0;                         // units in this stage (> 0)
            mbar_wait(full0 + 8u * stage, phase);
            const uint32_t src = ring + (uint32_t)stage * kFwdStageBytes + (uint32_t)tid * 16u;
            uint32_t v[kFwdRounds][4];
            uint32_t mx2 = kFwdNegInf2;
#pragma unroll
            for (int k = 0; k < kFwdRounds; ++k) {
                const int u = k * kFwdConsumers + tid;
                if (u < left) {
                    lds128(v[k], src + k * (kFwdConsumers * 16));
                } else {
                    v[k][0] = v[k][1] = v[k][2] = v[k][3] = kFwdNegInf2;
                }
                if (u0 + u == y_unit) {
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        v[k][j] = (j == y_word) ? ((v[k][j] & y_keep) | (kFwdNegInf2 & ~y_keep)) : v[k][j];
                }
                mx2 = max_bf16x2(mx2, max_bf16x2(max_bf16x2(v[k][0], v[k][1]), max_bf16x2(v[k][2], v[k][3])));
            }
            // the registers hold the data: hand the stage back before the MUFU-bound part
            __syncwarp();
            if (lane == 0) mbar_arrive(empty0 + 8u * stage);
            if (++stage == kFwdStages) { stage = 0; phase ^= 1u; }

            const float cm = fmaxf(bf16_lo(mx2), bf16_hi(mx2));
            if (cm > m) {                                                // rescale once per stage
                const float sc = ex2_approx((m - cm) * kLog2e);          // m = -inf: 0 (s is 0 then)
                s *= sc;
                if (ENT) sz *= sc;
                m = cm;
            }
            const float nref = (m == -INFINITY) ? 0.f : -m * kLog2e;
            // FFMA2 / FADD2: the (low, high) elements of a word are one packed f32x2 operation (half
            // the issue slots of the scaling and the sums; the kernel sat at 70 % issue-slot use)
            const float2 l2 = make_float2(kLog2e, kLog2e), nref2 = make_float2(nref, nref);
            float2 acc[4] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f),
                             make_float2(0.f, 0.f)};
            float2 accz = make_float2(0.f, 0.f);
#pragma unroll
            for (int k = 0; k < kFwdRounds; ++k) {
                // a ragged last stage: skip the rounds in which this whole warp holds padding
                if (k * kFwdConsumers + (warp << 5) >= left) continue;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const float2 z = make_float2(bf16_lo(v[k][j]), bf16_hi(v[k][j]));
                    const float2 x = ptx::fma_f32x2(z, l2, nref2);
                    const float2 e = make_float2(ex2_approx(x.x), ex2_approx(x.y));
                    acc[j] = ptx::add_f32x2(acc[j], e);
                    if (ENT)
                        accz = ptx::fma_f32x2(e, make_float2(fmaxf(z.x, kZFloor), fmaxf(z.y, kZFloor)), accz);
                }
            }
            s += ((acc[0].x + acc[0].y) + (acc[1].x + acc[1].y)) + ((acc[2].x + acc[2].y) + (acc[3].x + acc[3].y));
            if (ENT) sz += accz.x + accz.y;
        }

        // ---- merge the 32 lanes and publish the warp's state of this row; no waiting for the
        // other warps (only for the a3 warp to have read this slot 8 rows ago)
        float wm = m;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) wm = fmaxf(wm, __shfl_xor_sync(kFull, wm, o));
        const float sc = (m == -INFINITY) ? 0.f : ex2_approx((m - wm) * kLog2e);
        float ws = s * sc;
        float wz = ENT ? sz * sc : 0.f;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            ws += __shfl_xor_sync(kFull, ws, o);
            if (ENT) wz += __shfl_xor_sync(kFull, wz, o);
        }
        if (lane == 0) {
            mbar_wait(freed0 + 8u * slot, sphase ^ 1u);
            ctrl->stats[slot][warp] = make_float2(wm, ws);
            if (ENT) ctrl->statz[slot][warp] = wz;
            mbar_arrive(done0 + 8u * slot);                              // release: the stores above
        }
        if (++slot == kFwdSlots) { slot = 0; sphase ^= 1u; }
    }
}

bool rows_fwd_supported(int64_t V, int64_t ld, int dtype) {
    return dtype == AWR_DTYPE_BF16 && V % 8 == 0 && ld % 8 == 0 && V >= 8 && V / 8 < (1 << 27);
}

cudaError_t launch_rows_fwd(const RowArgs& a, int num_sms, cudaStream_t st) {
    if (a.n_tok <= 0) return cudaSuccess;
    if (!rows_fwd_supported(a.V, a.ld, AWR_DTYPE_BF16) || a.dlogits != nullptr) return cudaErrorInvalidValue;
    static PerDeviceInt attr_set[2];                 // the attribute is per device
    const int dev = PerDeviceInt::device();
    const bool ent = a.token_entropy != nullptr;
    if (attr_set[ent].get(dev) < 0) {
        cudaError_t e = ent ? cudaFuncSetAttribute(rows_fwd_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kFwdSmemBytes)
                            : cudaFuncSetAttribute(rows_fwd_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kFwdSmemBytes);
        if (e != cudaSuccess) return e;
        attr_set[ent].set(dev, 1);
    }
    const int grid = (int)(a.n_tok < num_sms ? a.n_tok : num_sms);
    const int units = (int)(a.V / 8);
    if (ent) rows_fwd_kernel<true><<<grid, kFwdThreads, kFwdSmemBytes, st>>>(a, units);
    else rows_fwd_kernel<false><<<grid, kFwdThreads, kFwdSmemBytes, st>>>(a, units);
    return cudaGetLastError();
}

}  // namespace awr
