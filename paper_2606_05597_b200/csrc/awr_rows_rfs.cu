// Register-file row kernel with a service warp ("RFS"): a2 + a3 + a4 for bf16 vocabularies with one
// HBM read and one HBM write per element.  PAPER.md:57 (Eq. 1), :435; gradient SURVEY.md 8(c) O8.
//
// Same residency idea as awr_rows_rf.cu - a row is split over a 2-CTA cluster and each half lives in
// the REGISTER FILE of its SM between the log-sum-exp pass and the gradient pass - but nobody who
// holds data ever issues a copy or waits at a barrier:
//   * 15 consumer warps per CTA hold the row half (round r of warp w = the 32 16-byte units
//     [(15 r + w) 32, +32) of the half: the rounds of all warps are CONTIGUOUS in memory) and one
//     service warp does everything else.
//   * Loads: the ring is two slots of 10 rounds x 15 warps (75 KB each = the whole next row half);
//     ONE 1-D TMA bulk copy per slot, issued by the service lane as soon as the 15 warps have moved
//     the slot to registers.  (A bulk copy holds its issuing warp for ~600 clocks whatever its
//     size: with per-warp 5 KB copies that was 7 x 600 clocks per row of every data warp.)
//   * Gradient: the consumers write e * F into a staging buffer of 5 rounds x 15 warps (37.5 KB,
//     contiguous in memory, two buffers: all the shared memory the ring leaves) at shared-memory
//     speed (128 B/clk) and go on; the service lane hands each full buffer to a TMA bulk store.
//     An SM writes to L2 at 32 B/clk whatever the instruction (measured for per-lane stores and for
//     TMA stores alike), so the 148 KB of a row half need 4.7 k clocks of that port; what staging
//     buys is that the last 75 KB drain while the warps are already in the next row - and the
//     first 75 KB too: the waits for a free staging buffer are filled with pass 0 (ring ->
//     registers, max) of the NEXT row, slot by slot, into the registers whose gradient has just
//     been staged.  With that the kernel is HBM-bound (config 1: 3.87 ms, 0.99 of the copy peak).
//   * Exchange: every consumer warp sends its (max, sum[, sum e z]) with st.async to BOTH CTAs; the
//     16 bytes complete a transaction count on the receiver's mbarrier - no cluster barrier, no
//     fence.  The service warp of each CTA merges the 30 states, evaluates a3 once (header loads
//     issued a row ahead) and publishes (c_t, lse, c_t (p_y - 1)) in shared memory; the consumers
//     wait for that on an mbarrier and scale their registers by c_t exp(m_w - lse).
// Rows are dealt round-robin to clusters (static schedule, fixed merge order: bit-reproducible).
#include "awr_common.cuh"
#include "awr_kernels.h"
#include "awr_ptx.cuh"

namespace awr {

constexpr int kSvConsumers = 15;                         // data warps per CTA
constexpr int kSvThreads = (kSvConsumers + 1) * 32;      // + the service warp
constexpr int kSvRoundUnits = kSvConsumers * 32;         // 16-byte units per round of the CTA (480)
constexpr int kSvRoundBytes = kSvRoundUnits * 16;        // 7,680
constexpr int kSvSlotRounds = 10;                        // rounds per ring slot / per TMA load
constexpr int kSvSlotBytes = kSvSlotRounds * kSvRoundBytes;           // 76,800
constexpr int kSvStageRounds = 5;                        // rounds per staging buffer / per TMA store (all the
                                                         // shared memory that is left: 2 x 37.5 KB)
constexpr int kSvStageBufs = 2;
constexpr int kSvStageBytes = kSvStageRounds * kSvRoundBytes;         // 38,400
constexpr int kSvCtrlBytes = 2048;
constexpr int kSvSmemBytes = kSvCtrlBytes + 2 * kSvSlotBytes + kSvStageBufs * kSvStageBytes;
constexpr int kSvMinNU = 3, kSvMaxNU = 2 * kSvSlotRounds;            // rounds per row half
constexpr uint32_t kSvNegInf2 = 0xff80ff80u;             // bf16x2 (-inf, -inf)
static_assert(kSvSmemBytes <= 232448, "227 KB of dynamic shared memory per CTA");

struct SvCtrl {
    uint64_t full[2], empty[2];                          // ring slots
    uint64_t sfull[kSvStageBufs], sfree[kSvStageBufs];   // staging buffers
    uint64_t stats_full[2];                              // [row parity] 30 x 16 bytes have arrived
    uint64_t row_ready[2];                               // [row parity] rowinfo is valid
    float4 stats[2][2 * kSvConsumers + 2];               // [row parity][cluster-wide warp] (m, s, sz, -)
    float4 rowinfo[2];                                   // [row parity] (c_t, lse, c_t (p_y - 1), y as bits)
};
static_assert(sizeof(SvCtrl) <= kSvCtrlBytes, "control block");

struct SvPlan {
    int half_units[2];   // 16-byte units of the row held by CTA rank 0 / 1
    int num_clusters;
};

// NU = rounds per row half = ceil(max half units / 480), compile time: the register array of a
// consumer thread is v[NU][4] (one 16-byte unit per round).
template <int NU, bool ENT>
__global__ void __launch_bounds__(kSvThreads, 1)
rows_rfs_kernel(RowArgs a, SvPlan p) {
    using namespace ptx;
    constexpr int NCH = (NU + kSvSlotRounds - 1) / kSvSlotRounds;          // ring slots in use (1 or 2)
    extern __shared__ __align__(128) uint8_t smem[];
    SvCtrl* ctrl = reinterpret_cast<SvCtrl*>(smem);
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    const uint32_t rank = cluster_ctarank();
    const int cluster = (int)cluster_id_x();
    const int half_units = p.half_units[rank];
    const int half_base = rank ? p.half_units[0] : 0;                      // first unit of this half
    const int nr = (half_units + kSvRoundUnits - 1) / kSvRoundUnits;       // rounds of THIS half (<= NU)
    const int npieces = (nr + kSvStageRounds - 1) / kSvStageRounds;        // staging buffers per row
    const uint32_t ring = smem_u32(smem + kSvCtrlBytes);
    const uint32_t stage = ring + 2u * kSvSlotBytes;
    const uint32_t full0 = smem_u32(&ctrl->full[0]), empty0 = smem_u32(&ctrl->empty[0]);
    const uint32_t sfull0 = smem_u32(&ctrl->sfull[0]), sfree0 = smem_u32(&ctrl->sfree[0]);
    const uint32_t stats_full0 = smem_u32(&ctrl->stats_full[0]), ready0 = smem_u32(&ctrl->row_ready[0]);
    const int n_tok = (int)a.n_tok;                     // < 2^31 (checked by the entry point)
    const int nc = p.num_clusters;
    const int64_t row_bytes = a.ld * 2;
    const bool backward = a.dlogits != nullptr;

    if (tid == 0) {
        for (int s = 0; s < 2; ++s) {
            mbar_init(full0 + 8u * s, 1);
            mbar_init(empty0 + 8u * s, kSvConsumers);
            mbar_init(stats_full0 + 8u * s, 1);
            mbar_init(ready0 + 8u * s, 1);
        }
        for (int b = 0; b < kSvStageBufs; ++b) { mbar_init(sfull0 + 8u * b, kSvConsumers); mbar_init(sfree0 + 8u * b, 1); }
        fence_mbar_init();
    }
    __syncthreads();
    cluster_arrive();     // both CTAs' barriers exist before any st.async crosses over
    cluster_wait();

    if (warp == kSvConsumers) {
        // =============================================================== service warp
        const uint8_t* lbase = reinterpret_cast<const uint8_t*>(a.logits) + (int64_t)half_base * 16;
        uint8_t* gbase = reinterpret_cast<uint8_t*>(a.dlogits) + (int64_t)half_base * 16;
        auto load_slot = [&](int s, int row) {            // lane 0: one bulk copy fills the slot
            const int u0 = s * kSvSlotRounds * kSvRoundUnits;
            const int units = min(kSvSlotRounds * kSvRoundUnits, half_units - u0);
            if (lane == 0 && units > 0) {
                mbar_expect_tx(full0 + 8u * s, (uint32_t)units * 16u);
                bulk_load(ring + (uint32_t)s * kSvSlotBytes, lbase + (int64_t)row * row_bytes + (int64_t)u0 * 16,
                          (uint32_t)units * 16u, full0 + 8u * s);
            }
        };
#pragma unroll
        for (int s = 0; s < NCH; ++s) load_slot(s, cluster);
        RowHeader h, hn;
        bool valid = false, validn = false;
        if (lane == 0) hn = load_row_header(a, cluster, validn, true);
        uint32_t gpiece = 0;                              // staging buffers handed to the TMA so far
        int it = 0;
        for (int row = cluster; row < n_tok; row += nc, ++it) {
            const int par = it & 1;
            const uint32_t ph2 = (uint32_t)(it >> 1) & 1u;      // phase of the per-parity barriers
            h = hn; valid = validn;
            const int next = row + nc;
            if (lane == 0) {
                mbar_expect_tx(stats_full0 + 8u * par, 2u * kSvConsumers * 16u);
                if (next < n_tok) hn = load_row_header(a, next, validn, true);   // in flight behind this row
            }
            // ---- ring: refill each slot with the next row as soon as the 15 warps have read it out
            if (next < n_tok) {
#pragma unroll
                for (int s = 0; s < NCH; ++s) {
                    if (s * kSvSlotRounds < nr) mbar_wait(empty0 + 8u * s, (uint32_t)it & 1u);
                    load_slot(s, next);
                }
            }
            // ---- a3: merge the 30 (max, sum) states, token scalars, publish (c_t, lse, gy)
            mbar_wait(stats_full0 + 8u * par, ph2);
            const bool mine = lane < 2 * kSvConsumers;
            const float4 st = ctrl->stats[par][mine ? lane : 0];
            // max over the warp in ONE instruction: floats order like their bits once the negative
            // ones are flipped (this chain is on the critical path of every data warp of the cluster)
            int mi = __float_as_int(mine ? st.x : -INFINITY);
            mi ^= (mi >> 31) & 0x7fffffff;
            mi = __reduce_max_sync(kFull, mi);
            mi ^= (mi >> 31) & 0x7fffffff;
            const float M = __int_as_float(mi);
            const float rs = (!mine || st.x == -INFINITY) ? 0.f : ex2_approx((st.x - M) * kLog2e);
            float S = st.y * rs;
            float SZ = ENT ? st.z * rs : 0.f;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                S += __shfl_xor_sync(kFull, S, o);
                if (ENT) SZ += __shfl_xor_sync(kFull, SZ, o);
            }
            if (lane == 0) {
                const float lse_rest = M + fast_log(S);               // -inf if nothing but the target
                const TokenScalars ts = token_scalars(h, lse_rest, valid, a.clip_eps, a.stale_cap, a.dual_c);
                ctrl->rowinfo[par] = make_float4(ts.coef, ts.lse, ts.gy, 0.f);
                mbar_arrive(ready0 + 8u * par);                       // release: rowinfo is visible
                if (rank == 0) {
                    store_token_outputs(a, row, h, ts, valid);
                    if (ENT) a.token_entropy[row] = valid ? row_entropy(ts.lse, M, SZ, ts.lp, h.zy) : 0.f;
                }
            }
            __syncwarp();
            // ---- gradient: every full staging buffer goes out with one TMA bulk store
            if (backward) {
                uint8_t* g = gbase + (int64_t)row * row_bytes;
                for (int pc = 0; pc < npieces; ++pc, ++gpiece) {
                    const uint32_t b = gpiece & 1u;
                    mbar_wait(sfull0 + 8u * b, (gpiece >> 1) & 1u);
                    if (lane == 0) {
                        const int u0 = pc * kSvStageRounds * kSvRoundUnits;
                        const int units = min(kSvStageRounds * kSvRoundUnits, half_units - u0);
                        bulk_store(g + (int64_t)u0 * 16, stage + b * kSvStageBytes, (uint32_t)units * 16u);
                        bulk_commit();
                        // all but this newest store have read their buffer out: the other buffer is free
                        bulk_wait_read<1>();
                        if (gpiece > 0) mbar_arrive(sfree0 + 8u * (b ^ 1u));
                    }
                    __syncwarp();
                }
            }
        }
        if (lane == 0) bulk_wait_all();                   // gradient writes complete before the CTA ends
    } else {
        // =============================================================== consumer warps
        // The entropy sum (sum e z) is always accumulated: its serial FMA chain costs nothing in the
        // MUFU-bound exp pass and keeps ptxas from hoisting the exponentials of the fully unrolled
        // loop ahead of their consumers (without it the same code spilled part of the row).
        constexpr bool want_ent = true;
        const uint32_t my_off = (uint32_t)(warp * 32 + lane) * 16u;      // byte offset inside a round
        const int my_unit0 = warp * 32 + lane;                           // unit of round 0
        uint32_t v[NU][4];
        uint32_t gpiece = 0;
        uint32_t mx2 = kSvNegInf2;

        // One ring slot of row index `it` -> registers (rounds [10 s, 10 s + 10)), target entry masked
        // to -inf (token_scalars works from lse_rest), packed running max; then the slot is released.
        auto load_slot = [&](int s, int it, int y_round, int y_word, uint32_t y_keep) {
            const bool have = s * kSvSlotRounds < nr;                                   // warp-uniform
            if (have) mbar_wait(full0 + 8u * s, (uint32_t)it & 1u);
            const uint32_t src = ring + (uint32_t)s * kSvSlotBytes + my_off;
#pragma unroll
            for (int kk = 0; kk < kSvSlotRounds; ++kk) {
                const int k = s * kSvSlotRounds + kk;
                if (k < NU) {
                    if (k * kSvRoundUnits + my_unit0 < half_units) {
                        lds128(v[k], src + (uint32_t)kk * kSvRoundBytes);
                    } else {
                        v[k][0] = v[k][1] = v[k][2] = v[k][3] = kSvNegInf2;
                    }
                    if (k == y_round) {
#pragma unroll
                        for (int j = 0; j < 4; ++j)
                            v[k][j] = (j == y_word) ? ((v[k][j] & y_keep) | (kSvNegInf2 & ~y_keep)) : v[k][j];
                    }
                    mx2 = max_bf16x2(mx2, max_bf16x2(max_bf16x2(v[k][0], v[k][1]), max_bf16x2(v[k][2], v[k][3])));
                }
            }
            if (have) {
                __syncwarp();                                 // the slot has been read out by the warp
                if (lane == 0) mbar_arrive(empty0 + 8u * s);
            }
        };
        // where the target of a row sits for this thread: its round (or -1), word and the OTHER half
        auto locate = [&](int y, int& y_round, int& y_word, uint32_t& y_keep) {
            const bool valid = (y >= 0) && (y < a.V);
            const int y_unit = valid ? (y >> 3) - half_base : -1;                       // unit inside this half
            const bool holder = y_unit >= 0 && y_unit < half_units && (y_unit % kSvRoundUnits) == my_unit0;
            y_round = holder ? y_unit / kSvRoundUnits : -1;
            y_word = (y & 7) >> 1;
            y_keep = (y & 1) ? 0x0000ffffu : 0xffff0000u;
        };

        int y = a.target_ids[cluster];
        int y_round, y_word;
        uint32_t y_keep;
        locate(y, y_round, y_word, y_keep);
#pragma unroll
        for (int s = 0; s < NCH; ++s) load_slot(s, 0, y_round, y_word, y_keep);     // pass 0 of the first row

        int it = 0;
        for (int row = cluster; row < n_tok; row += nc, ++it) {
            const int par = it & 1;
            const uint32_t ph2 = (uint32_t)(it >> 1) & 1u;
            const bool have_next = row + nc < n_tok;
            const int y_nx = have_next ? a.target_ids[row + nc] : -1;     // in flight behind the exp pass

            float m = fmaxf(bf16_lo(mx2), bf16_hi(mx2));
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(kFull, m, o));

            // ---- pass 1: z -> e = exp2((z - m) log2 e) as bf16, in registers; f32 sum
            const float nref = (m == -INFINITY) ? 0.f : -m * kLog2e;
            float acc[4] = {0.f, 0.f, 0.f, 0.f};
            float accz = 0.f;                          // sum e z (entropy output; the pass is MUFU-bound)
#pragma unroll
            for (int k = 0; k < NU; ++k) {
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const float z0 = bf16_lo(v[k][j]), z1 = bf16_hi(v[k][j]);
                    const float e0 = ex2_approx(fmaf(z0, kLog2e, nref));
                    const float e1 = ex2_approx(fmaf(z1, kLog2e, nref));
                    acc[j] += e0;
                    acc[j] += e1;
                    if (want_ent) {
                        accz = fmaf(e0, fmaxf(z0, kZFloor), accz);
                        accz = fmaf(e1, fmaxf(z1, kZFloor), accz);
                    }
                    v[k][j] = pack_bf16x2(e0, e1);
                }
            }
            float s = (acc[0] + acc[1]) + (acc[2] + acc[3]);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                s += __shfl_xor_sync(kFull, s, o);
                if (ENT) accz += __shfl_xor_sync(kFull, accz, o);     // merged only if it is an output
            }
            // ---- exchange: (m_w, s_w, sz_w) to both CTAs, data and signal in one st.async each
            if (lane < 2)
                st_async_f32x4(smem_u32(&ctrl->stats[par][(int)rank * kSvConsumers + warp]),
                               stats_full0 + 8u * par, (uint32_t)lane, m, s, accz, 0.f);

            // where the next row's target sits (for its pass 0, interleaved below)
            int yn_round, yn_word;
            uint32_t yn_keep;
            locate(y_nx, yn_round, yn_word, yn_keep);

            // ---- a3 runs on the service warp; wait for (c_t, lse, c_t (p_y - 1))
            mbar_wait(ready0 + 8u * par, ph2);
            const float4 ri = ctrl->rowinfo[par];

            // ---- pass 2 (a4): dlogits = e * (c_t exp(m - lse)) through the staging buffers, with pass
            // 0 of the NEXT row slot by slot in between: after ten rounds both staging buffers are
            // full and the warp would wait for the TMA store to drain one (32 B/clk); the registers
            // of those ten rounds are free, so the next row's first ring slot is moved into them
            // meanwhile.  e was taken relative to m (0 if the part held nothing finite); c_t = 0
            // (masked, zero advantage, clip triggered): F = +0 and e >= 0 give all-bits-zero products
            const float F = ri.x == 0.f ? 0.f : ri.x * ex2_approx(fmaf(-ri.y, kLog2e, -nref));
            const __nv_bfloat16 fh = __float2bfloat16_rn(F);
            const __nv_bfloat16 fl = __float2bfloat16_rn(F - __bfloat162float(fh));
            const uint32_t Fh = (uint32_t)__bfloat16_as_ushort(fh) * 0x00010001u;
            const uint32_t Fl = (uint32_t)__bfloat16_as_ushort(fl) * 0x00010001u;
            const uint32_t gy_bits = (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(ri.z));
            const uint32_t gy2 = (y & 1) ? (gy_bits << 16) : gy_bits;
            const int y_patch = ri.x != 0.f ? y_round : -1;
            mx2 = kSvNegInf2;
#pragma unroll
            for (int sl = 0; sl < NCH; ++sl) {
                if (backward) {
#pragma unroll
                    for (int kk2 = 0; kk2 < kSvSlotRounds; ++kk2) {
                        const int k = sl * kSvSlotRounds + kk2;
                        if (k < NU && k < nr) {                                   // k < nr: warp-uniform
                            const int kk = k % kSvStageRounds;
                            const uint32_t gp = gpiece + (uint32_t)(k / kSvStageRounds);
                            const uint32_t buf = stage + (gp & 1u) * kSvStageBytes;
                            if (kk == 0) mbar_wait(sfree0 + 8u * (gp & 1u), ((gp >> 1) & 1u) ^ 1u);
                            uint4 o;
                            o.x = fma_bf16x2(v[k][0], Fh, mul_bf16x2(v[k][0], Fl));
                            o.y = fma_bf16x2(v[k][1], Fh, mul_bf16x2(v[k][1], Fl));
                            o.z = fma_bf16x2(v[k][2], Fh, mul_bf16x2(v[k][2], Fl));
                            o.w = fma_bf16x2(v[k][3], Fh, mul_bf16x2(v[k][3], Fl));
                            if (k == y_patch) {                                   // target entry: c (p_y - 1)
                                o.x = y_word == 0 ? ((o.x & y_keep) | gy2) : o.x;
                                o.y = y_word == 1 ? ((o.y & y_keep) | gy2) : o.y;
                                o.z = y_word == 2 ? ((o.z & y_keep) | gy2) : o.z;
                                o.w = y_word == 3 ? ((o.w & y_keep) | gy2) : o.w;
                            }
                            sts128(buf + (uint32_t)kk * kSvRoundBytes + my_off, o);
                            if (kk == kSvStageRounds - 1 || k == nr - 1) {
                                fence_proxy_async();                              // generic writes -> TMA read
                                __syncwarp();
                                if (lane == 0) mbar_arrive(sfull0 + 8u * (gp & 1u));
                            }
                        }
                    }
                }
                if (have_next) load_slot(sl, it + 1, yn_round, yn_word, yn_keep);
            }
            if (backward) gpiece += (uint32_t)npieces;
            y = y_nx; y_round = yn_round; y_word = yn_word; y_keep = yn_keep;
        }
    }
    cluster_arrive();     // nobody leaves while the peer may still send to its shared memory
    cluster_wait();
}

// ---------------------------------------------------------------- host side
static bool make_sv_plan(int64_t V, int64_t ld, int dtype, SvPlan& p, int& nu) {
    if (dtype != AWR_DTYPE_BF16) return false;
    if (V % 8 != 0 || ld % 8 != 0) return false;
    const int64_t units = V / 8;
    const int64_t h0 = (units + 1) / 2;
    const int64_t n = (h0 + kSvRoundUnits - 1) / kSvRoundUnits;
    if (n < kSvMinNU || n > kSvMaxNU) return false;
    p.half_units[0] = (int)h0;
    p.half_units[1] = (int)(units - h0);
    p.num_clusters = 0;
    nu = (int)n;
    return true;
}

bool rows_rfs_supported(int64_t V, int64_t ld, int dtype) {
    SvPlan p;
    int nu;
    return make_sv_plan(V, ld, dtype, p, nu);
}

template <int NU, bool ENT>
static cudaError_t launch_sv(const RowArgs& a, SvPlan p, int num_sms, cudaStream_t st) {
    static PerDeviceInt cached;              // co-resident clusters (device query, cached per device)
    const int dev = PerDeviceInt::device();
    int max_clusters = cached.get(dev);
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(kSvThreads, 1, 1);
    cfg.dynamicSmemBytes = kSvSmemBytes;
    cfg.stream = st;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (max_clusters < 0) {
        cudaError_t e = cudaFuncSetAttribute(rows_rfs_kernel<NU, ENT>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, kSvSmemBytes);
        if (e != cudaSuccess) return e;
        cfg.gridDim = dim3(2 * num_sms, 1, 1);
        int n = 0;
        e = cudaOccupancyMaxActiveClusters(&n, rows_rfs_kernel<NU, ENT>, &cfg);
        if (e != cudaSuccess) return e;
        const int want = num_sms / 2;
        max_clusters = n < 1 ? 1 : (n > want ? want : n);
        cached.set(dev, max_clusters);
    }
    int nc = max_clusters;
    if ((int64_t)nc > a.n_tok) nc = (int)a.n_tok;
    p.num_clusters = nc;
    cfg.gridDim = dim3(2 * nc, 1, 1);
    return cudaLaunchKernelEx(&cfg, rows_rfs_kernel<NU, ENT>, a, p);
}

cudaError_t launch_rows_rfs(const RowArgs& a, int num_sms, cudaStream_t st) {
    if (a.n_tok <= 0) return cudaSuccess;
    SvPlan p;
    int nu = 0;
    if (!make_sv_plan(a.V, a.ld, AWR_DTYPE_BF16, p, nu)) return cudaErrorInvalidValue;
    switch (nu) {
#define AWR_SV_CASE(N)                                                                  \
    case N:                                                                             \
        return a.token_entropy != nullptr ? launch_sv<N, true>(a, p, num_sms, st)       \
                                          : launch_sv<N, false>(a, p, num_sms, st);
        AWR_SV_CASE(3) AWR_SV_CASE(4) AWR_SV_CASE(5) AWR_SV_CASE(6) AWR_SV_CASE(7) AWR_SV_CASE(8)
        AWR_SV_CASE(9) AWR_SV_CASE(10) AWR_SV_CASE(11) AWR_SV_CASE(12) AWR_SV_CASE(13)
        AWR_SV_CASE(14) AWR_SV_CASE(15) AWR_SV_CASE(16) AWR_SV_CASE(17) AWR_SV_CASE(18)
        AWR_SV_CASE(19) AWR_SV_CASE(20)
#undef AWR_SV_CASE
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace awr
