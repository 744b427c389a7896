// Register-file row kernel: a2 + a3 + a4 for bf16 vocabularies of 16K..163K entries with one HBM
// read and one HBM write per element.  PAPER.md:57 (Eq. 1), :435; gradient SURVEY.md 8(c) O8.
//
// Design:
//   * A 151,936-entry bf16 row (303,872 B) fits neither one SM's shared memory (227 KB) nor one
//     SM's register file (256 KB) next to the staging it needs, so a row is split across a
//     2-CTA thread-block cluster and each half (148 KB) lives in the REGISTER FILE of its SM:
//     16 warps x 32 lanes x up to 20 packed 16-byte units per lane.
//   * Shared memory is a pure FIFO between HBM and the registers: every warp owns a ring of
//     5 KB slots that TMA bulk copies (cp.async.bulk + mbarrier complete_tx) fill with its part
//     of the rows to come; a slot is refilled the moment the warp has moved it into registers,
//     so the whole next row (148 KB per SM) is in flight while the current row is being worked on.
//   * Pass 0 moves the warp's part to registers and takes its max with packed bf16x2 max.
//     Pass 1 replaces every logit, in registers, by e = exp2((z - m_w) log2 e) rounded to bf16
//     and sums the unrounded values in f32.  The 32 warps of the cluster exchange (m_w, s_w)
//     through distributed shared memory, one cluster barrier per row.  Pass 2 is then a packed
//     multiply: dlogits = e * (c_t exp(m_w - lse)), two bf16x2 instructions per pair (the factor
//     is split hi + lo so that it carries 16 significant bits), written with 16-byte coalesced
//     global stores straight from registers.  One MUFU and ~8 issue slots per element in total.
//   * Persistent: one cluster per SM pair, rows dealt round-robin to clusters (static schedule,
//     deterministic results).  Rows with c_t = 0 (masked, zero advantage, clip triggered) skip
//     pass 2 and are written as zeros.
#include "awr_common.cuh"
#include "awr_kernels.h"
#include "awr_ptx.cuh"

namespace awr {

constexpr int kRfParts = 32;                // warps per row (over the whole cluster)
// A bulk copy holds its issuing thread for ~450 clocks (measured with clock()), and a warp issues
// the copies of its ring one after the other: with 2 KB chunks (5 per row part) the refills were
// 2.2-2.7 k of the 5.4 k clocks of pass 0.  So chunks are as large as the ring allows: two slots of
// 10 rounds (5 KB), i.e. two copies per row part, issued while the part is moved to registers;
// they have the rest of the row's time to land.
constexpr int kRfChunkRounds = 10;          // rounds (32 units each) per slot / per TMA copy
constexpr int kRfChunkUnits = 32 * kRfChunkRounds;
constexpr int kRfSlotBytes = kRfChunkUnits * 16;
constexpr int kRfStageRounds = 4;           // rounds (512 B each) per staging buffer / per TMA store
constexpr int kRfCtrlBytes = 2048;
constexpr int kRfMinNU = 3, kRfMaxNU = 20;
constexpr uint32_t kNegInf2 = 0xff80ff80u;  // bf16x2 (-inf, -inf)

// Two shapes of the same kernel (CL CTAs per cluster x WARPS warps per CTA = 32 parts per row):
//   CL = 2, WARPS = 16: one CTA per SM, a row half per SM, 2 ring slots of 5 KB per warp (160 KB).
//   CL = 4, WARPS = 8 : two CTAs per SM (of different rows), a row quarter per CTA, 2 ring slots
//                       per warp (80 KB per CTA).  The two co-resident CTAs drift out of phase,
//                       so one's exp pass overlaps the other's load / store passes.
template <int CL>
struct RfShape {
    static constexpr int kWarps = kRfParts / CL;
    static constexpr int kThreads = kWarps * 32;
    static constexpr int kSlots = 2;
    static constexpr int kCtasPerSm = CL == 2 ? 1 : 2;
    // CL = 2: the gradient leaves through a per-warp staging area (two buffers of kRfStageRounds
    // rounds) and TMA bulk stores instead of per-lane 16-byte global stores
    static constexpr bool kStaged = CL == 2;
    static constexpr int kStageBytes = kStaged ? 2 * kRfStageRounds * 512 : 0;      // per warp
    static constexpr int kRingBytes = kWarps * kSlots * kRfSlotBytes;
    static constexpr int kSmemBytes = kRfCtrlBytes + kRingBytes + kWarps * kStageBytes;
};
static_assert(RfShape<2>::kSmemBytes <= 232448, "227 KB of dynamic shared memory per CTA");
static_assert(2 * (RfShape<4>::kSmemBytes + 1024) <= 233472, "two CTAs in 228 KB per SM");

struct RfPlan {
    int units_per_row;   // 16-byte units in one row (V / 8)
    int num_clusters;
};

struct RfCtrl {
    uint64_t full[16 * 8];         // one mbarrier per ring slot per warp (8 >= slots)
    float2 stats[2][kRfParts];     // [row parity][part] (max, sum) of every warp of the cluster
    float statz[2][kRfParts];      // [row parity][part] sum e z of the part (entropy output only)
};
static_assert(sizeof(RfCtrl) <= kRfCtrlBytes, "control block");


// ---------------------------------------------------------------- the kernel
// NU = rounds per warp part = ceil(max part units / 32); every round but the last is full for
// every warp (parts differ by at most one unit and NU is exact, see make_rf_plan).
template <int NU, int CL, bool ENT>
__global__ void __launch_bounds__(RfShape<CL>::kThreads, RfShape<CL>::kCtasPerSm)
rows_rf_kernel(RowArgs a, RfPlan p) {
    using namespace ptx;
    constexpr int kRfWarps = RfShape<CL>::kWarps;
    constexpr int kRfSlots = RfShape<CL>::kSlots;
    constexpr int NCH = (NU + kRfChunkRounds - 1) / kRfChunkRounds;
    extern __shared__ __align__(128) uint8_t smem[];
    RfCtrl* ctrl = reinterpret_cast<RfCtrl*>(smem);
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    const uint32_t rank = cluster_ctarank();
    const int cluster = (int)cluster_id_x();
    const uint32_t ring = smem_u32(smem + kRfCtrlBytes) + (uint32_t)warp * (kRfSlots * kRfSlotBytes);
    const uint32_t bar0 = smem_u32(&ctrl->full[warp * 8]);
    const uint32_t stage = smem_u32(smem + kRfCtrlBytes + RfShape<CL>::kRingBytes) +
                           (uint32_t)warp * RfShape<CL>::kStageBytes;

    // this warp's part of the row, in 16-byte units: [part0, part0 + part_units)
    const int part_idx = (int)rank * kRfWarps + warp;
    constexpr int nparts = kRfParts;
    const int part0 = (int)(((int64_t)p.units_per_row * part_idx) / nparts);
    const int part_units = (int)(((int64_t)p.units_per_row * (part_idx + 1)) / nparts) - part0;
    const int nch = (part_units + kRfChunkUnits - 1) / kRfChunkUnits;     // <= NCH

    const int my_rows = (int)((a.n_tok - cluster + p.num_clusters - 1) / p.num_clusters);
    const int total_seq = my_rows * nch;
    const bool backward = a.dlogits != nullptr;
    constexpr bool want_ent = ENT;        // token_entropy output (its own instantiation: the extra
                                          // accumulator must not cost the default path anything)
    const uint8_t* lbase = reinterpret_cast<const uint8_t*>(a.logits) + (int64_t)part0 * 16;
    uint8_t* gbase = reinterpret_cast<uint8_t*>(a.dlogits) + (int64_t)part0 * 16 + lane * 16;
    const int64_t row_bytes = a.ld * 2;

    if (lane == 0)
        for (int s = 0; s < kRfSlots; ++s) mbar_init(bar0 + 8u * s, 1);
    fence_mbar_init();
    __syncwarp();
    cluster_arrive();     // both CTAs are resident before any distributed-shared-memory store
    cluster_wait();

    // ---- TMA producer state (warp-uniform; lane 0 issues)
    int ld_seq = 0, ld_ch = 0, ld_slot = 0;
    int64_t ld_row = cluster;
    int cons_seq = 0, cons_slot = 0;
    uint32_t cons_phase = 0;
    auto refill = [&]() {
        while (ld_seq < total_seq && ld_seq < cons_seq + kRfSlots) {
            if (lane == 0) {
                const int u0 = ld_ch * kRfChunkUnits;
                const uint32_t bytes = (uint32_t)min(kRfChunkUnits, part_units - u0) * 16u;
                const uint32_t bar = bar0 + 8u * ld_slot;
                mbar_expect_tx(bar, bytes);
                bulk_load(ring + (uint32_t)ld_slot * kRfSlotBytes,
                          lbase + ld_row * row_bytes + (int64_t)u0 * 16, bytes, bar);
            }
            ++ld_seq;
            if (++ld_ch == nch) { ld_ch = 0; ld_row += p.num_clusters; }
            if (++ld_slot == kRfSlots) ld_slot = 0;
        }
    };
    refill();

    int y_next = -1, traj_next = -1;
    if (cluster < a.n_tok) { y_next = a.target_ids[cluster]; traj_next = a.tok_traj[cluster]; }
    int par = 0;
    uint32_t stage_par = 0;               // staging buffers handed to the TMA so far (parity = next buffer)
    for (int64_t row = cluster; row < a.n_tok; row += p.num_clusters, par ^= 1) {
        // ---- row header: every thread loads the same words (one sector each).  Only the raw
        // loads are issued here; nothing consumes them before the cluster barrier (the selects
        // and the bf16 widening sit after it), so their latency hides behind passes 0 and 1.
        RowHeader h;
        h.y = y_next;
        const int traj = traj_next;
        {
            const int64_t nrow = row + p.num_clusters;
            if (nrow < a.n_tok) { y_next = a.target_ids[nrow]; traj_next = a.tok_traj[nrow]; }
        }
        const bool valid = (h.y >= 0) && (h.y < a.V);
        const float q_raw = a.prox_lp[row];
        const float b_raw = a.behave_lp[row];
        float A_raw = 0.f, scale_raw = 0.f;
        if (traj >= 0) { A_raw = a.adv[traj]; scale_raw = a.traj_scale[traj]; }
        unsigned short zy_raw = 0;
        if (valid) zy_raw = reinterpret_cast<const unsigned short*>(a.logits)[row * a.ld + h.y];
        // The target entry is left out of the (max, sum) state (token_scalars works from
        // lse_rest): the warp whose part holds it masks it to -inf on the way to registers.
        const int y_unit = valid ? (h.y >> 3) - part0 : -1;
        const bool owner = (y_unit >= 0) && (y_unit < part_units);        // warp-uniform
        const int y_word = (h.y & 7) >> 1;
        const uint32_t y_keep = (h.y & 1) ? 0x0000ffffu : 0xffff0000u;     // the OTHER half

        // ---- pass 0: ring -> registers, packed running max
        uint32_t v[NU][4];
        uint32_t mx2 = kNegInf2;
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
            const bool have = c < nch;                                    // warp-uniform
            if (have) mbar_wait(bar0 + 8u * cons_slot, cons_phase);
            const uint32_t src = ring + (uint32_t)cons_slot * kRfSlotBytes + (uint32_t)lane * 16u;
#pragma unroll
            for (int kk = 0; kk < kRfChunkRounds; ++kk) {
                const int k = c * kRfChunkRounds + kk;
                if (k < NU) {
                    if (k < NU - 1 || k * 32 + lane < part_units) {
                        lds128(v[k], src + kk * (32 * 16));
                    } else {
                        v[k][0] = v[k][1] = v[k][2] = v[k][3] = kNegInf2;
                    }
                    if (owner && k * 32 + lane == y_unit) {
#pragma unroll
                        for (int j = 0; j < 4; ++j)
                            v[k][j] = (j == y_word) ? ((v[k][j] & y_keep) | (kNegInf2 & ~y_keep))
                                                    : v[k][j];
                    }
                    mx2 = max_bf16x2(mx2, max_bf16x2(max_bf16x2(v[k][0], v[k][1]),
                                                     max_bf16x2(v[k][2], v[k][3])));
                }
            }
            if (have) {
                // the max above consumed the loaded registers: the slot has been read out
                ++cons_seq;
                if (++cons_slot == kRfSlots) { cons_slot = 0; cons_phase ^= 1u; }
                __syncwarp();
                refill();
            }
        }
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
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(kFull, s, o);

        // ---- exchange: every warp of the cluster publishes (m_w, s_w) to both CTAs
        if (lane < CL) st_cluster_f32x2(smem_u32(&ctrl->stats[par][part_idx]), (uint32_t)lane, m, s);
        if (want_ent) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) accz += __shfl_xor_sync(kFull, accz, o);
            if (lane < CL) st_cluster_f32(smem_u32(&ctrl->statz[par][part_idx]), (uint32_t)lane, accz);
        }
        __syncwarp();
        cluster_arrive();
        cluster_wait();
        const float2 st = ctrl->stats[par][lane];
        float M = st.x;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(kFull, M, o));
        float S = (M == -INFINITY) ? 0.f : st.y * ex2_approx((st.x - M) * kLog2e);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) S += __shfl_xor_sync(kFull, S, o);
        const float lse_rest = M + fast_log(S);               // -inf if nothing but the target
        h.q = q_raw; h.b = b_raw; h.A = A_raw; h.scale = scale_raw;
        h.zy = __uint_as_float((uint32_t)zy_raw << 16);

        // ---- a3: per-token scalars (every thread, identical arithmetic)
        const TokenScalars ts = token_scalars(h, lse_rest, valid, a.clip_eps, a.stale_cap, a.dual_c);
        if (want_ent) {
            float SZ = (st.x == -INFINITY) ? 0.f : ctrl->statz[par][lane] * ex2_approx((st.x - M) * kLog2e);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) SZ += __shfl_xor_sync(kFull, SZ, o);
            if (tid == 0 && rank == 0)
                a.token_entropy[row] = valid ? row_entropy(ts.lse, M, SZ, ts.lp, h.zy) : 0.f;
        }
        if (tid == 0 && rank == 0) {
            if (h.y >= a.V) atomicOr(a.err_word, AWR_ERRBIT_TARGET_RANGE);
            store_token_outputs(a, row, h, ts, valid);
        }

        // ---- pass 2 (a4): dlogits = e * (c_t exp(m - lse)), straight from registers
        if (backward) {
            // e was taken relative to m (0 if the part held nothing finite); c_t = 0 (masked, zero
            // advantage, clip triggered): F = +0 and e >= 0 give all-bits-zero products
            const float F = ts.coef == 0.f ? 0.f : ts.coef * ex2_approx(fmaf(-ts.lse, kLog2e, -nref));
            const __nv_bfloat16 fh = __float2bfloat16_rn(F);
            const __nv_bfloat16 fl = __float2bfloat16_rn(F - __bfloat162float(fh));
            const uint32_t Fh = (uint32_t)__bfloat16_as_ushort(fh) * 0x00010001u;
            const uint32_t Fl = (uint32_t)__bfloat16_as_ushort(fl) * 0x00010001u;
            const uint32_t gy_bits = (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(ts.gy));
            const uint32_t gy2 = (h.y & 1) ? (gy_bits << 16) : gy_bits;
            const bool patch = owner && ts.coef != 0.f;
            if constexpr (RfShape<CL>::kStaged) {
                // The SM's path for per-lane global stores takes 32 B/clk: 148 KB of gradient per row
                // half held every warp ~5 k clocks in this pass.  Instead the warp writes its part to
                // a staging buffer in shared memory (128 B/clk) and lane 0 hands each buffer to a TMA
                // bulk store, which drains it to global memory while the warp is already in the next
                // row; the registers are free as soon as the shared-memory write has been issued.
                uint8_t* g = reinterpret_cast<uint8_t*>(a.dlogits) + (int64_t)part0 * 16 + row * row_bytes;
#pragma unroll
                for (int k = 0; k < NU; ++k) {
                    const int kk = k % kRfStageRounds;
                    const uint32_t buf = stage + (((uint32_t)(k / kRfStageRounds) + stage_par) & 1u) * (kRfStageRounds * 512);
                    if (kk == 0) {
                        // the bulk store issued two buffers ago has read this buffer out
                        if (lane == 0) bulk_wait_read<1>();
                        __syncwarp();
                    }
                    uint4 o;
                    o.x = fma_bf16x2(v[k][0], Fh, mul_bf16x2(v[k][0], Fl));
                    o.y = fma_bf16x2(v[k][1], Fh, mul_bf16x2(v[k][1], Fl));
                    o.z = fma_bf16x2(v[k][2], Fh, mul_bf16x2(v[k][2], Fl));
                    o.w = fma_bf16x2(v[k][3], Fh, mul_bf16x2(v[k][3], Fl));
                    if (patch && k * 32 + lane == y_unit) {     // target entry: c (p_y - 1)
                        o.x = y_word == 0 ? ((o.x & y_keep) | gy2) : o.x;
                        o.y = y_word == 1 ? ((o.y & y_keep) | gy2) : o.y;
                        o.z = y_word == 2 ? ((o.z & y_keep) | gy2) : o.z;
                        o.w = y_word == 3 ? ((o.w & y_keep) | gy2) : o.w;
                    }
                    sts128(buf + (uint32_t)kk * 512u + (uint32_t)lane * 16u, o);
                    if (kk == kRfStageRounds - 1 || k == NU - 1) {
                        const int k0 = k - kk;                                  // first round of the buffer
                        const int units = min(part_units, (k + 1) * 32) - k0 * 32;
                        fence_proxy_async();                                    // generic writes -> TMA read
                        __syncwarp();
                        if (lane == 0 && units > 0) {
                            bulk_store(g + (int64_t)k0 * 512, buf, (uint32_t)units * 16u);
                            bulk_commit();
                        }
                    }
                }
                // the two buffers alternate across rows as well (a row has an odd number of pieces
                // for most V): the next row starts with the buffer this row did not end on
                stage_par += (uint32_t)((NU + kRfStageRounds - 1) / kRfStageRounds);
            } else {
                uint8_t* g = gbase + row * row_bytes;
#pragma unroll
                for (int k = 0; k < NU; ++k) {
                    uint32_t o[4];
#pragma unroll
                    for (int j = 0; j < 4; ++j) o[j] = fma_bf16x2(v[k][j], Fh, mul_bf16x2(v[k][j], Fl));
                    if (patch && k * 32 + lane == y_unit) {     // target entry: c (p_y - 1)
#pragma unroll
                        for (int j = 0; j < 4; ++j)
                            o[j] = (j == y_word) ? ((o[j] & y_keep) | gy2) : o[j];
                    }
                    if (k < NU - 1 || k * 32 + lane < part_units)
                        stg128_cs(g + k * (32 * 16), o[0], o[1], o[2], o[3]);
                }
            }
        }
    }
    if (lane == 0) bulk_wait_all();       // staged gradient writes complete before the CTA ends
    cluster_arrive();
    cluster_wait();
}

// ---------------------------------------------------------------- host side
static bool make_rf_plan(int64_t V, int64_t ld, int dtype, RfPlan& p, int& nu) {
    if (dtype != AWR_DTYPE_BF16) return false;
    if (V % 8 != 0 || ld % 8 != 0) return false;
    const int64_t units = V / 8;
    const int64_t part_max = (units + kRfParts - 1) / kRfParts;
    const int64_t n = (part_max + 31) / 32;
    if (n < kRfMinNU || n > kRfMaxNU) return false;
    p.units_per_row = (int)units;
    p.num_clusters = 0;
    nu = (int)n;
    return true;
}

bool rows_rf_supported(int64_t V, int64_t ld, int dtype) {
    RfPlan p;
    int nu;
    return make_rf_plan(V, ld, dtype, p, nu);
}

template <int NU, int CL, bool ENT>
static cudaError_t launch_nu(const RowArgs& a, RfPlan p, int num_sms, cudaStream_t st) {
    using S = RfShape<CL>;
    static PerDeviceInt cached;              // co-resident clusters (device query, cached per device)
    const int dev = PerDeviceInt::device();
    int max_clusters = cached.get(dev);
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CL;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(S::kThreads, 1, 1);
    cfg.dynamicSmemBytes = S::kSmemBytes;
    cfg.stream = st;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (max_clusters < 0) {
        cudaError_t e = cudaFuncSetAttribute(rows_rf_kernel<NU, CL, ENT>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             S::kSmemBytes);
        if (e != cudaSuccess) return e;
        cfg.gridDim = dim3(CL * num_sms, 1, 1);
        int n = 0;
        e = cudaOccupancyMaxActiveClusters(&n, rows_rf_kernel<NU, CL, ENT>, &cfg);
        if (e != cudaSuccess) return e;
        const int want = num_sms * S::kCtasPerSm / CL;
        max_clusters = n < 1 ? 1 : (n > want ? want : n);
        cached.set(dev, max_clusters);
    }
    int nc = max_clusters;
    if ((int64_t)nc > a.n_tok) nc = (int)a.n_tok;
    p.num_clusters = nc;
    cfg.gridDim = dim3(CL * nc, 1, 1);
    return cudaLaunchKernelEx(&cfg, rows_rf_kernel<NU, CL, ENT>, a, p);
}

cudaError_t launch_rows_rf(const RowArgs& a, int num_sms, int cluster_size, cudaStream_t st) {
    if (a.n_tok <= 0) return cudaSuccess;
    RfPlan p;
    int nu = 0;
    if (!make_rf_plan(a.V, a.ld, AWR_DTYPE_BF16, p, nu)) return cudaErrorInvalidValue;
    if (cluster_size != 2 && cluster_size != 4) return cudaErrorInvalidValue;
    switch (nu) {
#define AWR_RF_CASE(N)                                                                   \
    case N:                                                                              \
        if (a.token_entropy != nullptr)                                                  \
            return cluster_size == 2 ? launch_nu<N, 2, true>(a, p, num_sms, st)          \
                                     : launch_nu<N, 4, true>(a, p, num_sms, st);         \
        return cluster_size == 2 ? launch_nu<N, 2, false>(a, p, num_sms, st)             \
                                 : launch_nu<N, 4, false>(a, p, num_sms, st);
        AWR_RF_CASE(3) AWR_RF_CASE(4) AWR_RF_CASE(5) AWR_RF_CASE(6) AWR_RF_CASE(7) AWR_RF_CASE(8)
        AWR_RF_CASE(9) AWR_RF_CASE(10) AWR_RF_CASE(11) AWR_RF_CASE(12) AWR_RF_CASE(13)
        AWR_RF_CASE(14) AWR_RF_CASE(15) AWR_RF_CASE(16) AWR_RF_CASE(17) AWR_RF_CASE(18)
        AWR_RF_CASE(19) AWR_RF_CASE(20)
#undef AWR_RF_CASE
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace awr
