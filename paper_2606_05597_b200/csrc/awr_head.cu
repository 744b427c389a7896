// a5: fused LM-head variant (BASELINE.json config 4, readings A17).
//
//   logits Z = H W_head are produced tile by tile in tensor memory; the full matrix never exists.
//   Per panel of P <= 9,472 rows, row-reference mode (AUTO; DESIGN.md section 5 for the others):
//     ref      zref_t = the row's largest logit among the first 256 vocabulary entries: one column
//              tile of the forward GEMM                                          (GEMM, kEpiRowMax)
//     pass F   Z tile -> per-row sum of e = exp(z - zref_t) + target gather, and E = bf16(e) into
//              the dS panel (2 bytes per logit of the panel, 2.9 GB at the default P), ONE pass over
//              the accumulator                                                  (GEMM, kEpiLseRef)
//     scalars  partials -> lse, l_t, ratio / clip / normalizer (a3), c_t; then f_t = c_t exp(zref_t -
//              lse), the target entry of E, and Hs = bf16(f_t h_t)                 (one warp per row)
//     fix-up   rows with a logit > 88 nats above zref_t (none on ordinary logits) redone exactly from
//              hidden and w_head on the CUDA cores                                  (one CTA per such row)
//     pass G2  dhidden[panel] = diag(f) (E W_head^T): row scale in the epilogue    (GEMM, kEpiStoreBf16)
//     pass G3  dw_head += Hs^T E   (fp32 running sum, bf16 at the end)             (GEMM, kEpiAccum)
//   so dS = diag(f) E is never formed.  E16 mode: E relative to the tile's row max (kEpiLse16, two
//   passes over the accumulator) and an in-place streaming pass E -> dS; stored mode: the fp32 tile is
//   kept instead (kEpiLse + head_ds_kernel on a side stream); the recompute modes form dS with a
//   second logits GEMM (kEpiDs).
// Every GEMM is the tcgen05 kernel below; see awr_head_gemm.cuh for the engine.
#include <mutex>

#include "awr_head_gemm.cuh"
#include "awr_kernels.h"

namespace awr {
namespace head {

__device__ __forceinline__ void tile_coords(const GemmArgs& g, int tile, int& m_blk, int& n_blk) {
    if (g.order == 0) {
        const int per_group = g.group_m * g.n_tiles;
        const int gi = tile / per_group;
        const int r = tile - gi * per_group;
        const int gm = min(g.group_m, g.m_tiles - gi * g.group_m);
        m_blk = gi * g.group_m + r % gm;
        n_blk = r / gm;
    } else {
        m_blk = tile / g.n_tiles;
        n_blk = tile - m_blk * g.n_tiles;
    }
}

template <int EPI, int CTAS, int NT>
__global__ void __launch_bounds__(kThreads, 1)
head_gemm_kernel(const __grid_constant__ CUtensorMap tmap_a,
                 const __grid_constant__ CUtensorMap tmap_b, const GemmArgs g) {
    using G = Geo<CTAS, NT>;
    constexpr int kTN = G::kTileN;
    constexpr int kStages = EpiGeo<EPI, CTAS, NT>::kStages;
    constexpr int kStageBytes = G::kStageBytes;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bars = smem_base + kStages * kStageBytes;
    // barrier words: full[kStages], empty[kStages], tmem_full[2], tmem_empty[2], tmem ptr
    auto full_bar = [&](int s) { return bars + 8u * s; };
    auto empty_bar = [&](int s) { return bars + 8u * (kStages + s); };
    auto tfull_bar = [&](int s) { return bars + 8u * (2 * kStages + s); };
    auto tempty_bar = [&](int s) { return bars + 8u * (2 * kStages + 2 + s); };
    const uint32_t tmem_slot = bars + 8u * (2 * kStages + 4);
    // staging tiles of the LSE epilogue (kEpiLse only), behind the 256-byte barrier block
    float* zstage = reinterpret_cast<float*>(smem_raw + (bars + 256u - smem_u32(smem_raw)));
    uint32_t* tmem_slot_ptr =
        reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int num_tiles = g.m_tiles * g.n_tiles;
    const int num_kb = (g.Kc + kBK - 1) / kBK;
    // CTAS = 2: both CTAs of a pair walk the same tile sequence; rank 0 is the leader
    const uint32_t rank = CTAS == 2 ? cluster_rank() : 0u;
    const int tile0 = CTAS == 2 ? (int)cluster_id() : (int)blockIdx.x;
    const int tile_step = CTAS == 2 ? (int)num_clusters() : (int)gridDim.x;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap_a) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap_b) : "memory");
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < kStages; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(tfull_bar(s), 1); mbar_init(tempty_bar(s), 4 * CTAS); }
        fence_mbar_init();
    }
    if (warp == 2) {
        if constexpr (CTAS == 1) {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot),
                         "n"(kTmemCols)
                         : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        } else {
            asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot),
                         "n"(kTmemCols)
                         : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
        }
    }
    tc_fence_before();
    if constexpr (CTAS == 2) cluster_sync_all(); else __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        // ===================== TMA producer (every CTA stages its own rows of A and columns of B)
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int tile = tile0; tile < num_tiles; tile += tile_step) {
                int m_blk, n_blk;
                tile_coords(g, tile, m_blk, n_blk);
                const int m0 = m_blk * G::kTileM + (int)rank * kBM;
                const int n0 = n_blk * kTN + (int)rank * G::kLoadN;
                for (int kb = 0; kb < num_kb; ++kb) {
                    mbar_wait(empty_bar(stage), phase ^ 1u);
                    const uint32_t sa = smem_base + stage * kStageBytes;
                    const uint32_t sb = sa + kABytes;
                    uint32_t bar = full_bar(stage);
                    if (rank == 0) mbar_expect_tx(bar, kStageBytes * CTAS);
                    if constexpr (CTAS == 2) bar = map_to_cta(bar, 0);
                    const int k0 = kb * kBK;
                    if (g.a.rank3) {
                        tma_load_3d<CTAS>(sa, &tmap_a, 0, k0, m0 >> 6, bar);
                    } else {
                        for (uint32_t j = 0; j < g.a.boxes; ++j) {
                            if (g.a.major == kMajorK) tma_load_2d<CTAS>(sa, &tmap_a, k0, m0, bar);
                            else tma_load_2d<CTAS>(sa + j * g.a.box_bytes, &tmap_a, m0 + 64 * (int)j, k0, bar);
                        }
                    }
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) {
                        const uint32_t sbn = sb + nt * G::kBBytes1;
                        const int nn = n0 + nt * kBN;
                        if (g.b.rank3) {
                            tma_load_3d<CTAS>(sbn, &tmap_b, 0, k0, nn >> 6, bar);
                        } else {
                            for (uint32_t j = 0; j < g.b.boxes; ++j) {
                                if (g.b.major == kMajorK) tma_load_2d<CTAS>(sbn, &tmap_b, k0, nn, bar);
                                else tma_load_2d<CTAS>(sbn + j * g.b.box_bytes, &tmap_b, nn + 64 * (int)j, k0, bar);
                            }
                        }
                    }
                    if (++stage == kStages) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (leader CTA only)
        if (lane == 0 && rank == 0) {
            int stage = 0;
            uint32_t phase = 0;
            int as = 0;
            uint32_t aphase = 0;
            for (int tile = tile0; tile < num_tiles; tile += tile_step) {
                mbar_wait(tempty_bar(as), aphase ^ 1u);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + (uint32_t)as * kBN;      // NT = 2: as is always 0
                for (int kb = 0; kb < num_kb; ++kb) {
                    mbar_wait(full_bar(stage), phase);
                    tc_fence_after();
                    const uint32_t sa = smem_base + stage * kStageBytes;
                    const uint32_t sb = sa + kABytes;
                    const uint32_t a_lo = ((sa >> 4) & 0x3fffu) | g.a.desc_lo;
                    const uint32_t b_lo = ((sb >> 4) & 0x3fffu) | g.b.desc_lo;
#pragma unroll
                    for (int k = 0; k < kBK / kUmmaK; ++k) {
                        const uint64_t adesc =
                            ((uint64_t)g.a.desc_hi << 32) | (uint64_t)(a_lo + k * g.a.k_step);
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) {
                            const uint64_t bdesc = ((uint64_t)g.b.desc_hi << 32) |
                                (uint64_t)(b_lo + nt * (G::kBBytes1 >> 4) + k * g.b.k_step);
                            tc_mma<CTAS>(d_tmem + nt * kBN, adesc, bdesc, g.idesc, (uint32_t)((kb | k) != 0));
                        }
                    }
                    tc_commit<CTAS>(empty_bar(stage));    // smem slot free once these MMAs retire
                    if (++stage == kStages) { stage = 0; phase ^= 1u; }
                }
                tc_commit<CTAS>(tfull_bar(as));           // accumulator tile complete
                if (++as == G::kAccStages) { as = 0; aphase ^= 1u; }
            }
        }
    } else if (warp >= 4) {
        // ===================== epilogue: one accumulator row per thread
        const int q = warp & 3;                           // TMEM lane quarter of this warp
        int as = 0;
        uint32_t aphase = 0;
        for (int tile = tile0; tile < num_tiles; tile += tile_step) {
            int m_blk, n_blk;
            tile_coords(g, tile, m_blk, n_blk);
            const int row = m_blk * G::kTileM + (int)rank * kBM + q * 32 + lane;
            const int n0 = n_blk * kTN;
            const bool row_ok = row < g.M;
            // kEpiAccum: the running fp32 sum of this thread's row is fetched one 32-column chunk
            // ahead (chunk 0 before the accumulator is even complete), so the global-memory
            // latency overlaps the MMAs / the previous chunk instead of serialising 8 round trips
            float4 pre[8];
            auto fetch_acc = [&](int c) {
                if constexpr (EPI == kEpiAccum) {
                    const int c0 = n0 + c * 32;
                    if (!g.e.first_panel && row_ok && c < kTN / 32) {
                        const float* ap = g.e.acc + (int64_t)row * g.e.out_ld + c0;
#pragma unroll
                        for (int j = 0; j < 8; ++j)
                            pre[j] = (c0 + 4 * j < g.N) ? __ldcs(reinterpret_cast<const float4*>(ap + 4 * j))
                                                        : make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                }
            };
            fetch_acc(0);
            mbar_wait(tfull_bar(as), aphase);
            tc_fence_after();
            const uint32_t t_addr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)as * kBN;
            float v[32];

            if constexpr (EPI == kEpiLse) {
                const int y = row_ok ? g.e.target_ids[row] : -1;
                float m = -INFINITY, s = 0.f, zy = 0.f, sz = 0.f;
                const bool want_ent = g.e.partz != nullptr;
                const bool y_here = (y >= n0) && (y < n0 + kTN) && (y < g.N);
                auto process = [&](int c, float (&v)[32]) {
                    const int c0 = n0 + c * 32;
                    if (g.e.zout != nullptr) {            // warp-uniform
                        // keep the fp32 logits of this row panel for the dS pass (no recompute):
                        // thread = row after the TMEM load; transposed through this warp's padded
                        // shared-memory tile so that every store instruction writes 4 whole
                        // 128-byte row segments instead of 16 bytes of 32 different rows
                        float* stg = zstage + q * (32 * kZStageLd);
#pragma unroll
                        for (int j = 0; j < 8; ++j)
                            *reinterpret_cast<float4*>(stg + lane * kZStageLd + 4 * j) =
                                make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
                        __syncwarp();
                        const int cc = (lane & 7) * 4;
                        const int row_w = row - lane;         // tile row of this warp's TMEM lane 0
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            const int r = i * 4 + (lane >> 3);
                            const float4 t = *reinterpret_cast<const float4*>(stg + r * kZStageLd + cc);
                            if (row_w + r < g.M && c0 + cc < g.N)
                                __stcs(reinterpret_cast<float4*>(g.e.zout + (int64_t)(row_w + r) * g.e.zout_ld + c0 + cc), t);
                        }
                        __syncwarp();
                    }
                    if (c0 + 32 > g.N) {
#pragma unroll
                        for (int j = 0; j < 32; ++j) if (c0 + j >= g.N) v[j] = -INFINITY;
                    }
                    if (y_here && y >= c0 && y < c0 + 32) {
                        // the target entry is gathered and left out of the (max, sum) state
#pragma unroll
                        for (int j = 0; j < 32; ++j) if (c0 + j == y) { zy = v[j]; v[j] = -INFINITY; }
                    }
                    float cm = v[0];
#pragma unroll
                    for (int j = 1; j < 32; ++j) cm = fmaxf(cm, v[j]);
                    const float mn = fmaxf(m, cm);
                    if (mn != -INFINITY) {
                        const float ref = mn * kLog2e;
                        const float resc = ex2_approx(fmaf(m, kLog2e, -ref));
                        float acc = 0.f;
                        if (want_ent) {
                            float accz = 0.f;
#pragma unroll
                            for (int j = 0; j < 32; ++j) {
                                const float e = ex2_approx(fmaf(v[j], kLog2e, -ref));
                                acc += e;
                                accz = fmaf(e, fmaxf(v[j], kZFloor), accz);
                            }
                            sz = sz * resc + accz;
                        } else {
#pragma unroll
                            for (int j = 0; j < 32; ++j) acc += ex2_approx(fmaf(v[j], kLog2e, -ref));
                        }
                        s = s * resc + acc;
                        m = mn;
                    }
                };
                // two register buffers: the TMEM load of chunk c + 1 is in flight while chunk c is
                // reduced (the exposed load latency was 30 % of the epilogue's stall samples)
                float vb[32];
                tmem_ld32_issue(t_addr, v);
#pragma unroll 1
                for (int c = 0; c < kTN / 32; c += 2) {
                    tmem_ld_wait(v);
                    tmem_ld32_issue(t_addr + (c + 1) * 32, vb);
                    process(c, v);
                    tmem_ld_wait(vb);
                    if (c + 2 < kTN / 32) tmem_ld32_issue(t_addr + (c + 2) * 32, v);
                    process(c + 1, vb);
                }
                if (row_ok) {
                    g.e.part[(int64_t)n_blk * g.e.part_ld + row] = make_float2(m, s);
                    if (want_ent) g.e.partz[(int64_t)n_blk * g.e.part_ld + row] = sz;
                    if (y_here) g.e.zy[row] = zy;
                }
            } else if constexpr (EPI == kEpiLse16) {
                // The tile is kept as E = bf16(exp(z - m)), m = this row's max over the tile (target
                // left out): 2 bytes per logit instead of 4, and the same exponentials feed the
                // log-sum-exp partial (unrounded).  Pass A takes the max, pass B the rest.
                const int y = row_ok ? g.e.target_ids[row] : -1;
                const bool want_ent = g.e.partz != nullptr;
                const bool y_here = (y >= n0) && (y < n0 + kTN) && (y < g.N);
                float m = -INFINITY, zy = 0.f;
                auto mask = [&](int c, float (&v)[32]) {      // columns >= N and the target -> -inf
                    const int c0 = n0 + c * 32;
                    if (c0 + 32 > g.N) {
#pragma unroll
                        for (int j = 0; j < 32; ++j) if (c0 + j >= g.N) v[j] = -INFINITY;
                    }
                    if (y_here && y >= c0 && y < c0 + 32) {
#pragma unroll
                        for (int j = 0; j < 32; ++j) if (c0 + j == y) { zy = v[j]; v[j] = -INFINITY; }
                    }
                };
                float vb[32];
                tmem_ld32_issue(t_addr, v);
#pragma unroll 1
                for (int c = 0; c < kTN / 32; c += 2) {
                    tmem_ld_wait(v);
                    tmem_ld32_issue(t_addr + (c + 1) * 32, vb);
                    mask(c, v);
#pragma unroll
                    for (int j = 0; j < 32; ++j) m = fmaxf(m, v[j]);
                    tmem_ld_wait(vb);
                    if (c + 2 < kTN / 32) tmem_ld32_issue(t_addr + (c + 2) * 32, v);
                    mask(c + 1, vb);
#pragma unroll
                    for (int j = 0; j < 32; ++j) m = fmaxf(m, vb[j]);
                }
                const float nref = (m == -INFINITY) ? 0.f : -m * kLog2e;
                float s = 0.f, sz = 0.f;
                uint32_t* stg = reinterpret_cast<uint32_t*>(zstage) + q * (32 * kZStageLd);
                const int row_w = row - lane;                 // tile row of this warp's TMEM lane 0
                auto expchunk = [&](int c, float (&v)[32], int half) {
                    mask(c, v);
                    float acc = 0.f, accz = 0.f;
#pragma unroll
                    for (int j = 0; j < 32; ++j) {
                        const float z = v[j];
                        v[j] = ex2_approx(fmaf(z, kLog2e, nref));
                        acc += v[j];
                        if (want_ent) accz = fmaf(v[j], fmaxf(z, kZFloor), accz);
                    }
                    s += acc;
                    sz += accz;
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        *reinterpret_cast<uint4*>(stg + lane * kZStageLd + half * 16 + 4 * j) = make_uint4(
                            pack_bf16x2(v[8 * j], v[8 * j + 1]), pack_bf16x2(v[8 * j + 2], v[8 * j + 3]),
                            pack_bf16x2(v[8 * j + 4], v[8 * j + 5]), pack_bf16x2(v[8 * j + 6], v[8 * j + 7]));
                };
                tmem_ld32_issue(t_addr, v);
#pragma unroll 1
                for (int c = 0; c < kTN / 32; c += 2) {
                    tmem_ld_wait(v);
                    tmem_ld32_issue(t_addr + (c + 1) * 32, vb);
                    expchunk(c, v, 0);
                    tmem_ld_wait(vb);
                    if (c + 2 < kTN / 32) tmem_ld32_issue(t_addr + (c + 2) * 32, v);
                    expchunk(c + 1, vb, 1);
                    __syncwarp();
                    // 64 columns of 32 rows are staged: every store instruction writes 4 whole
                    // 128-byte row segments
                    const int c0 = n0 + c * 32;
                    const int cc = (lane & 7) * 8;            // bf16 column inside the 64
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const int r = i * 4 + (lane >> 3);
                        const uint4 t = *reinterpret_cast<const uint4*>(stg + r * kZStageLd + (lane & 7) * 4);
                        if (row_w + r < g.M && c0 + cc < g.N)
                            *reinterpret_cast<uint4*>(g.e.eout + (int64_t)(row_w + r) * g.e.eout_ld + c0 + cc) = t;
                    }
                    __syncwarp();
                }
                if (row_ok) {
                    g.e.part[(int64_t)n_blk * g.e.part_ld + row] = make_float2(m, s);
                    if (want_ent) g.e.partz[(int64_t)n_blk * g.e.part_ld + row] = sz;
                    if (y_here) g.e.zy[row] = zy;
                }
            } else if constexpr (EPI == kEpiLseRef) {
                // The row's exp reference is known before the GEMM (zref: the largest of the row's
                // first 256 logits), so ONE pass over the accumulator gives both the sum and
                // E = bf16(exp(z - zref)).  The unrounded e feed the partial; an overflowing e (a logit
                // 88 nats above the reference) makes the sum +inf: head_scalars_kernel marks the row and
                // head_fix_rows_kernel redoes it; the stored E is clamped to a finite value meanwhile.
                const int y = row_ok ? g.e.target_ids[row] : -1;
                const bool want_ent = g.e.partz != nullptr;
                const bool y_here = (y >= n0) && (y < n0 + kTN) && (y < g.N);
                const float ref = row_ok ? g.e.zref[row] : 0.f;
                const float nref = -ref * kLog2e;
                float zy = 0.f, s = 0.f, sz = 0.f;
                uint32_t* stg = reinterpret_cast<uint32_t*>(zstage) + q * (32 * kZStageLd);
                const int row_w = row - lane;                 // tile row of this warp's TMEM lane 0
                auto expchunk = [&](int c, float (&v)[32], int half) {
                    const int c0 = n0 + c * 32;
                    if (c0 + 32 > g.N) {
#pragma unroll
                        for (int j = 0; j < 32; ++j) if (c0 + j >= g.N) v[j] = -INFINITY;
                    }
                    if (y_here && y >= c0 && y < c0 + 32) {
                        // the target entry is gathered and left out of the sum; its place in E is
                        // written by head_scalars_kernel
#pragma unroll
                        for (int j = 0; j < 32; ++j) if (c0 + j == y) { zy = v[j]; v[j] = -INFINITY; }
                    }
                    float acc0 = 0.f, acc1 = 0.f, accz = 0.f;
#pragma unroll
                    for (int j = 0; j < 32; j += 2) {
                        const float z0 = v[j], z1 = v[j + 1];
                        v[j] = ex2_approx(fmaf(z0, kLog2e, nref));
                        v[j + 1] = ex2_approx(fmaf(z1, kLog2e, nref));
                        acc0 += v[j];
                        acc1 += v[j + 1];
                        if (want_ent) {
                            accz = fmaf(v[j], fmaxf(z0, kZFloor), accz);
                            accz = fmaf(v[j + 1], fmaxf(z1, kZFloor), accz);
                        }
                    }
                    s += acc0 + acc1;
                    sz += accz;
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        *reinterpret_cast<uint4*>(stg + lane * kZStageLd + half * 16 + 4 * j) = make_uint4(
                            pack_bf16x2_sat(v[8 * j], v[8 * j + 1]), pack_bf16x2_sat(v[8 * j + 2], v[8 * j + 3]),
                            pack_bf16x2_sat(v[8 * j + 4], v[8 * j + 5]), pack_bf16x2_sat(v[8 * j + 6], v[8 * j + 7]));
                };
                float vb[32];
                tmem_ld32_issue(t_addr, v);
#pragma unroll 1
                for (int c = 0; c < kTN / 32; c += 2) {
                    tmem_ld_wait(v);
                    tmem_ld32_issue(t_addr + (c + 1) * 32, vb);
                    expchunk(c, v, 0);
                    tmem_ld_wait(vb);
                    if (c + 2 < kTN / 32) tmem_ld32_issue(t_addr + (c + 2) * 32, v);
                    expchunk(c + 1, vb, 1);
                    __syncwarp();
                    const int c0 = n0 + c * 32;
                    const int cc = (lane & 7) * 8;            // bf16 column inside the 64
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const int r = i * 4 + (lane >> 3);
                        const uint4 t = *reinterpret_cast<const uint4*>(stg + r * kZStageLd + (lane & 7) * 4);
                        if (row_w + r < g.M && c0 + cc < g.N)
                            *reinterpret_cast<uint4*>(g.e.eout + (int64_t)(row_w + r) * g.e.eout_ld + c0 + cc) = t;
                    }
                    __syncwarp();
                }
                if (row_ok) {
                    g.e.part[(int64_t)n_blk * g.e.part_ld + row] = make_float2(ref, s);
                    if (want_ent) g.e.partz[(int64_t)n_blk * g.e.part_ld + row] = sz;
                    if (y_here) g.e.zy[row] = zy;
                }
            } else if constexpr (EPI == kEpiRowMax) {
                float m = -INFINITY;
#pragma unroll 1
                for (int c = 0; c < kTN / 32; ++c) {
                    tmem_ld32(t_addr + c * 32, v);
                    const int c0 = n0 + c * 32;
#pragma unroll
                    for (int j = 0; j < 32; ++j) if (c0 + j < g.N) m = fmaxf(m, v[j]);
                }
                // a finite reference whatever the accumulators hold (NaN / inf logits: garbage in)
                if (row_ok) g.e.zref_out[row] = (fabsf(m) <= 3.0e38f) ? m : 0.f;
            } else if constexpr (EPI == kEpiDs) {
                int y = -1;
                float lse = 0.f, coef = 0.f, gy = 0.f;
                if (row_ok) {
                    y = g.e.target_ids[row]; lse = g.e.row_lse[row];
                    coef = g.e.row_coef[row]; gy = g.e.row_gy[row];
                }
                const float nref = -lse * kLog2e;
                __nv_bfloat16* dst = g.e.ds + (int64_t)row * g.e.ds_ld + n0;
#pragma unroll 1
                for (int c = 0; c < kTN / 32; ++c) {
                    tmem_ld32(t_addr + c * 32, v);
                    const int c0 = n0 + c * 32;
                    if (!row_ok || c0 >= g.N) continue;
                    uint32_t o[16];
                    if (coef == 0.f) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) o[j] = 0u;
                    } else {
#pragma unroll
                        for (int j = 0; j < 32; ++j) v[j] = coef * ex2_approx(fmaf(v[j], kLog2e, nref));
                        if (y >= c0 && y < c0 + 32) {
#pragma unroll
                            for (int j = 0; j < 32; ++j) if (c0 + j == y) v[j] = gy;
                        }
#pragma unroll
                        for (int j = 0; j < 16; ++j) o[j] = pack_bf16x2(v[2 * j], v[2 * j + 1]);
                    }
                    // ds_ld and N are multiples of 8: 16-byte stores, whole 8-column groups
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        if (c0 + 8 * j < g.N)
                            *reinterpret_cast<uint4*>(dst + c * 32 + 8 * j) =
                                make_uint4(o[4 * j], o[4 * j + 1], o[4 * j + 2], o[4 * j + 3]);
                }
            } else {
                const int64_t ro = (int64_t)row * g.e.out_ld + n0;
                float rs = 1.f;                               // kEpiStoreBf16: optional row scale
                if constexpr (EPI == kEpiStoreBf16) {
                    if (g.e.row_scale != nullptr && row_ok) rs = g.e.row_scale[row];
                }
#pragma unroll 1
                for (int c = 0; c < kTN / 32; ++c) {
                    tmem_ld32(t_addr + c * 32, v);
                    const int c0 = n0 + c * 32;
                    if (!row_ok || c0 >= g.N) continue;
                    bool to_bf16 = true;
                    if constexpr (EPI == kEpiStoreBf16) {
                        if (g.e.row_scale != nullptr) {       // warp-uniform
#pragma unroll
                            for (int j = 0; j < 32; ++j) v[j] = rs == 0.f ? 0.f : v[j] * rs;
                        }
                    }
                    if constexpr (EPI == kEpiAccum) {
                        float* ap = g.e.acc + ro + c * 32;
                        if (!g.e.first_panel) {
#pragma unroll
                            for (int j = 0; j < 8; ++j) {
                                v[4 * j] += pre[j].x; v[4 * j + 1] += pre[j].y;
                                v[4 * j + 2] += pre[j].z; v[4 * j + 3] += pre[j].w;
                            }
                            fetch_acc(c + 1);
                        }
                        to_bf16 = g.e.last_panel != 0;
                        if (!to_bf16) {
#pragma unroll
                            for (int j = 0; j < 8; ++j)
                                if (c0 + 4 * j < g.N)
                                    *reinterpret_cast<float4*>(ap + 4 * j) =
                                        make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
                        }
                    }
                    if (to_bf16) {
                        __nv_bfloat16* dst = g.e.out + ro + c * 32;
#pragma unroll
                        for (int j = 0; j < 4; ++j)
                            if (c0 + 8 * j < g.N)
                                *reinterpret_cast<uint4*>(dst + 8 * j) = make_uint4(
                                    pack_bf16x2(v[8 * j], v[8 * j + 1]), pack_bf16x2(v[8 * j + 2], v[8 * j + 3]),
                                    pack_bf16x2(v[8 * j + 4], v[8 * j + 5]), pack_bf16x2(v[8 * j + 6], v[8 * j + 7]));
                    }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
                // the accumulator buffer is released on the leader's barrier (the MMA issuer's)
                if constexpr (CTAS == 2) mbar_arrive_cluster(map_to_cta(tempty_bar(as), 0));
                else mbar_arrive(tempty_bar(as));
            }
            if (++as == G::kAccStages) { as = 0; aphase ^= 1u; }
        }
    }

    tc_fence_before();
    if constexpr (CTAS == 2) cluster_sync_all(); else __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        if constexpr (CTAS == 1)
            asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base),
                         "n"(kTmemCols)
                         : "memory");
        else
            asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base),
                         "n"(kTmemCols)
                         : "memory");
    }
}

}  // namespace head
}  // namespace awr

// ================================================================== scalars (a3 for the head path)
namespace awr {
namespace head {

// One warp per row: combine the per-column-tile (max, sum) partials into the log-sum-exp of
// the row without its target entry, then the same token_scalars() as the logits path.
//
// Row-reference mode (ref.zref != nullptr; the forward epilogue was kEpiLseRef, every partial is
// relative to zref[row]): dS = E f_row with f_row = c_t exp(zref - lse), so instead of a pass over
// the panel this warp writes f_row (the dhidden GEMM scales its output rows by it), the row of
// Hs = bf16(f_row H) (the A operand of the dw_head GEMM) and ONE element of E: the target entry,
// (p_y - 1) exp(lse - zref), so that E f_row = c_t (p_y - 1) there.  A row whose sum overflowed
// (a logit 88 nats above the reference) is marked in `fix` and written as a row that contributes
// nothing; head_fix_rows_kernel then redoes exactly that row from hidden and w_head.
struct HeadRefArgs {
    const float* zref;            // [n_tok] or nullptr
    float* row_f;                 // [n_tok]
    __nv_bfloat16* e;             // E panel, row 0 = token row0
    int64_t e_ld;
    const __nv_bfloat16* hidden;  // [n_tok, K]
    __nv_bfloat16* hs;            // [panel rows, K], row 0 = token row0
    int64_t K;
    uint8_t* fix;                 // [n_tok] 1 = the row's sum overflowed relative to zref
};

__global__ void __launch_bounds__(256)
head_scalars_kernel(RowArgs a, const float2* __restrict__ part, int64_t part_ld, int n_tiles,
                    const float* __restrict__ partz, const float* __restrict__ zy,
                    float* __restrict__ row_lse,
                    float* __restrict__ row_coef, float* __restrict__ row_gy, int64_t row0,
                    int64_t row1, HeadRefArgs ref) {
    const int lane = threadIdx.x & 31;
    const int64_t row = row0 + (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= row1) return;
    MaxSum st{-INFINITY, 0.f};
    for (int j = lane; j < n_tiles; j += 32) {
        const float2 p = part[(int64_t)j * part_ld + row];
        st = combine(st, MaxSum{p.x, p.y});
    }
    st = warp_combine(st);
    float sz = 0.f;
    if (partz != nullptr) {                      // entropy: sum e^{z - M} z over the tiles
        for (int j = lane; j < n_tiles; j += 32) {
            const float2 p = part[(int64_t)j * part_ld + row];
            if (p.x != -INFINITY) sz += partz[(int64_t)j * part_ld + row] * ex2_approx((p.x - st.m) * kLog2e);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) sz += __shfl_xor_sync(kFull, sz, o);
    }

    const float lse_rest = st.m + logf(st.s);          // -inf when nothing but the target
    RowHeader h;
    h.y = a.target_ids[row];
    bool valid = (h.y >= 0) && (h.y < a.V);
    const bool overflow = ref.zref != nullptr && valid && !(st.s <= 3.0e38f);
    if (overflow) valid = false;
    const int traj = a.tok_traj[row];
    h.q = a.prox_lp[row];
    h.b = a.behave_lp[row];
    h.A = traj >= 0 ? a.adv[traj] : 0.f;
    h.scale = traj >= 0 ? a.traj_scale[traj] : 0.f;
    h.zy = valid ? zy[row] : 0.f;
    const TokenScalars ts = token_scalars(h, lse_rest, valid, a.clip_eps, a.stale_cap, a.dual_c);
    if (lane == 0) {
        if (h.y >= a.V) atomicOr(a.err_word, AWR_ERRBIT_TARGET_RANGE);
        store_token_outputs(a, row, h, ts, valid);
        if (a.token_entropy) a.token_entropy[row] = valid ? row_entropy(ts.lse, st.m, sz, ts.lp, h.zy) : 0.f;
        row_lse[row] = ts.lse;
        row_coef[row] = ts.coef;
        row_gy[row] = ts.gy;
    }
    if (ref.zref != nullptr) {
        const float zr = ref.zref[row];
        const float f = ts.coef == 0.f ? 0.f : ts.coef * ex2_approx((zr - ts.lse) * kLog2e);
        if (lane == 0) {
            ref.row_f[row] = f;
            ref.fix[row] = overflow ? 1 : 0;
            if (f != 0.f) {
                const float ty = (ts.gy / ts.coef) * ex2_approx((ts.lse - zr) * kLog2e);
                ref.e[(row - row0) * ref.e_ld + h.y] = __float2bfloat16_rn(fmaxf(ty, -3.0e38f));
            }
        }
        const uint4* src = reinterpret_cast<const uint4*>(ref.hidden + row * ref.K);
        uint4* dst = reinterpret_cast<uint4*>(ref.hs + (row - row0) * ref.K);
        for (int u = lane; u < (int)(ref.K >> 3); u += 32) {
            uint4 o = make_uint4(0u, 0u, 0u, 0u);
            if (f != 0.f) {
                const uint4 x = src[u];
                o.x = pack_bf16x2(bf16_lo(x.x) * f, bf16_hi(x.x) * f);
                o.y = pack_bf16x2(bf16_lo(x.y) * f, bf16_hi(x.y) * f);
                o.z = pack_bf16x2(bf16_lo(x.z) * f, bf16_hi(x.z) * f);
                o.w = pack_bf16x2(bf16_lo(x.w) * f, bf16_hi(x.w) * f);
            }
            dst[u] = o;
        }
    }
}

// Row-reference mode, the rows head_scalars_kernel marked in `fix` (some logit more than ~88 nats
// above the row's reference: exp(z - zref) overflowed).  Such a row is redone here from scratch, one
// CTA per row, on the CUDA cores: logits by plain fp32 dot products of hidden_t with the columns of
// w_head, an online (max, sum[, sum e z]) over them (target left out), a3, then E relative to the
// row's TRUE maximum, f_t, Hs and the per-token outputs - everything the forward GEMM and
// head_scalars_kernel would have written.  Two passes over the dot products (~2 ms per row): the
// path exists so that the mode is exact for every finite input, not to be fast; on ordinary
// logits no row is marked and every CTA leaves after one byte load per row.
struct Triple { float m, s, sz; };
__device__ __forceinline__ Triple combine3(Triple a, Triple b) {
    const float M = fmaxf(a.m, b.m);
    if (M == -INFINITY) return Triple{M, 0.f, 0.f};
    const float fa = ex2_approx((a.m - M) * kLog2e), fb = ex2_approx((b.m - M) * kLog2e);
    return Triple{M, a.s * fa + b.s * fb, a.sz * fa + b.sz * fb};
}

__global__ void __launch_bounds__(512)
head_fix_rows_kernel(RowArgs a, HeadRefArgs ref, const __nv_bfloat16* __restrict__ w_head, int kv_layout,
                     float* __restrict__ row_lse, float* __restrict__ row_coef, float* __restrict__ row_gy,
                     int64_t row0, int64_t row1) {
    __shared__ Triple wstate[16];
    __shared__ float sh[6];                       // zy, ref, f, target entry of E, -, -
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t V = a.V, K = ref.K;
    for (int64_t row = row0 + blockIdx.x; row < row1; row += gridDim.x) {
        if (!ref.fix[row]) continue;              // the same byte for the whole CTA
        const int y = a.target_ids[row];          // valid: only valid rows are marked
        const __nv_bfloat16* hr = ref.hidden + row * K;
        auto logit = [&](int64_t v) {
            float acc = 0.f;
            if (kv_layout) {
                const __nv_bfloat16* wc = w_head + v;
                for (int64_t k = 0; k < K; ++k)
                    acc = fmaf(__bfloat162float(hr[k]), __bfloat162float(wc[k * V]), acc);
            } else {
                const __nv_bfloat16* wr = w_head + v * K;
                for (int64_t k = 0; k < K; ++k)
                    acc = fmaf(__bfloat162float(hr[k]), __bfloat162float(wr[k]), acc);
            }
            return acc;
        };
        // ---- pass 1: online (max, sum, sum e z) of the row without its target; the target's logit
        Triple t{-INFINITY, 0.f, 0.f};
        for (int64_t v = tid; v < V; v += blockDim.x) {
            const float z = logit(v);
            if (v == y) { sh[0] = z; continue; }
            t = combine3(t, Triple{z, 1.f, fmaxf(z, kZFloor)});
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1)
            t = combine3(t, Triple{__shfl_xor_sync(kFull, t.m, o), __shfl_xor_sync(kFull, t.s, o),
                                   __shfl_xor_sync(kFull, t.sz, o)});
        if (lane == 0) wstate[warp] = t;
        __syncthreads();
        if (tid == 0) {
            Triple r = wstate[0];
            for (int i = 1; i < (int)(blockDim.x >> 5); ++i) r = combine3(r, wstate[i]);
            RowHeader h;
            h.y = y;
            const int traj = a.tok_traj[row];
            h.q = a.prox_lp[row];
            h.b = a.behave_lp[row];
            h.A = traj >= 0 ? a.adv[traj] : 0.f;
            h.scale = traj >= 0 ? a.traj_scale[traj] : 0.f;
            h.zy = sh[0];
            const float lse_rest = r.m + logf(r.s);                   // -inf when nothing but the target
            const TokenScalars ts = token_scalars(h, lse_rest, true, a.clip_eps, a.stale_cap, a.dual_c);
            store_token_outputs(a, row, h, ts, true);
            if (a.token_entropy) a.token_entropy[row] = row_entropy(ts.lse, r.m, r.sz, ts.lp, h.zy);
            row_lse[row] = ts.lse;
            row_coef[row] = ts.coef;
            row_gy[row] = ts.gy;
            const float zr = fmaxf(r.m, h.zy);                        // every e <= 1 relative to it
            const float f = ts.coef == 0.f ? 0.f : ts.coef * ex2_approx((zr - ts.lse) * kLog2e);
            sh[1] = zr;
            sh[2] = f;
            sh[3] = f != 0.f ? (ts.gy / ts.coef) * ex2_approx((ts.lse - zr) * kLog2e) : 0.f;
            ref.row_f[row] = f;
            ref.fix[row] = 0;
        }
        __syncthreads();
        // ---- pass 2: E relative to the row's maximum, the target entry, Hs
        const float nref = -sh[1] * kLog2e, f = sh[2], ty = sh[3];
        __nv_bfloat16* er = ref.e + (row - row0) * ref.e_ld;
        for (int64_t v = tid; v < V; v += blockDim.x)
            er[v] = __float2bfloat16_rn(v == y ? ty : ex2_approx(fmaf(logit(v), kLog2e, nref)));
        __nv_bfloat16* hsr = ref.hs + (row - row0) * K;
        for (int64_t k = tid; k < K; k += blockDim.x)
            hsr[k] = __float2bfloat16_rn(f * __bfloat162float(hr[k]));
        __syncthreads();                                              // sh / wstate are reused by the next row
    }
}

// a4 for the stored-logits mode: dS = c_t (exp(z - lse) - onehot) from the fp32 logits panel the
// forward GEMM kept, rounded to bf16.  The same arithmetic, instruction for instruction, as the
// kEpiDs epilogue of the recompute mode, so both modes produce the same bits.  HBM-bound:
// 4 B read + 2 B written per element; rows with c_t = 0 are written as zeros without a read.
__global__ void __launch_bounds__(512)
head_ds_kernel(const float* __restrict__ z, int64_t z_ld, int64_t rows, int64_t V,
               const int32_t* __restrict__ target_ids, const float* __restrict__ row_lse,
               const float* __restrict__ row_coef, const float* __restrict__ row_gy,
               __nv_bfloat16* __restrict__ ds, int64_t ds_ld) {
    const int nq = (int)(V >> 2);                       // V is a multiple of 8
    for (int64_t row = blockIdx.x; row < rows; row += gridDim.x) {
        const float coef = row_coef[row];
        uint2* dst = reinterpret_cast<uint2*>(ds + row * ds_ld);
        if (coef == 0.f) {
            for (int i = threadIdx.x; i < nq; i += blockDim.x) dst[i] = make_uint2(0u, 0u);
            continue;
        }
        const int y = target_ids[row];
        const float gy = row_gy[row];
        const float nref = -row_lse[row] * kLog2e;
        const float4* src = reinterpret_cast<const float4*>(z + row * z_ld);
#pragma unroll 4
        for (int i = threadIdx.x; i < nq; i += blockDim.x) {
            const float4 a = __ldcs(src + i);
            float v0 = coef * ex2_approx(fmaf(a.x, kLog2e, nref));
            float v1 = coef * ex2_approx(fmaf(a.y, kLog2e, nref));
            float v2 = coef * ex2_approx(fmaf(a.z, kLog2e, nref));
            float v3 = coef * ex2_approx(fmaf(a.w, kLog2e, nref));
            if ((y >> 2) == i) {
                const int w = y & 3;
                v0 = w == 0 ? gy : v0; v1 = w == 1 ? gy : v1;
                v2 = w == 2 ? gy : v2; v3 = w == 3 ? gy : v3;
            }
            dst[i] = make_uint2(pack_bf16x2(v0, v1), pack_bf16x2(v2, v3));
        }
    }
}

// a4 for the E16 mode: the panel holds E = bf16(exp(z - m_j)), m_j the row's max over column tile
// j (the .x of the forward partials).  In place: dS = bf16(E c_t exp(m_j - lse)); the target entry
// becomes c_t (p_y - 1); rows with c_t = 0 are written as zeros without a read.  HBM-bound:
// 2 B read + 2 B written per element.
__global__ void __launch_bounds__(512)
head_ds16_kernel(__nv_bfloat16* __restrict__ e, int64_t ld, int64_t rows, int64_t V,
                 const int32_t* __restrict__ target_ids, const float2* __restrict__ part,
                 int64_t part_ld, const float* __restrict__ row_lse, const float* __restrict__ row_coef,
                 const float* __restrict__ row_gy) {
    const int units = (int)(V >> 3);                    // V is a multiple of 8
    constexpr int kUnitsPerTile = kBN / 8;
    for (int64_t row = blockIdx.x; row < rows; row += gridDim.x) {
        const float coef = row_coef[row];
        uint4* p = reinterpret_cast<uint4*>(e + row * ld);
        if (coef == 0.f) {
            for (int i = threadIdx.x; i < units; i += blockDim.x) p[i] = make_uint4(0u, 0u, 0u, 0u);
            continue;
        }
        const int y = target_ids[row];
        const float gy = row_gy[row];
        const float nlse = -row_lse[row] * kLog2e;
#pragma unroll 4
        for (int i = threadIdx.x; i < units; i += blockDim.x) {
            const float mj = part[(int64_t)(i / kUnitsPerTile) * part_ld + row].x;
            const float gj = (mj == -INFINITY) ? 0.f : coef * ex2_approx(fmaf(mj, kLog2e, nlse));
            const uint4 a = p[i];
            float v[8] = {bf16_lo(a.x), bf16_hi(a.x), bf16_lo(a.y), bf16_hi(a.y),
                          bf16_lo(a.z), bf16_hi(a.z), bf16_lo(a.w), bf16_hi(a.w)};
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] *= gj;
            if ((y >> 3) == i && y >= 0) {
#pragma unroll
                for (int k = 0; k < 8; ++k) v[k] = (k == (y & 7)) ? gy : v[k];
            }
            p[i] = make_uint4(pack_bf16x2(v[0], v[1]), pack_bf16x2(v[2], v[3]),
                              pack_bf16x2(v[4], v[5]), pack_bf16x2(v[6], v[7]));
        }
    }
}

// ================================================================== host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// A bf16 matrix as the GEMM sees one operand: `mn` rows or columns of the product, `kc`
// contraction length, element (i_mn, i_k) at base[i_mn * s_mn + i_k * s_k] with one of the two
// strides equal to 1.
struct OperandView {
    const void* base;
    int64_t mn, kc;
    int64_t ld;        // the non-unit stride, in elements
    int major;         // kMajorK: i_k contiguous; kMajorMN: i_mn contiguous
};

static bool make_operand(const OperandView& v, int tile_mn, CUtensorMap* map, Operand* op) {
    EncodeTiledFn enc = encode_fn();
    if (!enc) return false;
    cuuint64_t dims[3], strides[2];
    cuuint32_t box[3], estr[3] = {1, 1, 1};
    cuuint32_t rank = 2;
    strides[0] = (cuuint64_t)v.ld * 2;
    op->rank3 = 0;
    if (v.major == kMajorK) {
        dims[0] = (cuuint64_t)v.kc; dims[1] = (cuuint64_t)v.mn;
        box[0] = kBK; box[1] = (cuuint32_t)tile_mn;
        op->boxes = 1; op->box_bytes = (uint32_t)tile_mn * kBK * 2;
        op->desc_lo = 1u << 16;                       // leading byte offset: unused with swizzle
        op->k_step = (kUmmaK * 2) >> 4;               // 32 bytes inside the 128-byte row
    } else {
        dims[0] = (cuuint64_t)v.mn; dims[1] = (cuuint64_t)v.kc;
        box[0] = 64; box[1] = kBK;
        op->boxes = (uint32_t)tile_mn / 64; op->box_bytes = 64 * kBK * 2;
        op->desc_lo = (uint32_t)(op->box_bytes >> 4) << 16;   // next 64-wide MN chunk
        op->k_step = (kUmmaK * 128) >> 4;             // 16 contraction rows of 128 bytes
        if (v.mn % 64 == 0) {
            // the same bytes as a rank-3 tensor [mn / 64][kc][64]: one copy per stage fills all the
            // 64-wide chunks (shared-memory order chunk, k, 64 = the layout described above)
            rank = 3;
            op->rank3 = 1;
            dims[0] = 64; dims[1] = (cuuint64_t)v.kc; dims[2] = (cuuint64_t)(v.mn / 64);
            strides[0] = (cuuint64_t)v.ld * 2; strides[1] = 128;
            box[0] = 64; box[1] = kBK; box[2] = (cuuint32_t)tile_mn / 64;
        }
    }
    op->major = (uint32_t)v.major;
    op->desc_hi = (1024u >> 4) | (1u << 14) | (2u << 29);     // SBO 1024 B, version 1, SWIZZLE_128B
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, rank, const_cast<void*>(v.base), dims,
                     strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

template <int EPI, int CTAS, int NT>
static cudaError_t launch_gemm_epi(const CUtensorMap& ta, const CUtensorMap& tb, const GemmArgs& g,
                                   int grid, cudaStream_t st) {
    static PerDeviceInt attr_set;                    // the attribute is per device
    const int dev = PerDeviceInt::device();
    if (attr_set.get(dev) < 0) {
        cudaError_t e = cudaFuncSetAttribute(head_gemm_kernel<EPI, CTAS, NT>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             EpiGeo<EPI, CTAS, NT>::kSmemBytes);
        if (e != cudaSuccess) return e;
        attr_set.set(dev, 1);
    }
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CTAS;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(kThreads, 1, 1);
    cfg.dynamicSmemBytes = EpiGeo<EPI, CTAS, NT>::kSmemBytes;
    cfg.stream = st;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, head_gemm_kernel<EPI, CTAS, NT>, ta, tb, g);
}

// C[M, N] = A * B with epilogue `epi`; `order` / `group_m` pick the tile raster (group_m in row
// tiles of 128 * ctas rows); ctas = 1: one CTA per tile, 2: a CTA pair per 256-row tile.
static cudaError_t launch_gemm(int epi, const OperandView& A, const OperandView& B, int order,
                               int group_m, const EpiArgs& e, int num_sms, int ctas, cudaStream_t st,
                               bool wide = false) {
    if (A.mn <= 0 || B.mn <= 0 || A.kc <= 0) return cudaSuccess;
    // wide: 256 x 512 tiles (kEpiStoreBf16 on CTA pairs, N a multiple of 512)
    const int nt = (wide && ctas == 2 && epi == kEpiStoreBf16 && B.mn % (2 * kBN) == 0) ? 2 : 1;
    if (A.kc != B.kc) return cudaErrorInvalidValue;
    CUtensorMap ta, tb;
    GemmArgs g;
    if (!make_operand(A, kBM, &ta, &g.a) || !make_operand(B, kBN / ctas, &tb, &g.b)) return cudaErrorInvalidValue;
    const int tile_m = kBM * ctas;
    g.M = (int32_t)A.mn; g.N = (int32_t)B.mn; g.Kc = (int32_t)A.kc;
    g.m_tiles = (g.M + tile_m - 1) / tile_m;
    g.n_tiles = (g.N + kBN * nt - 1) / (kBN * nt);
    g.order = order; g.group_m = group_m < 1 ? 1 : group_m;
    g.idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)A.major << 15) |
              ((uint32_t)B.major << 16) | ((uint32_t)(kBN >> 3) << 17) | ((uint32_t)(tile_m >> 4) << 24);
    g.e = e;
    const int64_t tiles = (int64_t)g.m_tiles * g.n_tiles;
    const int slots = num_sms / ctas;                    // persistent CTAs / CTA pairs
    const int grid = (int)(tiles < slots ? tiles : slots) * ctas;
#define AWR_HEAD_CASE(E)                                                            \
    case E:                                                                         \
        return ctas == 2 ? launch_gemm_epi<E, 2, 1>(ta, tb, g, grid, st)            \
                         : launch_gemm_epi<E, 1, 1>(ta, tb, g, grid, st);
    if (nt == 2) return launch_gemm_epi<kEpiStoreBf16, 2, 2>(ta, tb, g, grid, st);
    switch (epi) {
        AWR_HEAD_CASE(kEpiLse) AWR_HEAD_CASE(kEpiDs) AWR_HEAD_CASE(kEpiStoreBf16) AWR_HEAD_CASE(kEpiAccum)
        AWR_HEAD_CASE(kEpiLse16) AWR_HEAD_CASE(kEpiLseRef) AWR_HEAD_CASE(kEpiRowMax)
        default: return cudaErrorInvalidValue;
    }
#undef AWR_HEAD_CASE
}

}  // namespace head
}  // namespace awr

// ================================================================== the a5 pass sequence
namespace awr {

using namespace head;

static inline size_t up256(size_t x) { return (x + 255) / 256 * 256; }

// Stored-logits mode: the dS pass of a row panel runs on a library-owned side stream beside the
// forward GEMM of the next panel.  Side streams (each with its fork / join event pair) live in a
// small per-device pool KEYED BY THE CALLER'S STREAM: calls on different user streams - from
// different host threads, or one of them inside a CUDA-graph capture - never share a side stream
// or an event, so one call's fork record cannot be overtaken by another's.  An entry is pinned
// (refcount) while a call is enqueuing with it; an unpinned entry whose side stream is not part
// of an ongoing capture may be handed to another user stream (least recently used first).  If
// every entry is busy the call runs its dS pass on the caller's stream (no overlap, same result).
struct SideStream {
    cudaStream_t user;
    cudaStream_t stream;
    cudaEvent_t fork, join;
    bool ok;
    int pinned;
    uint64_t last_use;
};
constexpr int kSidePerDevice = 8;
struct SidePool {
    std::mutex mu;
    SideStream e[kMaxDevices][kSidePerDevice] = {};
    uint64_t tick = 0;
};
static SidePool& side_pool() {
    static SidePool pool;
    return pool;
}
static SideStream* side_acquire(cudaStream_t user) {
    const int dev = PerDeviceInt::device();
    if (dev < 0) return nullptr;
    SidePool& pool = side_pool();
    std::lock_guard<std::mutex> lock(pool.mu);
    SideStream* row = pool.e[dev];
    SideStream* pick = nullptr;
    for (int i = 0; i < kSidePerDevice && !pick; ++i)
        if (row[i].ok && row[i].user == user) pick = &row[i];
    for (int i = 0; i < kSidePerDevice && !pick; ++i) {
        if (row[i].ok) continue;
        SideStream& s = row[i];
        if (cudaStreamCreateWithFlags(&s.stream, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&s.fork, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&s.join, cudaEventDisableTiming) != cudaSuccess) {
            cudaGetLastError();
            return nullptr;
        }
        s.ok = true; s.pinned = 0;
        pick = &s;
    }
    if (!pick) {                         // re-key the least recently used idle entry
        for (int i = 0; i < kSidePerDevice; ++i) {
            SideStream& s = row[i];
            if (s.pinned > 0 || (pick && s.last_use >= pick->last_use)) continue;
            cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
            if (cudaStreamIsCapturing(s.stream, &cs) != cudaSuccess) { cudaGetLastError(); continue; }
            if (cs == cudaStreamCaptureStatusNone) pick = &s;
        }
    }
    if (!pick) return nullptr;
    pick->user = user;
    pick->pinned += 1;
    pick->last_use = ++pool.tick;
    return pick;
}
static void side_release(SideStream* s) {
    if (!s) return;
    std::lock_guard<std::mutex> lock(side_pool().mu);
    s->pinned -= 1;
}
struct SideGuard {
    SideStream* s;
    ~SideGuard() { side_release(s); }
};

struct HeadWs {
    float *zy, *row_lse, *row_coef, *row_gy;
    float2* part;
    float* partz;            // entropy output only
    __nv_bfloat16* ds;
    float* dw_acc;
    float* zpanel;           // stored-logits mode: fp32 [panel_rows, z_ld]
    float* zpanel2;          // second buffer: the forward of panel p + 1 runs beside the dS pass of p
    float *zref, *row_f;     // row-reference mode: exp reference and dS scale of every row
    uint8_t* fix;            // row-reference mode: rows to be redone by head_fix_rows_kernel
    __nv_bfloat16* hs;       // row-reference mode: bf16(f_row H) of the panel [panel_rows, K]
    int64_t part_ld, ds_ld, z_ld, panel_rows;
    int n_vtiles, n_panels;
    size_t total;
};

// Rows per panel: the dhidden GEMM of a panel has (rows / tile rows) x (K / 256) tiles of V-long
// contractions, so the panel is sized to fill whole waves of the persistent grid at K = 2048:
// 37 x 8 = 296 tiles = 2 x 148 CTAs (ctas = 1) or 4 x 74 CTA pairs (ctas = 2).
static int64_t head_panel_rows(int ctas) { return ctas == 2 ? 2 * kHeadPanelRows : kHeadPanelRows; }

static HeadWs head_carve(void* base, int64_t n_tok, int64_t V, int64_t K, int ctas, int mode,
                         bool entropy = true) {
    const bool store_z = mode == kHeadStored32;
    HeadWs w;
    uint8_t* p = reinterpret_cast<uint8_t*>(base);
    size_t off = 0;
    auto take = [&](size_t bytes) { void* r = p + off; off += up256(bytes); return r; };
    const int64_t n_pad = (n_tok + kBM - 1) / kBM * kBM;
    w.part_ld = n_pad;
    w.ds_ld = (V + 7) / 8 * 8;
    w.n_vtiles = (int)((V + kBN - 1) / kBN);
    w.panel_rows = n_pad < head_panel_rows(ctas) ? n_pad : head_panel_rows(ctas);
    w.n_panels = n_tok > 0 ? (int)((n_tok + w.panel_rows - 1) / w.panel_rows) : 0;
    w.zy = (float*)take((size_t)n_pad * 4);
    w.row_lse = (float*)take((size_t)n_pad * 4);
    w.row_coef = (float*)take((size_t)n_pad * 4);
    w.row_gy = (float*)take((size_t)n_pad * 4);
    w.part = (float2*)take((size_t)w.n_vtiles * n_pad * 8);
    w.partz = (float*)take(entropy ? (size_t)w.n_vtiles * n_pad * 4 : 0);
    w.ds = (__nv_bfloat16*)take((size_t)w.panel_rows * w.ds_ld * 2);
    w.dw_acc = (float*)take(w.n_panels > 1 ? (size_t)K * V * 4 : 0);
    w.z_ld = w.ds_ld;
    w.zpanel = (float*)take(store_z ? (size_t)w.panel_rows * w.z_ld * 4 : 0);
    w.zpanel2 = (float*)take(store_z && w.n_panels > 1 ? (size_t)w.panel_rows * w.z_ld * 4 : 0);
    const bool rowref = mode == kHeadRowRef;
    w.zref = (float*)take(rowref ? (size_t)n_pad * 4 : 0);
    w.row_f = (float*)take(rowref ? (size_t)n_pad * 4 : 0);
    w.fix = (uint8_t*)take(rowref ? (size_t)n_pad : 0);
    w.hs = (__nv_bfloat16*)take(rowref ? (size_t)w.panel_rows * K * 2 : 0);
    w.total = off;
    return w;
}

size_t head_ws_bytes(int64_t n_tok, int64_t V, int64_t K, int ctas, int mode) {
    return head_carve(nullptr, n_tok, V, K, ctas == 1 ? 1 : 2, mode).total;
}

cudaError_t launch_head(const HeadCall& c, int num_sms, cudaStream_t st) {
    if (c.n_tok <= 0) {
        // no rows: the gradient of the head is zero
        return cudaMemsetAsync(c.dw_head, 0, (size_t)c.K * c.V * 2, st);
    }
    const int ctas = c.ctas == 1 ? 1 : 2;
    const int gm = 4096 / (kBM * ctas);               // raster groups of 4096 rows
    const bool store_z = c.mode == kHeadStored32;
    const bool e16 = c.mode == kHeadE16;
    const bool rowref = c.mode == kHeadRowRef;
    const HeadWs w = head_carve(c.ws, c.n_tok, c.V, c.K, ctas, c.mode);
    const bool kv = c.w_layout == AWR_W_K_BY_V;
    const __nv_bfloat16* H = reinterpret_cast<const __nv_bfloat16*>(c.hidden);
    // W as the B operand of Z = H W (n = v, contraction = k) and of dH = dS W^T (n = k, contraction = v)
    const OperandView w_fwd{c.w_head, c.V, c.K, kv ? c.V : c.K, kv ? kMajorMN : kMajorK};
    const OperandView w_bwd{c.w_head, c.K, c.V, kv ? c.V : c.K, kv ? kMajorK : kMajorMN};
    cudaError_t e = cudaMemsetAsync(w.zy, 0, (size_t)w.part_ld * 4, st);
    if (e != cudaSuccess) return e;

    // pass F + a3 over rows [r0, r0 + rows): log-sum-exp partials + gather, then the scalars.
    // Partials / gathered logits are indexed by global row (pointers pre-offset by r0).
    auto forward = [&](int64_t r0, int64_t rows, float* zout) -> cudaError_t {
        EpiArgs ea = {};
        ea.eout = (e16 || rowref) ? w.ds : nullptr; ea.eout_ld = w.ds_ld;
        ea.zref = rowref ? w.zref + r0 : nullptr;
        ea.part = w.part + r0; ea.part_ld = w.part_ld; ea.zy = w.zy + r0;
        ea.partz = c.rows->token_entropy ? w.partz + r0 : nullptr;
        ea.target_ids = c.rows->target_ids + r0;
        ea.zout = zout; ea.zout_ld = w.z_ld;
        // raster: when the H rows of this call fit in L2 (a panel: 39 MB at K = 2048) walk all of
        // its row tiles before the next W column tile, so W_head streams from HBM exactly once
        const int fgm = rows * c.K * 2 <= (48ll << 20) ? (int)((rows + kBM * ctas - 1) / (kBM * ctas)) : gm;
        if (rowref) {
            // the exp reference of every row of the panel: its largest logit among the first 256
            // vocabulary entries (one column tile of the same GEMM, 1 / 594 of the forward flops)
            EpiArgs er = {};
            er.zref_out = w.zref + r0;
            OperandView w_ref = w_fwd;
            w_ref.mn = c.V < kBN ? c.V : kBN;
            cudaError_t err = launch_gemm(kEpiRowMax, OperandView{H + r0 * c.K, rows, c.K, c.K, kMajorK},
                                          w_ref, 0, fgm, er, num_sms, ctas, st);
            if (err != cudaSuccess) return err;
        }
        cudaError_t err = launch_gemm(rowref ? kEpiLseRef : (e16 ? kEpiLse16 : kEpiLse),
                                      OperandView{H + r0 * c.K, rows, c.K, c.K, kMajorK},
                                      w_fwd, 0, fgm, ea, num_sms, ctas, st);
        if (err != cudaSuccess) return err;
        const int warps = 8;
        const unsigned blocks = (unsigned)((rows + warps - 1) / warps);
        HeadRefArgs ra = {};
        if (rowref) ra = HeadRefArgs{w.zref, w.row_f, w.ds, w.ds_ld, H, w.hs, c.K, w.fix};
        head_scalars_kernel<<<blocks, warps * 32, 0, st>>>(*c.rows, w.part, w.part_ld, w.n_vtiles,
                                                           c.rows->token_entropy ? w.partz : nullptr,
                                                           w.zy, w.row_lse, w.row_coef, w.row_gy,
                                                           r0, r0 + rows, ra);
        err = cudaGetLastError();
        if (err != cudaSuccess || !rowref) return err;
        // rows whose sum overflowed relative to their reference (none on ordinary logits): redone exactly
        const unsigned fblocks = (unsigned)(rows < 2 * (int64_t)num_sms ? rows : 2 * (int64_t)num_sms);
        head_fix_rows_kernel<<<fblocks, 512, 0, st>>>(*c.rows, ra, reinterpret_cast<const __nv_bfloat16*>(c.w_head),
                                                      kv ? 1 : 0, w.row_lse, w.row_coef, w.row_gy, r0, r0 + rows);
        return cudaGetLastError();
    };
    if (c.mode == kHeadRecompute) {
        e = forward(0, c.n_tok, nullptr);
        if (e != cudaSuccess) return e;
    }

    // Stored mode: the HBM-bound dS pass of panel p runs on a side stream beside the tensor-bound
    // forward GEMM of panel p + 1 (two logits buffers); both join before the panel's dhidden GEMM.
    // The side stream and its fork / join events come from the per-device pool keyed by the
    // caller's stream (side_acquire above: the only state the library keeps besides per-device
    // function attributes); the fork / join pattern is legal inside a CUDA-graph capture of the
    // caller's stream.
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    SideGuard guard{store_z ? side_acquire(st) : nullptr};       // E16 / recompute: no side stream
    if (guard.s) { side = guard.s->stream; ev_fork = guard.s->fork; ev_join = guard.s->join; }
    float* zbuf[2] = {w.zpanel, w.zpanel2};
    if (store_z && w.n_panels > 0) {
        const int64_t rows0 = c.n_tok < w.panel_rows ? c.n_tok : w.panel_rows;
        e = forward(0, rows0, zbuf[0]);
        if (e != cudaSuccess) return e;
    }

    // ---- row panels: dS, dhidden, dw_head
    for (int p = 0; p < w.n_panels; ++p) {
        const int64_t r0 = (int64_t)p * w.panel_rows;
        const int64_t rows = (c.n_tok - r0 < w.panel_rows) ? (c.n_tok - r0) : w.panel_rows;
        const __nv_bfloat16* Hp = H + r0 * c.K;
        if (store_z) {
            // dS of this panel from its stored fp32 logits: one streaming pass, on the side stream
            cudaStream_t ds_stream = side ? side : st;      // no idle side stream: in line
            if (side) {
                e = cudaEventRecord(ev_fork, st);
                if (e == cudaSuccess) e = cudaStreamWaitEvent(side, ev_fork, 0);
                if (e != cudaSuccess) return e;
            }
            const unsigned blocks = (unsigned)(rows < 4 * (int64_t)num_sms ? rows : 4 * (int64_t)num_sms);
            head_ds_kernel<<<blocks, 512, 0, ds_stream>>>(zbuf[p & 1], w.z_ld, rows, c.V,
                                                          c.rows->target_ids + r0, w.row_lse + r0,
                                                          w.row_coef + r0, w.row_gy + r0, w.ds, w.ds_ld);
            e = cudaGetLastError();
            if (e == cudaSuccess && side) e = cudaEventRecord(ev_join, side);
            if (e != cudaSuccess) return e;
            if (p + 1 < w.n_panels) {       // meanwhile: forward of the next panel into the other buffer
                const int64_t r1 = r0 + w.panel_rows;
                const int64_t rows1 = (c.n_tok - r1 < w.panel_rows) ? (c.n_tok - r1) : w.panel_rows;
                e = forward(r1, rows1, zbuf[(p + 1) & 1]);
                if (e != cudaSuccess) return e;
            }
            if (side) e = cudaStreamWaitEvent(st, ev_join, 0);
        } else if (e16) {
            // E16 mode: forward GEMM of this panel writes E = bf16(exp(z - tile max)) into the dS
            // panel; one in-place streaming pass turns it into dS.  One buffer, one stream.
            e = forward(r0, rows, nullptr);
            if (e != cudaSuccess) return e;
            const unsigned blocks = (unsigned)(rows < 4 * (int64_t)num_sms ? rows : 4 * (int64_t)num_sms);
            head_ds16_kernel<<<blocks, 512, 0, st>>>(w.ds, w.ds_ld, rows, c.V, c.rows->target_ids + r0,
                                                     w.part + r0, w.part_ld, w.row_lse + r0,
                                                     w.row_coef + r0, w.row_gy + r0);
            e = cudaGetLastError();
        } else if (rowref) {
            // row-reference mode: the forward GEMM leaves E = bf16(exp(z - zref)); the scalars kernel
            // patches the target entries and writes f_row and Hs = bf16(f_row H).  No pass over E.
            e = forward(r0, rows, nullptr);
        } else {
            EpiArgs e1 = {};
            e1.target_ids = c.rows->target_ids + r0; e1.row_lse = w.row_lse + r0;
            e1.row_coef = w.row_coef + r0; e1.row_gy = w.row_gy + r0;
            e1.ds = w.ds; e1.ds_ld = w.ds_ld;
            e = launch_gemm(kEpiDs, OperandView{Hp, rows, c.K, c.K, kMajorK}, w_fwd, 0, gm, e1, num_sms, ctas, st);
        }
        if (e != cudaSuccess) return e;

        EpiArgs e2 = {};
        e2.out = reinterpret_cast<__nv_bfloat16*>(c.dhidden) + r0 * c.K; e2.out_ld = c.K;
        e2.row_scale = rowref ? w.row_f + r0 : nullptr;
        e = launch_gemm(kEpiStoreBf16, OperandView{w.ds, rows, c.V, w.ds_ld, kMajorK}, w_bwd, 1, 1, e2,
                        num_sms, ctas, st, /*wide=*/true);
        if (e != cudaSuccess) return e;

        EpiArgs e3 = {};
        e3.out = reinterpret_cast<__nv_bfloat16*>(c.dw_head); e3.acc = w.dw_acc;
        e3.first_panel = p == 0; e3.last_panel = p == w.n_panels - 1;
        // H^T: m = k, contraction = t (row-reference mode: the rows of H already scaled by f_row)
        const OperandView ht{rowref ? w.hs : Hp, c.K, rows, c.K, kMajorMN};
        const OperandView dst{w.ds, c.V, rows, w.ds_ld, kMajorMN};   // dS:  n = v, contraction = t
        if (kv) {            // dw_head[k, v]
            e3.out_ld = c.V;
            e = launch_gemm(kEpiAccum, ht, dst, 0, 16 / ctas, e3, num_sms, ctas, st);
        } else {             // dw_head[v, k] = (dS^T H)[v, k]
            e3.out_ld = c.K;
            e = launch_gemm(kEpiAccum, dst, ht, 1, 1, e3, num_sms, ctas, st);
        }
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

int head_launches(int64_t n_tok, int64_t V, int64_t K, int ctas, int mode) {
    const HeadWs w = head_carve(nullptr, n_tok, V, K, ctas == 1 ? 1 : 2, mode);
    // recompute: F, scalars, then (dS GEMM, dH, dW) per panel; stored / E16: (F, scalars, dS pass, dH, dW) per panel
    // row reference: (reference tile, F, scalars, fix-up of overflowed rows, dH, dW) per panel
    if (mode == kHeadRowRef) return 6 * w.n_panels;
    return mode != kHeadRecompute ? 5 * w.n_panels : 2 + 3 * w.n_panels;
}

cudaError_t launch_gemm_bf16(const void* A, int a_major, int64_t lda, const void* B, int b_major,
                             int64_t ldb, int64_t M, int64_t N, int64_t Kc, void* C, int64_t ldc,
                             int num_sms, int ctas, cudaStream_t st) {
    EpiArgs e = {};
    e.out = reinterpret_cast<__nv_bfloat16*>(C); e.out_ld = ldc;
    ctas = ctas == 1 ? 1 : 2;
    return launch_gemm(kEpiStoreBf16, OperandView{A, M, Kc, lda, a_major}, OperandView{B, N, Kc, ldb, b_major},
                       0, 8 / ctas, e, num_sms, ctas, st);
}

}  // namespace awr
