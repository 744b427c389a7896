// tcgen05 / TMEM / TMA GEMM engine of the fused LM-head path (a5, BASELINE.json config 4).
//
//   C[M, N] = A[M, Kc] * B[Kc, N],  bf16 x bf16 -> fp32 accumulators in tensor memory,
//
// with the epilogue applied to the accumulator tile while it is still on chip: the log-sum-exp of
// Z = H * W_head is taken from the fp32 accumulators in tensor memory (reading
// A17); what an epilogue writes out of the tile besides the per-row partials depends on the mode
// (nothing / bf16 exp(z - max) / the fp32 tile of one row panel: awr_head.cu).
//
// One persistent CTA per SM, 256 threads, warp-specialised:
//   warp 0    TMA producer: cp.async.bulk.tensor (128-byte swizzle) into a smem ring
//   warp 1    MMA issuer: one lane issues tcgen05.mma.kind::f16, accumulating into one of two
//             256-column TMEM buffers
//   warp 2    TMEM allocator (512 columns = two accumulator tiles)
//   warps 4-7 epilogue: warp w reads TMEM lanes 32 (w % 4) .. +31 with tcgen05.ld, one
//             accumulator row per thread, 32 columns at a time; runs while the MMA warp fills
//             the other TMEM buffer with the next tile
// Two shapes of the same kernel (template parameter CTAS):
//   CTAS = 1  cta_group::1, tile 128 x 256, every CTA stages A 128 x 64 + B 256 x 64 per stage
//             (48 KB, 4 stages).  The tensor core reads 96 B/clk of operands from the shared
//             memory that TMA is filling at the same rate: the 128 B/clk port is the limit
//             (measured: tensor pipe 50-60 % active).
//   CTAS = 2  cta_group::2 (CTA pair on one TPC), tile 256 x 256: each CTA stages its 128 rows
//             of A and its 128 columns of B (32 KB, 6 stages); the pair's tensor cores share
//             the B halves, so each SM's shared memory serves 64 B/clk of operand reads and
//             takes 64 B/clk of fills.  The leader CTA issues the MMAs for both; all TMA
//             completions land on the leader's "full" barrier, tcgen05.commit multicasts the
//             "empty" and "accumulator ready" signals to both CTAs, and the epilogue warps of
//             both CTAs release the accumulator on the leader's barrier.
// Operands may be K-major (contraction index contiguous in memory) or MN-major (row / column
// index contiguous); both are staged by TMA in the canonical 128-byte-swizzled UMMA layouts,
// so H^T dS (both operands MN-major) needs no transposed copy of anything.
#pragma once

#include <cuda.h>

#include "awr_common.cuh"
#include "awr_ptx.cuh"

namespace awr {
namespace head {

constexpr int kBM = 128;           // tile rows  (UMMA M)
constexpr int kBN = 256;           // tile cols  (UMMA N)
constexpr int kBK = 64;            // contraction elements per stage (= one 128-byte swizzle row)
constexpr int kUmmaK = 16;         // contraction elements per tcgen05.mma (bf16)
constexpr int kThreads = 256;
constexpr int kABytes = kBM * kBK * 2;      // 16 KB: 128 rows of A per CTA in both shapes
constexpr int kTmemCols = 512;
constexpr int kMaxStages = 8;

// NT = 256-column accumulators per tile.  NT = 2 (CTA pairs only): a 256 x 512 tile fills all 512
// TMEM columns, so the accumulator is not double-buffered (the epilogue does not overlap the next
// tile) but every staged A row is used for twice as many columns: for the dhidden GEMM, whose
// contraction is 151,936 long and whose output is small, that cuts operand traffic by a quarter
// and halves the number of CTA pairs that must stream the same dS rows in step.
template <int CTAS, int NT = 1>
struct Geo {
    static constexpr int kTileM = kBM * CTAS;            // tile rows per CTA / CTA pair
    static constexpr int kTileN = kBN * NT;              // tile columns
    static constexpr int kLoadN = kBN / CTAS;            // B columns staged by one CTA per accumulator
    static constexpr int kBBytes1 = kLoadN * kBK * 2;    // 32 KB / 16 KB
    static constexpr int kBBytes = kBBytes1 * NT;
    static constexpr int kStageBytes = kABytes + kBBytes;
    static constexpr int kStages = CTAS == 1 ? 4 : (NT == 1 ? 7 : 4);
    static constexpr int kAccStages = 2 / NT;            // TMEM accumulator buffers
    static constexpr int kSmemBytes = kStages * kStageBytes + 1024 /* alignment */ + 256 /* barriers */;
};
// The LSE epilogue (kEpiLse) keeps the fp32 logits tile: a TMEM load hands every thread one ROW,
// and 16-byte stores to 32 different rows per instruction drain so slowly that the epilogue,
// not the tensor pipe, set the pace of the forward GEMM (ncu: its warps sat on the registers of
// outstanding stores).  Each epilogue warp therefore transposes its 32 x 32 chunk through a
// private padded shared-memory tile and stores whole 128-byte rows; the ring gives up one stage.
constexpr int kZStageLd = 36;                                   // floats per staged row (144 B)
constexpr int kZStageBytes = 4 * 32 * kZStageLd * 4;            // 4 epilogue warps: 18,432 B
template <int EPI, int CTAS, int NT>
struct EpiGeo {
    using G = Geo<CTAS, NT>;
    static constexpr bool kStaged = EPI == 0 || EPI == 4 || EPI == 5;   // kEpiLse, kEpiLse16, kEpiLseRef
    static constexpr int kStages = (kStaged && CTAS == 2 && NT == 1) ? G::kStages - 1 : G::kStages;
    static constexpr int kSmemBytes = kStages * G::kStageBytes + 1024 + 256 + (kStaged ? kZStageBytes : 0);
};
static_assert(EpiGeo<0, 2, 1>::kSmemBytes <= 232448 && EpiGeo<0, 1, 1>::kSmemBytes <= 232448, "shared memory");
static_assert(EpiGeo<4, 2, 1>::kSmemBytes <= 232448 && EpiGeo<4, 1, 1>::kSmemBytes <= 232448, "shared memory");
static_assert(EpiGeo<5, 2, 1>::kSmemBytes <= 232448 && EpiGeo<5, 1, 1>::kSmemBytes <= 232448, "shared memory");
static_assert(Geo<2>::kStages <= kMaxStages && Geo<2>::kSmemBytes <= 232448, "shared memory");
static_assert(Geo<2, 2>::kSmemBytes <= 232448, "shared memory");

enum { kMajorK = 0, kMajorMN = 1 };
enum { kEpiLse = 0,      // a2 on the tile: per-row (max, sum exp) partials + target gather
       kEpiDs = 1,       // a4 on the tile: dS = c_t (exp(z - lse) - onehot) -> bf16 panel
       kEpiStoreBf16 = 2,// C -> bf16 (dhidden)
       kEpiAccum = 3,    // C accumulated over row panels in fp32, bf16 on the last panel (dw_head)
       kEpiLse16 = 4,    // kEpiLse that also keeps the tile as E = bf16(exp(z - tile row max)): two
                         // passes over the accumulator (max, then exp + sum + store)
       kEpiLseRef = 5,   // the same with a PER-ROW reference known before the GEMM (zref[row]):
                         // E = bf16(exp(z - zref)) in ONE pass over the accumulator; dS = E * f_row, so
                         // the scale moves into the dhidden epilogue (row_scale) and into the H operand
                         // of the dw_head GEMM, and no dS pass is left
       kEpiRowMax = 6 }; // zref[row] = max of the tile's row (one column tile only: the reference of
                         // kEpiLseRef is the row's largest logit among the first 256 vocabulary entries)

// How one operand is staged and described to the tensor core (all runtime values).
struct Operand {
    uint32_t major;       // kMajorK / kMajorMN
    uint32_t rank3;       // MN-major operand described as a rank-3 tensor (64 x Kc x MN/64): the
                          // whole stage arrives with ONE bulk-tensor copy (a copy instruction
                          // costs its issuing thread ~250-300 clocks; with one 64-wide box per
                          // instruction the producer, not the tensor pipe, set the pace)
    uint32_t boxes;       // TMA boxes per stage
    uint32_t box_bytes;   // shared-memory bytes per box
    uint32_t desc_lo;     // leading-byte-offset field of the smem descriptor (bits 16..29)
    uint32_t desc_hi;     // stride-byte-offset, version 1, SWIZZLE_128B (upper 32 bits)
    uint32_t k_step;      // added to the start-address field per UMMA_K step (16-byte units)
};

struct EpiArgs {
    // kEpiLse
    float2* part;              // [n_tiles][part_ld] (max, sum) of every row over one column tile
    int64_t part_ld;
    float* partz;              // optional [n_tiles][part_ld]: sum e^{z - max} z of the tile (entropy)
    float* zy;                 // [M] gathered target logit (fp32 accumulator value)
    const int32_t* target_ids; // [M] (kEpiLse, kEpiDs), already offset to row 0 of this GEMM
    float* zout;               // optional [M, zout_ld]: the fp32 logits tile, kept for the dS pass
    int64_t zout_ld;
    __nv_bfloat16* eout;       // kEpiLse16 / kEpiLseRef [M, eout_ld]: E = exp(z - m), m the .x of part[]
    int64_t eout_ld;
    const float* zref;         // kEpiLseRef [M]: the row's exp reference (finite)
    float* zref_out;           // kEpiRowMax [M]
    // kEpiDs
    const float* row_lse;      // [M] log-sum-exp of the whole row
    const float* row_coef;     // [M] c_t
    const float* row_gy;       // [M] c_t (p_y - 1)
    __nv_bfloat16* ds;         // [M, ds_ld]
    int64_t ds_ld;
    // kEpiStoreBf16 / kEpiAccum
    const float* row_scale;    // kEpiStoreBf16, optional [M]: C row i is multiplied by row_scale[i]
                               // (0 gives an all-zero row whatever the accumulator holds)
    __nv_bfloat16* out;        // [M, out_ld]
    float* acc;                // [M, out_ld] fp32 running sum over panels
    int64_t out_ld;
    int32_t first_panel, last_panel;
};

struct GemmArgs {
    int32_t M, N, Kc;          // logical sizes (rows / cols beyond them are masked)
    int32_t m_tiles, n_tiles;
    int32_t order;             // 0: m fastest inside groups of group_m row tiles; 1: n fastest
    int32_t group_m;
    uint32_t idesc;            // tcgen05 instruction descriptor
    Operand a, b;
    EpiArgs e;
};

// ------------------------------------------------------------------ PTX wrappers (tcgen05; the rest: awr_ptx.cuh)
using namespace ptx;
__device__ __forceinline__ uint32_t cluster_rank() { return cluster_ctarank(); }
__device__ __forceinline__ uint32_t cluster_id() { return cluster_id_x(); }
__device__ __forceinline__ uint32_t num_clusters() { return num_clusters_x(); }
__device__ __forceinline__ void tc_fence_before() {
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tc_fence_after() {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}
// CTAS = 2: the arrive is multicast to the barrier at the same offset in both CTAs of the pair.
template <int CTAS>
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    if constexpr (CTAS == 1) {
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar)
                     : "memory");
    } else {
        asm volatile(
            "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 "
            "[%0], %1;" ::"r"(bar), "h"((uint16_t)3)
            : "memory");
    }
}
template <int CTAS>
__device__ __forceinline__ void tc_mma(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc,
                                       uint32_t idesc, uint32_t accumulate) {
    if constexpr (CTAS == 1) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "setp.ne.b32 p, %4, 0;\n"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
            "}\n" ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
            : "memory");
    } else {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "setp.ne.b32 p, %4, 0;\n"
            "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n"
            "}\n" ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
            : "memory");
    }
}
// 32 lanes x 32 consecutive columns -> 32 registers per thread (thread = TMEM lane = tile row)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32]) {
    uint32_t r[32];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]),
          "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]),
          "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]),
          "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]),
          "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}

// The same load without the wait, and the wait as a separate step that "touches" the 32
// registers so that the compiler cannot use them before it: lets the load of the next chunk fly
// while the current chunk is processed (ncu: 30 % of all stall samples of the LSE epilogue sat
// on the first consumer of a tcgen05.ld).
__device__ __forceinline__ void tmem_ld32_issue(uint32_t taddr, float (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]),
          "=f"(v[7]), "=f"(v[8]), "=f"(v[9]), "=f"(v[10]), "=f"(v[11]), "=f"(v[12]), "=f"(v[13]),
          "=f"(v[14]), "=f"(v[15]), "=f"(v[16]), "=f"(v[17]), "=f"(v[18]), "=f"(v[19]),
          "=f"(v[20]), "=f"(v[21]), "=f"(v[22]), "=f"(v[23]), "=f"(v[24]), "=f"(v[25]),
          "=f"(v[26]), "=f"(v[27]), "=f"(v[28]), "=f"(v[29]), "=f"(v[30]), "=f"(v[31])
        : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait(float (&v)[32]) {
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+f"(v[0]), "+f"(v[1]), "+f"(v[2]), "+f"(v[3]), "+f"(v[4]), "+f"(v[5]), "+f"(v[6]),
                   "+f"(v[7]), "+f"(v[8]), "+f"(v[9]), "+f"(v[10]), "+f"(v[11]), "+f"(v[12]),
                   "+f"(v[13]), "+f"(v[14]), "+f"(v[15]), "+f"(v[16]), "+f"(v[17]), "+f"(v[18]),
                   "+f"(v[19]), "+f"(v[20]), "+f"(v[21]), "+f"(v[22]), "+f"(v[23]), "+f"(v[24]),
                   "+f"(v[25]), "+f"(v[26]), "+f"(v[27]), "+f"(v[28]), "+f"(v[29]), "+f"(v[30]),
                   "+f"(v[31])
                 :
                 : "memory");
}

}  // namespace head
}  // namespace awr
