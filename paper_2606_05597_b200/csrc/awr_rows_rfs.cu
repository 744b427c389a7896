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
//     TMA stores alike), so the 148 KB of a row half need 4.7 k clocks of that port.
//   * Schedule: a software pipeline over rows in GROUPS of five rounds (= one staging buffer = 20
//     registers per thread).  In turn for each group: stage the gradient of row r out of the
//     group's registers (pass 2), refill them from the ring with the same group of row r + 1
//     (pass 0) and exponentiate it (pass 1).  Every group carries its own exp reference (the
//     thread's max over the group), so no warp-wide or row-wide max sits between the passes and
//     the MUFU-bound pass of the next row runs while the TMA stores of this row drain through the
//     write port.
//   * Statistics of the LAST group early (template parameter EARLY; AWR_KERNEL_CLUSTER_RFS, AUTO): the
//     row's (max, sum) can leave for a3 only when every element has been exponentiated, and the next
//     iteration needs a3's answer at once: st.async -> service warp -> publish is 1.5-2 k clocks that
//     every data warp waited for at the top of every row (14.7 % of the warp samples of a capture).
//     The last group's registers still hold the previous row at that point, so its statistics are
//     taken straight from the ring - two sweeps over shared memory (max; then exp, sum, and e written
//     back IN PLACE as bf16) - the statistics are sent, and only then is the previous row's last
//     group staged (pass 2) and the e reloaded from the ring: the hand-over runs behind that work.
//     EARLY = false (AWR_KERNEL_CLUSTER_RFS_LATE) keeps pass 2 / pass 0 / pass 1 for the last group
//     too and sends afterwards.  The row's last piece then reaches the TMA late, so the service lane
//     frees the staging buffer of the piece before it as soon as that piece's own store has read it
//     out (a blocking wait_group.read 0 at a point where nothing else is due) instead of at the next
//     hand-over.  Measured, config 1, same lease: EARLY 3.79 ms in the first
//     20 calls from an idle board (boost clock), 3.83-3.93 ms over the next 80, 3.97-4.07 ms at 1.65
//     GHz, 4.83-4.95 ms between bursts of dense GEMMs (1.35 GHz); late 3.97-4.09 / 3.78-3.91 /
//     3.91-4.04 / 4.90-4.99 ms; the predecessor schedule (pass 0 of the next row inside the staging
//     waits, then one MUFU pass per row) 3.69 / 4.12 / 4.30 / 5.45 ms.
//   * Exchange: every consumer warp sends its (max, sum[, sum e z]) with st.async to BOTH CTAs; the
//     16 bytes complete a transaction count on the receiver's mbarrier - no cluster barrier, no
//     fence.  The service warp of each CTA merges the 30 states, evaluates a3 once (header loads
//     issued a row ahead) and publishes (c_t, lse, c_t (p_y - 1)) in shared memory; the consumers
//     wait for that on an mbarrier and scale each group of registers by c_t exp(m_g - lse), m_g the
//     group's exp reference.
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
    float4 rowinfo[2];                                   // [row parity] (c_t, lse, c_t (p_y - 1), place of the NEXT row's target)
};
static_assert(sizeof(SvCtrl) <= kSvCtrlBytes, "control block");

struct SvPlan {
    int half_units[2];   // 16-byte units of the row held by CTA rank 0 / 1
    int half_base[2];    // first unit of each half
    int nr[2];           // rounds of each half: ceil(half_units / 480) (NU or NU - 1)
    int npieces[2];      // staging buffers per row of each half: ceil(nr / 5)
    int num_clusters;
};

// NU = rounds per row half = ceil(max half units / 480), compile time: the register array of a
// consumer thread is v[NU][4] (one 16-byte unit per round).
template <int NU, bool ENT, bool EARLY>
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
    // derived sizes come from the plan: kernel parameters cost no registers (selects, not indexing,
    // so that the parameter struct is not copied to local memory)
    const int half_units = rank ? p.half_units[1] : p.half_units[0];
    const int half_base = rank ? p.half_base[1] : p.half_base[0];          // first unit of this half
    const int nr = rank ? p.nr[1] : p.nr[0];                               // rounds of THIS half (<= NU)
    const int npieces = rank ? p.npieces[1] : p.npieces[0];                // staging buffers per row
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
        // An event loop over the three things the data warps hand over - a ring slot read out, the
        // 30 (max, sum) states of a row, a full staging buffer - so that a refill is issued the moment
        // its slot is free, whatever the stores are doing (polling with mbarrier.test_wait; the tests
        // are taken by the whole warp on one address and are warp-uniform).
        const uint8_t* lbase = reinterpret_cast<const uint8_t*>(a.logits) + (int64_t)half_base * 16;
        uint8_t* gbase = reinterpret_cast<uint8_t*>(a.dlogits) + (int64_t)half_base * 16;
        const int nrows = (n_tok - cluster + nc - 1) / nc;            // rows of this cluster
        auto issue_load = [&](int s, int j) {                          // lane 0: one bulk copy fills the slot
            const int u0 = s * kSvSlotRounds * kSvRoundUnits;
            const int units = min(kSvSlotRounds * kSvRoundUnits, half_units - u0);
            if (lane == 0 && units > 0) {
                mbar_expect_tx(full0 + 8u * s, (uint32_t)units * 16u);
                bulk_load(ring + (uint32_t)s * kSvSlotBytes,
                          lbase + (int64_t)(cluster + j * nc) * row_bytes + (int64_t)u0 * 16,
                          (uint32_t)units * 16u, full0 + 8u * s);
            }
        };
        int ld_j[NCH];                                    // next row index to load into each slot
#pragma unroll
        for (int s = 0; s < NCH; ++s) {
            issue_load(s, 0);
            ld_j[s] = (s * kSvSlotRounds < nr) ? 1 : nrows;           // a slot this half never uses
        }
        RowHeader h, hn;
        bool valid = false, validn = false;
        int yq = -1;                                      // lane 0: target of the row after the next a3
        if (lane == 0) {
            hn = load_row_header(a, cluster, validn, true);
            if (nrows > 1) yq = a.target_ids[cluster + nc];
            mbar_expect_tx(stats_full0, 2u * kSvConsumers * 16u);
            if (nrows > 1) mbar_expect_tx(stats_full0 + 8u, 2u * kSvConsumers * 16u);
        }
        int a3_j = 0;                                     // next row index to merge
        int st_j = backward ? 0 : nrows, st_pc = 0;       // next staging buffer to store: row index, piece
        uint32_t gpiece = 0;                              // staging buffers handed to the TMA so far
        bool freed_early = false;                         // lane 0: the previous piece's buffer is already free
        for (;;) {
            bool pending = false;
            // ---- a3: merge the 30 (max, sum) states, token scalars, publish (c_t, lse, gy, next target)
            if (a3_j < nrows) {
                pending = true;
                const int par = a3_j & 1;
                if (__all_sync(kFull, mbar_test(stats_full0 + 8u * par, (uint32_t)(a3_j >> 1) & 1u))) {
                    const int row = cluster + a3_j * nc;
                    h = hn; valid = validn;
                    // where the NEXT row's target sits in this half (the data warps mask it out of the
                    // row): holder thread << 16 | round * 8 + element of the unit, or -1
                    int hn_code = -1;
                    {
                        const int yu = (yq >= 0 && yq < a.V) ? (yq >> 3) - half_base : -1;
                        if (yu >= 0 && yu < half_units)
                            hn_code = ((yu % kSvRoundUnits) << 16) | ((yu / kSvRoundUnits) * 8 + (yq & 7));
                    }
                    const bool mine = lane < 2 * kSvConsumers;
                    const float4 st = ctrl->stats[par][mine ? lane : 0];
                    // max over the warp in ONE instruction: floats order like their bits once the
                    // negative ones are flipped (this chain is on the critical path of every data warp)
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
                        const float lse_rest = M + fast_log(S);           // -inf if nothing but the target
                        const TokenScalars ts = token_scalars(h, lse_rest, valid, a.clip_eps, a.stale_cap, a.dual_c);
                        ctrl->rowinfo[par] = make_float4(ts.coef, ts.lse, ts.gy, __int_as_float(hn_code));
                        mbar_arrive(ready0 + 8u * par);                   // release: rowinfo is visible
                        if (a3_j + 2 < nrows) mbar_expect_tx(stats_full0 + 8u * par, 2u * kSvConsumers * 16u);
                        // prefetches for the next a3, AFTER the publish: the header is a chain of
                        // dependent global loads (target -> its logit, trajectory -> its advantage)
                        // and in-order issue would hold the publish behind it (measured: 1.1-3.5 k
                        // clocks of every row with the loads in front, 530 behind)
                        if (a3_j + 1 < nrows) hn = load_row_header(a, row + nc, validn, true);
                        if (a3_j + 2 < nrows) yq = a.target_ids[row + 2 * nc];
                        if (rank == 0) {
                            store_token_outputs(a, row, h, ts, valid);
                            if (ENT) a.token_entropy[row] = valid ? row_entropy(ts.lse, M, SZ, ts.lp, h.zy) : 0.f;
                        }
                    }
                    __syncwarp();
                    ++a3_j;
                }
            }
            // ---- ring: refill a slot with its next row as soon as the 15 warps have read it out
#pragma unroll
            for (int s = 0; s < NCH; ++s) {
                if (ld_j[s] < nrows) {
                    pending = true;
                    if (__all_sync(kFull, mbar_test(empty0 + 8u * s, (uint32_t)(ld_j[s] - 1) & 1u))) {
                        issue_load(s, ld_j[s]);
                        ++ld_j[s];
                    }
                }
            }
            // ---- gradient: every full staging buffer goes out with one TMA bulk store
            if (st_j < nrows) {
                pending = true;
                const uint32_t b = gpiece & 1u;
                if (__all_sync(kFull, mbar_test(sfull0 + 8u * b, (gpiece >> 1) & 1u))) {
                    if (lane == 0) {
                        const int u0 = st_pc * kSvStageRounds * kSvRoundUnits;
                        const int units = min(kSvStageRounds * kSvRoundUnits, half_units - u0);
                        bulk_store(gbase + (int64_t)(cluster + st_j * nc) * row_bytes + (int64_t)u0 * 16,
                                   stage + b * kSvStageBytes, (uint32_t)units * 16u);
                        bulk_commit();
                        // all but this newest store have read their buffer out: the other buffer is free
                        bulk_wait_read<1>();
                        if (gpiece > 0 && !freed_early) mbar_arrive(sfree0 + 8u * (b ^ 1u));
                        freed_early = false;
                        // EARLY: the row's last piece is handed over late (after the sweeps over the
                        // ring), and the first piece of the NEXT row wants the buffer of the piece
                        // before it: free that one as soon as its own store has read it out instead of
                        // at the next hand-over (a capture had 8.9 % of all warp samples in that wait).
                        // Nothing else is due in these ~1.2 k clocks: the ring slots in use were
                        // refilled earlier, the row's statistics come after the sweeps.
                        if (EARLY && npieces >= 2 && st_pc == npieces - 2) {
                            bulk_wait_read<0>();
                            mbar_arrive(sfree0 + 8u * b);
                            freed_early = true;
                        }
                    }
                    __syncwarp();
                    ++gpiece;
                    if (++st_pc == npieces) { st_pc = 0; ++st_j; }
                }
            }
            if (!pending) break;
        }
        if (lane == 0) bulk_wait_all();                   // gradient writes complete before the CTA ends
    } else {
        // =============================================================== consumer warps
        // Software pipeline over rows in GROUPS of five rounds (= one staging buffer, half a ring
        // slot): iteration `it` stages the gradient of row `it` out of a group's 20 registers
        // (pass 2), refills them at once with the same group of row it + 1 (pass 0) and
        // exponentiates it (pass 1).  Every group of every thread carries its own exp reference
        // (the thread's max over the group, a bf16 value), so nothing in the loop body but the
        // hand-over barriers orders one group after another: the MUFU-bound pass of the next row
        // runs while the TMA stores of this row drain through the SM's 32 B/clk write port.
        // The kernel holds 80 data registers of its 128: all bookkeeping is packed (one int for the
        // place of a row's target, bf16 pairs for the exp references, rowinfo re-read from shared
        // memory) and the file is compiled with ptxas -O1 (build.py), where nothing spills.
        constexpr int NG = (NU + kSvStageRounds - 1) / kSvStageRounds;            // groups per row half
        constexpr int kGroupsPerSlot = kSvSlotRounds / kSvStageRounds;
        const uint32_t my_off = (uint32_t)(warp * 32 + lane) * 16u;      // byte offset inside a round
        uint32_t v[NU][4];
        uint32_t mref2[(NG + 1) / 2];                     // exp reference of each group's registers: bf16 pairs
#pragma unroll
        for (int g = 0; g < (NG + 1) / 2; ++g) mref2[g] = kSvNegInf2;
        auto get_mref = [&](int g) { return (g & 1) ? bf16_hi(mref2[g >> 1]) : bf16_lo(mref2[g >> 1]); };
        auto set_mref = [&](int g, float m) {            // m is a bf16 value: its high half, exactly
            const uint32_t b = __float_as_uint(m);
            mref2[g >> 1] = (g & 1) ? ((mref2[g >> 1] & 0x0000ffffu) | (b & 0xffff0000u))
                                    : ((mref2[g >> 1] & 0xffff0000u) | (b >> 16));
        };
        // where the target of a row sits for this thread: round * 8 + element inside the unit, or -1 if
        // another thread holds it.  First row: computed here; later rows: the service warp hands
        // (holder thread, place) over with rowinfo
        int ypos = -1;                                    // row being staged
        int ynpos;                                        // row being filled
        {
            const int y0 = a.target_ids[cluster];
            const int yu = (y0 >= 0 && y0 < a.V) ? (y0 >> 3) - half_base : -1;
            const bool holder = yu >= 0 && yu < half_units && (yu % kSvRoundUnits) == (int)(my_off >> 4);
            ynpos = holder ? (yu / kSvRoundUnits) * 8 + (y0 & 7) : -1;
        }
        int it = -1;                                      // iteration -1 only fills the first row
        for (int row = cluster - nc; row < n_tok; row += nc, ++it) {
            const int par = it & 1;
            const bool have_cur = it >= 0;
            const bool have_next = row + nc < n_tok;

            // ---- a3 of this row ran on the service warp: (c_t, lse, c_t (p_y - 1), place of the next
            // row's target).  rowinfo[par] stays valid for the whole iteration and is re-read where
            // it is needed instead of being held in registers
            const float4* rinfo = &ctrl->rowinfo[par];
            if (have_cur) {
                mbar_wait_hint(ready0 + 8u * par, (uint32_t)(it >> 1) & 1u, 1000u);
                const int code = __float_as_int(rinfo->w);
                ynpos = (code >> 16) == (int)(my_off >> 4) ? (code & 0xffff) : -1;
            }

            float mrun = -INFINITY, st = 0.f, szt = 0.f;  // this thread's (max, sum, sum e z) of the next row
            // the warp's state of the next row, then the exchange: (m_w, s_w, sz_w) to both CTAs, data
            // and signal in one st.async each
            auto send_stats = [&]() {
                // max over the warp in ONE instruction (floats order like their bits once the negative
                // ones are flipped): this chain is on the critical path of the a3 hand-over
                int mi = __float_as_int(mrun);
                mi ^= (mi >> 31) & 0x7fffffff;
                mi = __reduce_max_sync(kFull, mi);
                mi ^= (mi >> 31) & 0x7fffffff;
                const float wm = __int_as_float(mi);
                const float sc = (mrun == -INFINITY) ? 0.f : ex2_approx((mrun - wm) * kLog2e);
                st *= sc;
                if (ENT) szt *= sc;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    st += __shfl_xor_sync(kFull, st, o);
                    if (ENT) szt += __shfl_xor_sync(kFull, szt, o);
                }
                if (lane < 2)
                    st_async_f32x4(smem_u32(&ctrl->stats[par ^ 1][(int)rank * kSvConsumers + warp]),
                                   stats_full0 + 8u * (uint32_t)(par ^ 1), (uint32_t)lane, wm, st, szt, 0.f);
            };
            // fold a group's (m, sum, sum e z) into the thread's state of the row
            auto fold = [&](float m, float gsum, float gsz) {
                const float M = fmaxf(mrun, m);
                const float f_old = (mrun == -INFINITY) ? 0.f : ex2_approx((mrun - M) * kLog2e);
                const float f_new = (m == -INFINITY) ? 0.f : ex2_approx((m - M) * kLog2e);
                st = st * f_old + gsum * f_new;
                if (ENT) szt = szt * f_old + gsz * f_new;
                mrun = M;
            };
            const uint32_t src = ring + my_off;                  // the ring slots are contiguous
            // the last group's reference of THIS row: its slot in mref2 is overwritten (next row) before
            // this row's pass 2 of that group reads it
            const float mref_last = get_mref(NG - 1);
            auto mref_cur = [&](int g) { return g == NG - 1 ? mref_last : get_mref(g); };
#pragma unroll
            for (int g = 0; g < NG; ++g) {
                const int sl = g / kGroupsPerSlot;
                const bool slot_used = sl * kSvSlotRounds < nr;                       // warp-uniform
                const bool last = g == NG - 1;                                        // compile time
                // ---- LAST group of the next row, early: its (max, sum) straight from the ring while
                // its registers still hold this row, e = exp2((z - m) log2 e) written back IN PLACE as
                // bf16, so that the row's statistics leave for a3 before pass 2 of this group instead
                // of after its pass 1: the a3 hand-over (st.async -> service warp -> publish, 1.5-2 k
                // clocks that every data warp used to wait for at the top of the next row) runs
                // behind that pass 2 and the reload.  Two sweeps over shared memory (max, then exp):
                // every thread re-reads only the 16-byte units it wrote itself.
                if (EARLY && last && have_next) {
                    if (g % kGroupsPerSlot == 0 && slot_used) mbar_wait(full0 + 8u * sl, (uint32_t)(it + 1) & 1u);
                    // the target entry is left out of the row's state: its holder overwrites it with
                    // -inf in the ring (its own later loads of that unit follow in program order)
                    if (ynpos >= g * kSvStageRounds * 8) {
                        const uint32_t at = src + (uint32_t)(ynpos >> 3) * kSvRoundBytes + (uint32_t)(ynpos & 7) * 2u;
                        asm volatile("st.shared.u16 [%0], %1;" ::"r"(at), "h"((unsigned short)0xff80) : "memory");
                    }
                    auto load_masked = [&](int k, uint32_t (&t)[4]) {
                        lds128(t, src + (uint32_t)k * kSvRoundBytes);
                        if (k >= NU - 2 && k * kSvRoundUnits + (int)(my_off >> 4) >= half_units)
                            t[0] = t[1] = t[2] = t[3] = kSvNegInf2;
                    };
                    uint32_t mx2 = kSvNegInf2;
#pragma unroll
                    for (int kk = 0; kk < kSvStageRounds; ++kk) {
                        const int k = g * kSvStageRounds + kk;
                        if (k < NU) {
                            uint32_t t[4];
                            load_masked(k, t);
                            mx2 = max_bf16x2(mx2, max_bf16x2(max_bf16x2(t[0], t[1]), max_bf16x2(t[2], t[3])));
                        }
                    }
                    const float m = fmaxf(bf16_lo(mx2), bf16_hi(mx2));
                    const float nref = (m == -INFINITY) ? 0.f : -m * kLog2e;
                    const float2 l2 = make_float2(kLog2e, kLog2e), nref2 = make_float2(nref, nref);
                    float2 acc[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
                    float2 accz = make_float2(0.f, 0.f);
#pragma unroll
                    for (int kk = 0; kk < kSvStageRounds; ++kk) {
                        const int k = g * kSvStageRounds + kk;
                        if (k < NU) {
                            uint32_t t[4];
                            load_masked(k, t);
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                const float2 z = make_float2(bf16_lo(t[j]), bf16_hi(t[j]));
                                const float2 x = fma_f32x2(z, l2, nref2);
                                const float2 e = make_float2(ex2_approx(x.x), ex2_approx(x.y));
                                acc[j & 1] = add_f32x2(acc[j & 1], e);
                                if (ENT)
                                    accz = fma_f32x2(e, make_float2(fmaxf(z.x, kZFloor), fmaxf(z.y, kZFloor)), accz);
                                t[j] = pack_bf16x2(e.x, e.y);
                            }
                            sts128(src + (uint32_t)k * kSvRoundBytes, make_uint4(t[0], t[1], t[2], t[3]));
                        }
                    }
                    fold(m, (acc[0].x + acc[0].y) + (acc[1].x + acc[1].y), accz.x + accz.y);
                    set_mref(g, m);
                    send_stats();
                }
                // ---- pass 2 (a4) of this row, group g: dlogits = e * (c_t exp(m_g - lse)) into a
                // staging buffer.  c_t = 0 (masked, zero advantage, clip triggered): F = +0 and
                // e >= 0 give all-bits-zero products
                if (backward && have_cur && g * kSvStageRounds < nr) {
                    const float2 cl = *reinterpret_cast<const float2*>(rinfo);            // (c_t, lse)
                    const float F = cl.x == 0.f ? 0.f : cl.x * ex2_approx((mref_cur(g) - cl.y) * kLog2e);
                    const __nv_bfloat16 fh = __float2bfloat16_rn(F);
                    const __nv_bfloat16 fl = __float2bfloat16_rn(F - __bfloat162float(fh));
                    const uint32_t Fh = (uint32_t)__bfloat16_as_ushort(fh) * 0x00010001u;
                    const uint32_t Fl = (uint32_t)__bfloat16_as_ushort(fl) * 0x00010001u;
                    const uint32_t gp = (uint32_t)(it * npieces + g);          // staging buffers filled so far
                    const uint32_t buf = stage + (gp & 1u) * kSvStageBytes + my_off;
                    mbar_wait(sfree0 + 8u * (gp & 1u), ((gp >> 1) & 1u) ^ 1u);
#pragma unroll
                    for (int kk = 0; kk < kSvStageRounds; ++kk) {
                        const int k = g * kSvStageRounds + kk;
                        if (k < NU && (k < NU - 1 || k < nr)) {               // nr >= NU - 1; warp-uniform
                            uint4 o;
                            o.x = fma_bf16x2(v[k][0], Fh, mul_bf16x2(v[k][0], Fl));
                            o.y = fma_bf16x2(v[k][1], Fh, mul_bf16x2(v[k][1], Fl));
                            o.z = fma_bf16x2(v[k][2], Fh, mul_bf16x2(v[k][2], Fl));
                            o.w = fma_bf16x2(v[k][3], Fh, mul_bf16x2(v[k][3], Fl));
                            sts128(buf + (uint32_t)kk * kSvRoundBytes, o);
                        }
                    }
                    // target entry: c (p_y - 1), patched into the staged unit by the one thread that
                    // holds it (its own 16-byte store above is earlier in program order)
                    if (ypos >= g * kSvStageRounds * 8 && ypos < (g + 1) * kSvStageRounds * 8 && cl.x != 0.f) {
                        const uint32_t at = buf + (uint32_t)((ypos >> 3) - g * kSvStageRounds) * kSvRoundBytes +
                                            (uint32_t)(ypos & 7) * 2u;
                        const unsigned short gy = __bfloat16_as_ushort(__float2bfloat16_rn(rinfo->z));
                        asm volatile("st.shared.u16 [%0], %1;" ::"r"(at), "h"(gy) : "memory");
                    }
                    fence_proxy_async();                                          // generic writes -> TMA read
                    __syncwarp();
                    if (lane == 0) mbar_arrive(sfull0 + 8u * (gp & 1u));
                }
                if (!have_next) continue;
                if (EARLY && last) {
                    // ---- reload of the last group: the e written above, ring -> registers; the slot
                    // is released behind a proxy fence (the next fill of the slot is an async-proxy
                    // write over these generic-proxy writes)
#pragma unroll
                    for (int kk = 0; kk < kSvStageRounds; ++kk) {
                        const int k = g * kSvStageRounds + kk;
                        if (k < NU) lds128(v[k], src + (uint32_t)k * kSvRoundBytes);
                    }
                    if (slot_used) {
                        fence_proxy_async();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(empty0 + 8u * sl);
                    }
                    continue;
                }
                // ---- pass 0 of the next row, group g: ring -> registers, target entry masked to -inf
                // (token_scalars works from lse_rest), packed max; the slot is released after its
                // last group
                if (g % kGroupsPerSlot == 0 && slot_used) mbar_wait(full0 + 8u * sl, (uint32_t)(it + 1) & 1u);
#pragma unroll
                for (int kk = 0; kk < kSvStageRounds; ++kk) {
                    const int k = g * kSvStageRounds + kk;
                    if (k < NU) {
                        // rounds below NU - 2 are full on both ranks; a stale read of the ring is harmless
                        lds128(v[k], src + (uint32_t)k * kSvRoundBytes);
                        if (k >= NU - 2 && k * kSvRoundUnits + (int)(my_off >> 4) >= half_units)
                            v[k][0] = v[k][1] = v[k][2] = v[k][3] = kSvNegInf2;
                    }
                }
                if ((g % kGroupsPerSlot == kGroupsPerSlot - 1 || g == NG - 1) && slot_used) {
                    __syncwarp();                                 // the slot has been read out by the warp
                    if (lane == 0) mbar_arrive(empty0 + 8u * sl);
                }
                // one thread of the cluster holds the target: a warp-uniform branch around its masking
                if (__any_sync(kFull, ynpos >= g * kSvStageRounds * 8 && ynpos < (g + 1) * kSvStageRounds * 8)) {
                    const uint32_t half = (ynpos & 1) ? 0xffff0000u : 0x0000ffffu;     // the target's half of its word
#pragma unroll
                    for (int kk = 0; kk < kSvStageRounds; ++kk) {
                        const int k = g * kSvStageRounds + kk;
                        if (k < NU) {
#pragma unroll
                            for (int j = 0; j < 4; ++j) {      // every word by name: v must stay in registers
                                const uint32_t mk = (k * 4 + j == (ynpos >> 1)) ? half : 0u;
                                v[k][j] = (v[k][j] & ~mk) | (kSvNegInf2 & mk);
                            }
                        }
                    }
                }
                uint32_t mx2 = kSvNegInf2;
#pragma unroll
                for (int kk = 0; kk < kSvStageRounds; ++kk) {
                    const int k = g * kSvStageRounds + kk;
                    if (k < NU)
                        mx2 = max_bf16x2(mx2, max_bf16x2(max_bf16x2(v[k][0], v[k][1]), max_bf16x2(v[k][2], v[k][3])));
                }
                // ---- pass 1 of the next row, group g: z -> e = exp2((z - m) log2 e) as bf16, in
                // registers, m = this thread's max over the group; f32 sums.  FFMA2 / FADD2: the (low,
                // high) elements of a word are one packed f32x2 operation (half the issue slots)
                const float m = fmaxf(bf16_lo(mx2), bf16_hi(mx2));
                const float nref = (m == -INFINITY) ? 0.f : -m * kLog2e;
                const float2 l2 = make_float2(kLog2e, kLog2e), nref2 = make_float2(nref, nref);
                float2 acc[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
                float2 accz = make_float2(0.f, 0.f);
#pragma unroll
                for (int kk = 0; kk < kSvStageRounds; ++kk) {
                    const int k = g * kSvStageRounds + kk;
                    if (k < NU) {
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const float2 z = make_float2(bf16_lo(v[k][j]), bf16_hi(v[k][j]));
                            const float2 x = fma_f32x2(z, l2, nref2);
                            const float2 e = make_float2(ex2_approx(x.x), ex2_approx(x.y));
                            acc[j & 1] = add_f32x2(acc[j & 1], e);
                            if (ENT)
                                accz = fma_f32x2(e, make_float2(fmaxf(z.x, kZFloor), fmaxf(z.y, kZFloor)), accz);
                            v[k][j] = pack_bf16x2(e.x, e.y);
                        }
                    }
                }
                fold(m, (acc[0].x + acc[0].y) + (acc[1].x + acc[1].y), accz.x + accz.y);
                set_mref(g, m);
            }
            if (!EARLY && have_next) send_stats();     // the late schedule: after pass 1 of the last group
            ypos = ynpos;
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
    p.half_base[0] = 0;
    p.half_base[1] = (int)h0;
    for (int r = 0; r < 2; ++r) {
        p.nr[r] = (p.half_units[r] + kSvRoundUnits - 1) / kSvRoundUnits;
        p.npieces[r] = (p.nr[r] + kSvStageRounds - 1) / kSvStageRounds;
    }
    p.num_clusters = 0;
    nu = (int)n;
    return true;
}

bool rows_rfs_supported(int64_t V, int64_t ld, int dtype) {
    SvPlan p;
    int nu;
    return make_sv_plan(V, ld, dtype, p, nu);
}

template <int NU, bool ENT, bool EARLY>
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
        cudaError_t e = cudaFuncSetAttribute(rows_rfs_kernel<NU, ENT, EARLY>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, kSvSmemBytes);
        if (e != cudaSuccess) return e;
        cfg.gridDim = dim3(2 * num_sms, 1, 1);
        int n = 0;
        e = cudaOccupancyMaxActiveClusters(&n, rows_rfs_kernel<NU, ENT, EARLY>, &cfg);
        if (e != cudaSuccess) return e;
        const int want = num_sms / 2;
        max_clusters = n < 1 ? 1 : (n > want ? want : n);
        cached.set(dev, max_clusters);
    }
    int nc = max_clusters;
    if ((int64_t)nc > a.n_tok) nc = (int)a.n_tok;
    p.num_clusters = nc;
    cfg.gridDim = dim3(2 * nc, 1, 1);
    return cudaLaunchKernelEx(&cfg, rows_rfs_kernel<NU, ENT, EARLY>, a, p);
}

template <bool EARLY>
static cudaError_t launch_rows_rfs_t(const RowArgs& a, int num_sms, cudaStream_t st) {
    if (a.n_tok <= 0) return cudaSuccess;
    SvPlan p;
    int nu = 0;
    if (!make_sv_plan(a.V, a.ld, AWR_DTYPE_BF16, p, nu)) return cudaErrorInvalidValue;
    switch (nu) {
#define AWR_SV_CASE(N)                                                                       \
    case N:                                                                                  \
        return a.token_entropy != nullptr ? launch_sv<N, true, EARLY>(a, p, num_sms, st)     \
                                          : launch_sv<N, false, EARLY>(a, p, num_sms, st);
        AWR_SV_CASE(3) AWR_SV_CASE(4) AWR_SV_CASE(5) AWR_SV_CASE(6) AWR_SV_CASE(7) AWR_SV_CASE(8)
        AWR_SV_CASE(9) AWR_SV_CASE(10) AWR_SV_CASE(11) AWR_SV_CASE(12) AWR_SV_CASE(13)
        AWR_SV_CASE(14) AWR_SV_CASE(15) AWR_SV_CASE(16) AWR_SV_CASE(17) AWR_SV_CASE(18)
        AWR_SV_CASE(19) AWR_SV_CASE(20)
#undef AWR_SV_CASE
        default: return cudaErrorInvalidValue;
    }
}

// early_stats: the schedule (file header); both produce the same values up to fp32 rounding of the
// last group's sum
cudaError_t launch_rows_rfs(const RowArgs& a, int num_sms, bool early_stats, cudaStream_t st) {
    return early_stats ? launch_rows_rfs_t<true>(a, num_sms, st) : launch_rows_rfs_t<false>(a, num_sms, st);
}

}  // namespace awr
