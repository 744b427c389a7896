// Cluster row kernel: a2 + a3 + a4 for large bf16 vocabularies, one HBM read and one HBM write
// per element.  PAPER.md:57 (Eq. 1), :435; gradient SURVEY.md 8(c) O8.
//
// Design:
//   * A 151,936-entry bf16 row (303,872 B) does not fit one SM's 227 KB of shared memory, so a
//     row is split across a 2-CTA thread-block cluster; each CTA keeps its half resident in
//     shared memory between the log-sum-exp pass and the gradient pass.  The two CTAs exchange
//     only their (max, sum) pair through distributed shared memory.
//   * Inside a CTA every warp owns a contiguous part of the half row and runs its own
//     software pipeline on a private ring of shared-memory slots: TMA bulk copies
//     (cp.async.bulk, mbarrier complete_tx) fill slots, the warp reduces them (pass 1),
//     rewrites them in place with the gradient (pass 2) and hands them to a TMA bulk store;
//     a slot is refilled with data of a *later* row as soon as its store has been read out.
//     There is no block-wide barrier inside a pass; the only block / cluster synchronisation
//     is the once-per-row exchange of the log-sum-exp state.
//   * Persistent: one cluster per SM pair, rows dealt round-robin to clusters (static schedule).
//   * Rows whose coefficient c_t is zero (masked, zero advantage, clip triggered) skip pass 2
//     and are written from a shared zero page.
#include "awr_common.cuh"
#include "awr_kernels.h"
#include "awr_ptx.cuh"

namespace awr {

constexpr int kCWarps = 16;
constexpr int kCThreads = kCWarps * 32;
constexpr int kMaxSlots = 16;
constexpr int kRound = 128;             // 16-byte units per warp round (4 per lane)
constexpr int kSmemLimit = 232448;      // 227 KB: max dynamic shared memory per CTA on sm_100
constexpr int kCtrlBytes = 2560;        // control block at the start of shared memory

struct ClusterPlan {
    int units_per_row;   // 16-byte units in one row (V * 2 / 16)
    int chunk_units;     // CU: units per ring slot / per TMA copy
    int slots;           // S: ring slots per warp
    int num_clusters;
};

struct Ctrl {
    uint64_t full[kCWarps * kMaxSlots];   // one mbarrier per ring slot per warp     (2048 B)
    MaxSum red[kCWarps];                  // per-warp log-sum-exp state               (128 B)
    MaxSum stats[2][2];                   // [row parity][cta rank], written by both CTAs
    RowHeader hdr[2];                     // [row parity]
    int hdr_valid[2];
};
static_assert(sizeof(Ctrl) <= kCtrlBytes, "control block");

using namespace ptx;

// ---------------------------------------------------------------- the kernel
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kCThreads, 1)
rows_cluster_kernel(RowArgs a, ClusterPlan p) {
    extern __shared__ __align__(128) uint8_t smem[];
    Ctrl* ctrl = reinterpret_cast<Ctrl*>(smem);
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    const uint32_t rank = cluster_ctarank();
    const int cluster = (int)cluster_id_x();
    const int CU = p.chunk_units;
    const int S = p.slots;
    const int ring_units = S * CU;
    const uint32_t zero_page = smem_u32(smem + kCtrlBytes);
    const uint32_t ring = zero_page + (uint32_t)CU * 16u + (uint32_t)warp * (uint32_t)ring_units * 16u;
    const uint32_t bar0 = smem_u32(&ctrl->full[warp * kMaxSlots]);

    // this warp's part of the row, in 16-byte units: [part0, part0 + part_units)
    const int part_idx = (int)rank * kCWarps + warp;
    const int nparts = 2 * kCWarps;
    const int part0 = (int)(((int64_t)p.units_per_row * part_idx) / nparts);
    const int part_units = (int)(((int64_t)p.units_per_row * (part_idx + 1)) / nparts) - part0;
    const int nch = (part_units + CU - 1) / CU;

    const int64_t my_rows = (a.n_tok - cluster + p.num_clusters - 1) / p.num_clusters;
    const int64_t total_seq = my_rows * nch;
    const bool backward = a.dlogits != nullptr;
    const uint8_t* lbase = reinterpret_cast<const uint8_t*>(a.logits);
    uint8_t* gbase = reinterpret_cast<uint8_t*>(a.dlogits);
    const int64_t row_bytes = a.ld * 2;

    // ---- setup: zero page, barriers
    for (int i = tid; i < CU * 4; i += kCThreads)
        reinterpret_cast<uint32_t*>(smem + kCtrlBytes)[i] = 0u;
    if (lane == 0)
        for (int s = 0; s < S; ++s) mbar_init(bar0 + 8u * s, 1);
    fence_mbar_init();
    fence_proxy_async();      // zero page (generic writes) -> later TMA store reads
    __syncthreads();
    cluster_arrive();
    cluster_wait();

    // ---- per-warp pipeline state (uniform across the warp)
    int64_t ld_seq = 0;       // next chunk (sequence number) to load
    int64_t ld_row = cluster; // its row
    int ld_ch = 0, ld_slot = 0;
    uint32_t phase_bits = 0;  // bit s: parity the next wait on slot s uses
    int slot0 = 0;            // slot of the current row's first chunk
    int64_t seq0 = 0;         // sequence number of the current row's first chunk
    int64_t done_seq = -1;    // every slot of sequence <= done_seq may be overwritten
    bool lazy_free = false;   // the previous row's last store has not been waited for yet

    auto refill = [&]() {     // lane 0 only does the work, state stays warp-uniform
        while (ld_seq < total_seq && ld_seq - S <= done_seq) {
            if (lane == 0) {
                const int u0 = ld_ch * CU;
                const uint32_t bytes = (uint32_t)min(CU, part_units - u0) * 16u;
                const uint32_t bar = bar0 + 8u * ld_slot;
                mbar_expect_tx(bar, bytes);
                bulk_load(ring + (uint32_t)(ld_slot * CU) * 16u,
                          lbase + ld_row * row_bytes + (int64_t)(part0 + u0) * 16, bytes, bar);
            }
            ++ld_seq;
            if (++ld_ch == nch) { ld_ch = 0; ld_row += p.num_clusters; }
            if (++ld_slot == S) ld_slot = 0;
        }
    };
    refill();                 // prologue: sequence numbers 0 .. S-1 fill the ring

    int par = 0;
    int y_next = cluster < a.n_tok ? a.target_ids[cluster] : -1;
    for (int64_t row = cluster; row < a.n_tok; row += p.num_clusters, par ^= 1) {
        // ---- row header (one thread per CTA; both CTAs load the same values)
        if (tid == 0) {
            bool valid;
            RowHeader h = load_row_header(a, row, valid, true);
            ctrl->hdr[par] = h;
            ctrl->hdr_valid[par] = valid ? 1 : 0;
        }
        // The target entry is left out of the (max, sum) state (token_scalars works from
        // lse_rest).  Every thread knows its position; the next row's id is fetched now so
        // that its latency hides behind this row.  A masked / out-of-range id matches no unit.
        const int y_row = y_next;
        {
            const int64_t nrow = row + p.num_clusters;
            y_next = nrow < a.n_tok ? a.target_ids[nrow] : -1;
        }
        const int y_unit1 = (y_row >> 3) - part0;            // unit index inside this part
        const uint32_t y_word = (uint32_t)(y_row & 7) >> 1;
        const uint32_t y_keep = (y_row & 1) ? 0x0000ffffu : 0xffff0000u;
        const uint32_t y_ninf = 0xff80ff80u & ~y_keep;       // bf16 -inf in the target's half

        // ---- pass 1 (a2): online (max, sum) over this warp's part, as the chunks land
        MaxSum ms{-INFINITY, 0.f};
        const int start_unit = slot0 * CU;
        int waited = 0;       // chunks of this row already waited for
        for (int ubase = 0; ubase < part_units; ubase += kRound) {
            const int uend = min(ubase + kRound, part_units);
            while (waited * CU < uend) {
                int s = slot0 + waited; if (s >= S) s -= S;
                mbar_wait(bar0 + 8u * s, (phase_bits >> s) & 1u);
                phase_bits ^= 1u << s;
                ++waited;
            }
            uint4 v[4];
            bool ok[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int u = ubase + k * 32 + lane;
                ok[k] = u < part_units;
                int pos = start_unit + u; if (pos >= ring_units) pos -= ring_units;
                v[k] = ok[k] ? lds128(ring + (uint32_t)pos * 16u)
                             : make_uint4(0xff80ff80u, 0xff80ff80u, 0xff80ff80u, 0xff80ff80u);
            }
            if (y_unit1 >= ubase && y_unit1 < uend) {          // warp-uniform, once per row
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    if (ubase + k * 32 + lane == y_unit1) {
                        v[k].x = y_word == 0 ? (v[k].x & y_keep) | y_ninf : v[k].x;
                        v[k].y = y_word == 1 ? (v[k].y & y_keep) | y_ninf : v[k].y;
                        v[k].z = y_word == 2 ? (v[k].z & y_keep) | y_ninf : v[k].z;
                        v[k].w = y_word == 3 ? (v[k].w & y_keep) | y_ninf : v[k].w;
                    }
                }
            }
            // packed running max of the round (bf16x2), then one rescale check
            uint32_t m2 = max_bf16x2(max_bf16x2(v[0].x, v[0].y), max_bf16x2(v[0].z, v[0].w));
#pragma unroll
            for (int k = 1; k < 4; ++k) {
                m2 = max_bf16x2(m2, max_bf16x2(max_bf16x2(v[k].x, v[k].y),
                                               max_bf16x2(v[k].z, v[k].w)));
            }
            const float cm = fmaxf(bf16_lo(m2), bf16_hi(m2));
            if (cm > ms.m) {
                ms.s *= ex2_approx((ms.m - cm) * kLog2e);
                ms.m = cm;
            }
            // a lane that has only seen -inf so far must not form (-inf) - (-inf)
            const float nml = (ms.m == -INFINITY) ? 0.f : -ms.m * kLog2e;
            float acc0 = 0.f, acc1 = 0.f;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                if (ok[k]) {
                    acc0 += ex2_approx(fmaf(bf16_lo(v[k].x), kLog2e, nml));
                    acc1 += ex2_approx(fmaf(bf16_hi(v[k].x), kLog2e, nml));
                    acc0 += ex2_approx(fmaf(bf16_lo(v[k].y), kLog2e, nml));
                    acc1 += ex2_approx(fmaf(bf16_hi(v[k].y), kLog2e, nml));
                    acc0 += ex2_approx(fmaf(bf16_lo(v[k].z), kLog2e, nml));
                    acc1 += ex2_approx(fmaf(bf16_hi(v[k].z), kLog2e, nml));
                    acc0 += ex2_approx(fmaf(bf16_lo(v[k].w), kLog2e, nml));
                    acc1 += ex2_approx(fmaf(bf16_hi(v[k].w), kLog2e, nml));
                }
            }
            ms.s += acc0 + acc1;
            if (lazy_free) {
                // the previous row's last store has surely been read out by now
                if (lane == 0) bulk_wait_read<0>();
                done_seq = seq0 - 1;
                lazy_free = false;
                refill();
            }
        }

        // ---- exchange: warp -> CTA -> cluster
        ms = warp_combine(ms);
        if (lane == 0) ctrl->red[warp] = ms;
        __syncthreads();
        if (tid == 0) {
            MaxSum tot = ctrl->red[0];
#pragma unroll
            for (int w = 1; w < kCWarps; ++w) tot = combine(tot, ctrl->red[w]);
            const uint32_t addr = smem_u32(&ctrl->stats[par][rank]);
            st_cluster_f32x2(addr, 0, tot.m, tot.s);
            st_cluster_f32x2(addr, 1, tot.m, tot.s);
        }
        __syncwarp();
        cluster_arrive();
        cluster_wait();
        const MaxSum tot = combine(ctrl->stats[par][0], ctrl->stats[par][1]);
        const float lse_rest = tot.m + logf(tot.s);          // -inf if nothing but the target
        const RowHeader h = ctrl->hdr[par];
        const bool valid = ctrl->hdr_valid[par] != 0;

        // ---- a3: per-token scalars (every thread, identical arithmetic)
        const TokenScalars ts = token_scalars(h, lse_rest, valid, a.clip_eps, a.stale_cap, a.dual_c);
        const float lse = ts.lse;
        if (tid == 0 && rank == 0) store_token_outputs(a, row, h, ts, valid);

        // ---- pass 2 (a4)
        if (!backward) {
            done_seq = seq0 + nch - 1;      // nothing to store: the whole part is free
            refill();
        } else if (ts.coef == 0.f) {
            uint8_t* grow = gbase + row * row_bytes + (int64_t)part0 * 16;
            for (int c = 0; c < nch; ++c) {
                if (lane == 0) {
                    const int u0 = c * CU;
                    bulk_store(grow + (int64_t)u0 * 16, zero_page,
                               (uint32_t)min(CU, part_units - u0) * 16u);
                    bulk_commit();
                }
            }
            // the slots themselves are not read by those stores; earlier rows' stores are
            if (lane == 0) bulk_wait_read<0>();
            done_seq = seq0 + nch - 1;
            refill();
        } else {
            uint8_t* grow = gbase + row * row_bytes + (int64_t)part0 * 16;
            const float kk = fmaf(-lse, kLog2e, log2f(fabsf(ts.coef)));   // log2(|c| e^{-lse})
            const bool neg = ts.coef < 0.f;
            const uint32_t sign = neg ? 0x80008000u : 0u;
            // target entry: c (p_y - 1); patched by the lane that owns its 16-byte unit
            const int y_unit = y_unit1;
            const uint16_t gy_bits = __bfloat16_as_ushort(__float2bfloat16_rn(ts.gy));
            int stored = 0;   // chunks of this row already handed to the TMA store
            for (int ubase = 0; ubase < part_units; ubase += kRound) {
                const int uend = min(ubase + kRound, part_units);
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int u = ubase + k * 32 + lane;
                    if (u < part_units) {
                        int pos = start_unit + u; if (pos >= ring_units) pos -= ring_units;
                        const uint32_t addr = ring + (uint32_t)pos * 16u;
                        uint4 v = lds128(addr);
                        uint4 o;
                        o.x = pack_bf16x2(ex2_approx(fmaf(bf16_lo(v.x), kLog2e, kk)),
                                          ex2_approx(fmaf(bf16_hi(v.x), kLog2e, kk))) ^ sign;
                        o.y = pack_bf16x2(ex2_approx(fmaf(bf16_lo(v.y), kLog2e, kk)),
                                          ex2_approx(fmaf(bf16_hi(v.y), kLog2e, kk))) ^ sign;
                        o.z = pack_bf16x2(ex2_approx(fmaf(bf16_lo(v.z), kLog2e, kk)),
                                          ex2_approx(fmaf(bf16_hi(v.z), kLog2e, kk))) ^ sign;
                        o.w = pack_bf16x2(ex2_approx(fmaf(bf16_lo(v.w), kLog2e, kk)),
                                          ex2_approx(fmaf(bf16_hi(v.w), kLog2e, kk))) ^ sign;
                        sts128(addr, o);
                        if (u == y_unit)   // same thread, program order: overwrites its own store
                            asm volatile("st.shared.u16 [%0], %1;" ::"r"(addr + (uint32_t)(h.y & 7) * 2u),
                                         "h"(gy_bits) : "memory");
                    }
                }
                // hand every chunk that is now complete to the TMA store
                if ((stored + 1) * CU <= uend || uend == part_units) {
                    fence_proxy_async();
                    __syncwarp();
                    while (stored < nch && ((stored + 1) * CU <= uend || uend == part_units)) {
                        if (lane == 0) {
                            int s = slot0 + stored; if (s >= S) s -= S;
                            const int u0 = stored * CU;
                            bulk_store(grow + (int64_t)u0 * 16, ring + (uint32_t)(s * CU) * 16u,
                                       (uint32_t)min(CU, part_units - u0) * 16u);
                            bulk_commit();
                        }
                        ++stored;
                    }
                    // all but the newest store have been read out: their slots are free
                    if (lane == 0) bulk_wait_read<1>();
                    done_seq = seq0 + stored - 2;
                    refill();
                }
            }
            lazy_free = true;
        }

        seq0 += nch;
        slot0 += nch; while (slot0 >= S) slot0 -= S;
    }

    if (lane == 0) bulk_wait_all();   // gradient writes complete before the grid ends
    cluster_arrive();                 // peer may still be writing our stats block
    cluster_wait();
}

// ---------------------------------------------------------------- host side
static bool make_plan(int64_t V, int num_sms, int64_t n_tok, ClusterPlan& p) {
    const int units = (int)(V / 8);
    const int nparts = 2 * kCWarps;
    const int part_max = (units + nparts - 1) / nparts;
    if (part_max < kRound) return false;                 // small rows: generic kernel
    // choose CU (zero page = CU units) maximising prefetch depth  S*CU - part_max
    int best_cu = 0, best_s = 0, best_pref = -1;
    for (int cu = 48; cu <= 160; ++cu) {
        const int avail_units = (kSmemLimit - kCtrlBytes) / 16 - cu;     // minus zero page
        int s = avail_units / kCWarps / cu;
        if (s > kMaxSlots) s = kMaxSlots;
        const int nch = (part_max + cu - 1) / cu;
        if (s < nch + 1) continue;
        const int pref = s * cu - nch * cu;              // whole free slots while a row is resident
        if (pref > best_pref) { best_pref = pref; best_cu = cu; best_s = s; }
    }
    if (best_pref < 0) return false;                     // rows too long for a 2-CTA cluster
    p.units_per_row = units;
    p.chunk_units = best_cu;
    p.slots = best_s;
    int nc = num_sms / 2;
    if ((int64_t)nc > n_tok) nc = (int)n_tok;
    if (nc < 1) nc = 1;
    p.num_clusters = nc;
    return true;
}

bool rows_cluster_supported(int64_t V, int64_t ld, int dtype) {
    if (dtype != AWR_DTYPE_BF16) return false;
    if (V % 8 != 0 || ld % 8 != 0) return false;
    if (V / 8 > (1 << 24)) return false;
    ClusterPlan p;
    return make_plan(V, 2, 1, p);      // feasibility only: the SM count sets the grid, not the plan
}

cudaError_t launch_rows_cluster(const RowArgs& a, int num_sms, cudaStream_t st) {
    if (a.n_tok <= 0) return cudaSuccess;
    ClusterPlan p;
    if (!make_plan(a.V, num_sms, a.n_tok, p)) return cudaErrorInvalidValue;
    const int smem = kCtrlBytes + p.chunk_units * 16 + kCWarps * p.slots * p.chunk_units * 16;
    static PerDeviceInt attr_set;                    // the attribute is per device
    const int dev = PerDeviceInt::device();
    if (attr_set.get(dev) < 0) {
        cudaError_t e = cudaFuncSetAttribute(rows_cluster_kernel,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             kSmemLimit);
        if (e != cudaSuccess) return e;
        attr_set.set(dev, 1);
    }
    rows_cluster_kernel<<<2 * p.num_clusters, kCThreads, smem, st>>>(a, p);
    return cudaGetLastError();
}

}  // namespace awr
