// Internal launcher declarations (host side).  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

namespace awr {

struct RowArgs;

// One cached int per device ordinal (-1 = not set yet).  Function attributes
// (cudaFuncAttributeMaxDynamicSharedMemorySize) and occupancy answers belong to a DEVICE, not to
// the process: a process that drives several GPUs must set / query them on each.  Devices with an
// ordinal >= kMaxDevices are not cached (the setup simply runs on every call).
constexpr int kMaxDevices = 64;
struct PerDeviceInt {
    std::atomic<int> v[kMaxDevices];
    PerDeviceInt() { for (auto& x : v) x.store(-1, std::memory_order_relaxed); }
    static int device() {
        int d = 0;
        return (cudaGetDevice(&d) == cudaSuccess && d >= 0 && d < kMaxDevices) ? d : -1;
    }
    int get(int dev) const { return dev < 0 ? -1 : v[dev].load(std::memory_order_acquire); }
    void set(int dev, int x) { if (dev >= 0) v[dev].store(x, std::memory_order_release); }
};

cudaError_t launch_segment_expand(const int32_t* step_off, const int32_t* traj_off,
                                  const int32_t* group_off, int64_t n_tok, int n_steps,
                                  int n_traj, int n_groups, int32_t* tok_traj, uint32_t* err,
                                  int num_sms, cudaStream_t st);
cudaError_t launch_group_advantage(const float* rewards, const int32_t* group_off,
                                   const int32_t* traj_off, int n_groups, int n_traj,
                                   uint32_t flags, int normalizer, float k_norm,
                                   float loss_scale, float* adv, float* traj_scale,
                                   uint32_t* n_mixed /* zeroed scratch word, nullable */,
                                   cudaStream_t st);
cudaError_t launch_final_reduce(const float* tok_term, const uint8_t* tok_flag, int64_t n_tok,
                                float* loss, int64_t* clip_count, int64_t* dual_count,
                                cudaStream_t st);

// a2 + a3 + a4, one CTA per row, any V / dtype (second pass re-reads the row through L2).
cudaError_t launch_rows_generic(const RowArgs& a, int dtype, int num_sms, cudaStream_t st);

// a2 + a3 + a4, bf16 rows resident in the shared memory of a 2-CTA cluster (TMA bulk copies).
bool rows_cluster_supported(int64_t V, int64_t ld, int dtype);
cudaError_t launch_rows_cluster(const RowArgs& a, int num_sms, cudaStream_t st);

// a2 + a3 + a4, bf16 rows resident in the register files of a 2-CTA cluster; shared memory is a
// TMA load FIFO, gradient written with coalesced 16-byte stores.
bool rows_rf_supported(int64_t V, int64_t ld, int dtype);
cudaError_t launch_rows_rf(const RowArgs& a, int num_sms, int cluster_size, cudaStream_t st);

// a2 + a3 + a4, the register-file design with a service warp per CTA (awr_rows_rfs.cu): whole-slot
// TMA loads, staged TMA gradient stores, st.async exchange, a3 on the service warp.
bool rows_rfs_supported(int64_t V, int64_t ld, int dtype);
cudaError_t launch_rows_rfs(const RowArgs& a, int num_sms, bool early_stats, cudaStream_t st);

// a2 + a3 forward only (awr_loss_fwd), bf16 rows streamed once through a TMA-filled ring; no
// gradient, no row residency (awr_rows_fwd.cu).
bool rows_fwd_supported(int64_t V, int64_t ld, int dtype);
cudaError_t launch_rows_fwd(const RowArgs& a, int num_sms, cudaStream_t st);

// a5: fused LM head (awr_head.cu).  `rows` carries the per-token inputs / outputs of a3
// (its logits / dlogits members are unused); `ws` is head_ws_bytes() of device memory.
constexpr int64_t kHeadPanelRows = 4736;   // 37 row tiles of 128; doubled for CTA pairs (awr_head.cu)
struct HeadCall {
    const void* hidden;
    const void* w_head;
    int w_layout;
    int64_t n_tok, V, K;
    const RowArgs* rows;
    void* dhidden;
    void* dw_head;
    void* ws;
    int ctas;        // 1: cta_group::1 tiles of 128 rows; anything else: CTA pairs, 256-row tiles
    int mode;        // kHead*
};
enum { kHeadRecompute = 0,  // the logits tile is recomputed for dS (8 K V flops / token)
       kHeadStored32 = 1,   // the fp32 logits of a row panel are kept (two buffers, side stream); dS in
                            // a streaming pass (6 K V); same bits as recompute
       kHeadE16 = 2,        // the forward epilogue keeps E = bf16(exp(z - tile max)) IN the dS panel; one
                            // in-place pass rescales it to dS (6 K V; 2 bytes per logit of transient)
       kHeadRowRef = 3 };   // E = bf16(exp(z - zref_row)) with a per-row reference known before the GEMM
                            // (an estimate of the target logit): dS = E f_row, the scale applied by the
                            // dhidden epilogue and folded into the H operand of dw_head - no dS pass
size_t head_ws_bytes(int64_t n_tok, int64_t V, int64_t K, int ctas, int mode);
int head_launches(int64_t n_tok, int64_t V, int64_t K, int ctas, int mode);
cudaError_t launch_head(const HeadCall& c, int num_sms, cudaStream_t st);
// C[M, N] (bf16, row-major, ldc) = A B on the tcgen05 engine; majors: 0 = contraction index
// contiguous, 1 = row (A) / column (B) index contiguous.
cudaError_t launch_gemm_bf16(const void* A, int a_major, int64_t lda, const void* B, int b_major,
                             int64_t ldb, int64_t M, int64_t N, int64_t Kc, void* C, int64_t ldc,
                             int num_sms, int ctas, cudaStream_t st);

}  // namespace awr
