// C-ABI entry points of libawr.so (include/awr.h): argument checks, workspace layout, launch
// sequencing.  Every step of the path runs in the kernels; nothing here computes.
#include <math.h>
#include <string.h>

#include "awr_common.cuh"
#include "awr_kernels.h"

namespace awr {

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct DeviceInfo {
    int major = -1;
    int num_sms = 0;
};

static cudaError_t device_info(DeviceInfo& info) {
    static DeviceInfo cache[64];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64 && cache[dev].major >= 0) { info = cache[dev]; return cudaSuccess; }
    DeviceInfo d;
    e = cudaDeviceGetAttribute(&d.major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&d.num_sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64) cache[dev] = d;
    info = d;
    return cudaSuccess;
}

// Device workspace of awr_loss_fwd_bwd / awr_loss_fwd.
struct Workspace {
    uint32_t* err;
    float* adv;
    float* traj_scale;
    int32_t* tok_traj;
    float* tok_term;
    uint8_t* tok_flag;
    size_t zero_bytes;   // [err, adv, traj_scale] prefix that is memset to 0
    size_t total;
};

static Workspace carve(void* base, int64_t n_tok, int32_t n_traj) {
    Workspace w;
    uint8_t* p = reinterpret_cast<uint8_t*>(base);
    size_t off = 0;
    w.err = reinterpret_cast<uint32_t*>(p + off); off += 256;
    w.adv = reinterpret_cast<float*>(p + off); off += align_up((size_t)n_traj * 4, 256);
    w.traj_scale = reinterpret_cast<float*>(p + off); off += align_up((size_t)n_traj * 4, 256);
    w.zero_bytes = off;
    w.tok_traj = reinterpret_cast<int32_t*>(p + off); off += align_up((size_t)n_tok * 4, 256);
    w.tok_term = reinterpret_cast<float*>(p + off); off += align_up((size_t)n_tok * 4, 256);
    w.tok_flag = reinterpret_cast<uint8_t*>(p + off); off += align_up((size_t)n_tok, 256);
    w.total = off;
    return w;
}

static int check_params(const awr_params* p) {
    if (!(p->k_norm > 0.f) || !isfinite(p->k_norm)) return AWR_ERR_PARAM;
    if (!(p->clip_eps >= 0.f && p->clip_eps < 1.f)) return AWR_ERR_PARAM;
    if (isnan(p->stale_cap)) return AWR_ERR_PARAM;
    if (!isfinite(p->loss_scale)) return AWR_ERR_PARAM;
    if (isnan(p->dual_clip_c)) return AWR_ERR_PARAM;          // Eq. (2): > 1 = on, <= 1 = off
    if (p->normalizer != AWR_NORM_CONST_K && p->normalizer != AWR_NORM_PER_TRAJ) return AWR_ERR_PARAM;
    if (p->flags & ~(uint32_t)(AWR_FLAG_SAMPLE_STD | AWR_FLAG_SUCCESS_FILTER | AWR_FLAG_COUPLED |
                               AWR_FLAG_SKIP_UNIFORM))
        return AWR_ERR_PARAM;
    if (p->kernel < AWR_KERNEL_AUTO || p->kernel > AWR_KERNEL_CLUSTER_RFS_LATE) return AWR_ERR_PARAM;
    return AWR_OK;
}

static int check_segments(int64_t n_tok, int32_t n_steps, int32_t n_traj, int32_t n_groups) {
    if (n_tok < 0 || n_steps < 0 || n_traj < 0 || n_groups < 0) return AWR_ERR_SHAPE;
    if (n_tok > 0x7fffffffLL) return AWR_ERR_SHAPE;            // offsets are int32
    return AWR_OK;
}

// fused-head entry points: which tcgen05 shape (CTAs per tile) a kernel request means, or -1
static int resolve_head_ctas(int requested) {
    if (requested == AWR_KERNEL_AUTO || requested == AWR_KERNEL_HEAD_2CTA ||
        requested == AWR_KERNEL_HEAD_2CTA_STORED || requested == AWR_KERNEL_HEAD_2CTA_E16 ||
        requested == AWR_KERNEL_HEAD_2CTA_ROWREF) return 2;
    if (requested == AWR_KERNEL_HEAD_1CTA) return 1;
    return -1;
}
static int resolve_head_mode(int requested) {
    if (requested == AWR_KERNEL_AUTO || requested == AWR_KERNEL_HEAD_2CTA_ROWREF) return kHeadRowRef;
    if (requested == AWR_KERNEL_HEAD_2CTA_E16) return kHeadE16;
    return requested == AWR_KERNEL_HEAD_2CTA_STORED ? kHeadStored32 : kHeadRecompute;
}

static int resolve_kernel(int requested, int64_t V, int64_t ld, int dtype, bool want_entropy = false,
                          bool backward = true) {
    if (requested == AWR_KERNEL_FWD_STREAM)                   // forward only, bf16, 16-byte units
        return (!backward && rows_fwd_supported(V, ld, dtype)) ? AWR_KERNEL_FWD_STREAM : -1;
    if (requested == AWR_KERNEL_CLUSTER_RFS || requested == AWR_KERNEL_CLUSTER_RFS_LATE)
        return rows_rfs_supported(V, ld, dtype) ? requested : -1;
    if (requested > AWR_KERNEL_CLUSTER_RF4) return -1;        // a fused-head kernel id
    // forward only: nothing has to stay on chip for a second pass, so whole rows are streamed
    // (config 1: see DESIGN.md section 4 for the measured rates of all the kernels on this path)
    if (!backward && requested == AWR_KERNEL_AUTO && V * 2 >= 65536 && rows_fwd_supported(V, ld, dtype))
        return AWR_KERNEL_FWD_STREAM;
    // token_entropy is produced by the generic and the register-file kernels
    if (want_entropy && requested == AWR_KERNEL_CLUSTER) return -1;
    if (want_entropy && requested == AWR_KERNEL_AUTO && V * 2 >= 65536 && !rows_rf_supported(V, ld, dtype) &&
        !rows_rfs_supported(V, ld, dtype))
        return AWR_KERNEL_GENERIC;
    const bool ok = rows_cluster_supported(V, ld, dtype);
    const bool ok_rf = rows_rf_supported(V, ld, dtype);
    if (requested == AWR_KERNEL_CLUSTER) return ok ? AWR_KERNEL_CLUSTER : -1;
    if (requested == AWR_KERNEL_CLUSTER_RF) return ok_rf ? AWR_KERNEL_CLUSTER_RF : -1;
    if (requested == AWR_KERNEL_CLUSTER_RF4) return ok_rf ? AWR_KERNEL_CLUSTER_RF4 : -1;
    if (requested == AWR_KERNEL_GENERIC) return AWR_KERNEL_GENERIC;
    // auto: the cluster kernels pay off once a row is a sizeable fraction of shared memory
    if (V * 2 < 65536) return AWR_KERNEL_GENERIC;
    if (rows_rfs_supported(V, ld, dtype)) return AWR_KERNEL_CLUSTER_RFS;
    if (ok_rf) return AWR_KERNEL_CLUSTER_RF;
    return ok ? AWR_KERNEL_CLUSTER : AWR_KERNEL_GENERIC;
}

static cudaError_t launch_rows(int kernel, const RowArgs& a, int dtype, int num_sms,
                               cudaStream_t st) {
    if (kernel == AWR_KERNEL_FWD_STREAM) return launch_rows_fwd(a, num_sms, st);
    if (kernel == AWR_KERNEL_CLUSTER_RFS) return launch_rows_rfs(a, num_sms, /*early_stats=*/true, st);
    if (kernel == AWR_KERNEL_CLUSTER_RFS_LATE) return launch_rows_rfs(a, num_sms, /*early_stats=*/false, st);
    if (kernel == AWR_KERNEL_CLUSTER_RF) return launch_rows_rf(a, num_sms, 2, st);
    if (kernel == AWR_KERNEL_CLUSTER_RF4) return launch_rows_rf(a, num_sms, 4, st);
    if (kernel == AWR_KERNEL_CLUSTER) return launch_rows_cluster(a, num_sms, st);
    return launch_rows_generic(a, dtype, num_sms, st);
}

static int run(const awr_batch* b, const awr_params* p, const awr_outputs* o, void* ws_ptr,
               size_t ws_bytes, void* stream, bool backward) {
    if (!b || !p || !o) return AWR_ERR_NULL;
    int rc = check_segments(b->n_tok, b->n_steps, b->n_traj, b->n_groups);
    if (rc) return rc;
    if (b->V <= 0 || b->ld < b->V) return AWR_ERR_SHAPE;
    if (b->logits_dtype != AWR_DTYPE_BF16 && b->logits_dtype != AWR_DTYPE_F32) return AWR_ERR_DTYPE;
    rc = check_params(p);
    if (rc) return rc;
    if (!o->loss || !o->clip_count) return AWR_ERR_NULL;
    if (b->n_tok > 0 && (!o->token_lp || (backward && !o->dlogits))) return AWR_ERR_NULL;
    if (!b->step_off || !b->traj_off || !b->group_off) return AWR_ERR_NULL;
    const bool coupled = (p->flags & AWR_FLAG_COUPLED) != 0;      // prox_lp is not read (:114)
    if (b->n_tok > 0 && (!b->logits || !b->target_ids || !b->behave_lp || (!coupled && !b->prox_lp)))
        return AWR_ERR_NULL;
    if (b->n_traj > 0 && !b->rewards) return AWR_ERR_NULL;
    if ((o->ev_row_begin == nullptr) != (o->ev_row_end == nullptr)) return AWR_ERR_NULL;
    const size_t esz = b->logits_dtype == AWR_DTYPE_BF16 ? 2 : 4;
    if ((reinterpret_cast<uintptr_t>(b->logits) & 15) || ((size_t)b->ld * esz) % 16) return AWR_ERR_ALIGN;
    if (backward && (reinterpret_cast<uintptr_t>(o->dlogits) & 15)) return AWR_ERR_ALIGN;
    const size_t need = awr_workspace_bytes(b->n_tok, b->V, b->n_steps, b->n_traj, b->n_groups);
    if (!ws_ptr || (reinterpret_cast<uintptr_t>(ws_ptr) & 255) || ws_bytes < need) return AWR_ERR_WORKSPACE;
    const int kernel = resolve_kernel(p->kernel, b->V, b->ld, b->logits_dtype, o->token_entropy != nullptr,
                                      backward);
    if (kernel < 0) return AWR_ERR_PARAM;

    DeviceInfo info;
    if (device_info(info) != cudaSuccess) { cudaGetLastError(); return AWR_ERR_CUDA; }
    if (info.major != 10) return AWR_ERR_ARCH;

    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    Workspace w = carve(ws_ptr, b->n_tok, b->n_traj);
    uint32_t* err = o->err_word ? o->err_word : w.err;
    float* adv = o->adv ? o->adv : w.adv;
    int32_t* tok_traj = o->tok_traj ? o->tok_traj : w.tok_traj;
    float* tok_term = o->tok_term ? o->tok_term : w.tok_term;

    cudaError_t e = cudaMemsetAsync(ws_ptr, 0, w.zero_bytes, st);
    if (e == cudaSuccess && o->err_word) e = cudaMemsetAsync(o->err_word, 0, 4, st);
    if (e == cudaSuccess && o->adv && b->n_traj > 0) e = cudaMemsetAsync(o->adv, 0, (size_t)b->n_traj * 4, st);
    // a0
    if (e == cudaSuccess)
        e = launch_segment_expand(b->step_off, b->traj_off, b->group_off, b->n_tok, b->n_steps,
                                  b->n_traj, b->n_groups, tok_traj, err, info.num_sms, st);
    // a1 (+ O6 scale)
    if (e == cudaSuccess)
        e = launch_group_advantage(b->rewards, b->group_off, b->traj_off, b->n_groups, b->n_traj,
                                   p->flags, p->normalizer, p->k_norm, p->loss_scale, adv,
                                   w.traj_scale, w.err + 1, st);
    // a2 + a3 + a4
    RowArgs a;
    a.logits = b->logits;
    a.dlogits = backward ? o->dlogits : nullptr;
    a.n_tok = b->n_tok; a.V = b->V; a.ld = b->ld;
    a.target_ids = b->target_ids; a.behave_lp = b->behave_lp;
    a.prox_lp = (p->flags & AWR_FLAG_COUPLED) ? b->behave_lp : b->prox_lp;
    a.tok_traj = tok_traj; a.adv = adv; a.traj_scale = w.traj_scale;
    a.token_lp = o->token_lp; a.tok_term = tok_term; a.tok_coef = o->tok_coef;
    a.target_logit = o->target_logit; a.tok_flag = w.tok_flag; a.err_word = err;
    a.token_entropy = o->token_entropy;
    a.clip_eps = p->clip_eps; a.stale_cap = p->stale_cap; a.dual_c = p->dual_clip_c;
    // optional measurement events of THIS call (no library state): around the row kernel only
    cudaEvent_t ev0 = reinterpret_cast<cudaEvent_t>(o->ev_row_begin);
    cudaEvent_t ev1 = reinterpret_cast<cudaEvent_t>(o->ev_row_end);
    if (e == cudaSuccess && ev0) e = cudaEventRecord(ev0, st);
    if (e == cudaSuccess) {
        e = launch_rows(kernel, a, b->logits_dtype, info.num_sms, st);
    }
    if (e == cudaSuccess && ev1) e = cudaEventRecord(ev1, st);
    // a3 final reduction
    if (e == cudaSuccess) e = launch_final_reduce(tok_term, w.tok_flag, b->n_tok, o->loss, o->clip_count,
                                                    o->dual_clip_count, st);
    if (e != cudaSuccess) { cudaGetLastError(); return AWR_ERR_CUDA; }
    return AWR_OK;
}

// ---------------------------------------------------------------- no-allocation entry point
// Scratch of awr_loss_fwd_bwd_static: one fixed array per GPU that loads the library.  In host code
// the name is only a handle of the symbol, not a device address: the address comes from
// cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned char g_static_ws[AWR_STATIC_WS_BYTES];

static int static_workspace(void** out) {
    constexpr int kMax = 64;
    static void* cache[kMax];                 // per device ordinal; written once with one value
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return AWR_ERR_CUDA; }
    void* ptr = (dev >= 0 && dev < kMax) ? __atomic_load_n(&cache[dev], __ATOMIC_ACQUIRE) : nullptr;
    if (!ptr) {
        const cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_ws);
        if (e != cudaSuccess || !ptr) { cudaGetLastError(); return AWR_ERR_CUDA; }
        if (dev >= 0 && dev < kMax) __atomic_store_n(&cache[dev], ptr, __ATOMIC_RELEASE);
    }
    *out = ptr;
    return AWR_OK;
}

}  // namespace awr

using namespace awr;

extern "C" {

int awr_version(void) { return AWR_VERSION; }

const char* awr_status_string(int s) {
    switch (s) {
        case AWR_OK: return "ok";
        case AWR_ERR_NULL: return "required pointer is NULL";
        case AWR_ERR_SHAPE: return "bad sizes";
        case AWR_ERR_DTYPE: return "unknown dtype or layout";
        case AWR_ERR_ALIGN: return "rows must start on 16-byte boundaries";
        case AWR_ERR_PARAM: return "parameter out of range";
        case AWR_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
        case AWR_ERR_ARCH: return "device is not sm_100 (B200); no fallback exists";
        case AWR_ERR_CUDA: return "CUDA runtime error";
        case AWR_ERR_STATIC_LIMIT:
            return "batch needs more scratch than AWR_STATIC_WS_BYTES (1 MiB): use awr_loss_fwd_bwd with a workspace";
        default: return "unknown status";
    }
}

size_t awr_workspace_bytes(int64_t n_tok, int64_t V, int32_t n_steps, int32_t n_traj,
                           int32_t n_groups) {
    (void)V; (void)n_steps; (void)n_groups;
    if (n_tok < 0 || n_traj < 0) return 0;
    return carve(nullptr, n_tok, n_traj).total;
}

int awr_select_kernel(int64_t V, int64_t ld, int32_t logits_dtype) {
    return resolve_kernel(AWR_KERNEL_AUTO, V, ld, logits_dtype);
}

int awr_launches_per_call(void) { return 4; }

int awr_loss_fwd_bwd(const awr_batch* batch, const awr_params* params, const awr_outputs* out,
                     void* workspace, size_t workspace_bytes, void* stream) {
    return run(batch, params, out, workspace, workspace_bytes, stream, true);
}

int awr_loss_fwd_bwd_static(const awr_batch* batch, const awr_params* params, const awr_outputs* out,
                            void* stream) {
    if (!batch || !params || !out) return AWR_ERR_NULL;
    const int rc = check_segments(batch->n_tok, batch->n_steps, batch->n_traj, batch->n_groups);
    if (rc) return rc;
    if (awr_workspace_bytes(batch->n_tok, batch->V, batch->n_steps, batch->n_traj, batch->n_groups) >
        AWR_STATIC_WS_BYTES)
        return AWR_ERR_STATIC_LIMIT;
    void* ws = nullptr;
    const int rs = static_workspace(&ws);
    if (rs) return rs;
    // run() clears the zero-initialised prefix of the workspace on `stream` before anything reads it
    return run(batch, params, out, ws, AWR_STATIC_WS_BYTES, stream, true);
}

int awr_loss_fwd(const awr_batch* batch, const awr_params* params, const awr_outputs* out,
                 void* workspace, size_t workspace_bytes, void* stream) {
    return run(batch, params, out, workspace, workspace_bytes, stream, false);
}

int awr_group_advantage(const float* rewards, const int32_t* group_off, int32_t n_groups,
                        int32_t n_traj, uint32_t flags, float* adv, void* stream) {
    if (n_groups < 0 || n_traj < 0) return AWR_ERR_SHAPE;
    if (flags & ~(uint32_t)AWR_FLAG_SAMPLE_STD) return AWR_ERR_PARAM;
    if (!group_off || (n_traj > 0 && (!rewards || !adv))) return AWR_ERR_NULL;
    DeviceInfo info;
    if (device_info(info) != cudaSuccess) { cudaGetLastError(); return AWR_ERR_CUDA; }
    if (info.major != 10) return AWR_ERR_ARCH;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    cudaError_t e = cudaSuccess;
    if (n_traj > 0) e = cudaMemsetAsync(adv, 0, (size_t)n_traj * 4, st);
    if (e == cudaSuccess)
        e = launch_group_advantage(rewards, group_off, nullptr, n_groups, n_traj, flags,
                                   AWR_NORM_CONST_K, 1.f, 1.f, adv, nullptr, nullptr, st);
    if (e != cudaSuccess) { cudaGetLastError(); return AWR_ERR_CUDA; }
    return AWR_OK;
}

// ------------------------------------------------------------------ a5: fused LM head
size_t awr_head_workspace_bytes(int64_t n_tok, int64_t V, int64_t K, int32_t n_steps,
                                int32_t n_traj, int32_t n_groups, int32_t kernel) {
    (void)n_steps; (void)n_groups;
    if (n_tok < 0 || n_traj < 0 || V <= 0 || K <= 0 || resolve_head_ctas(kernel) < 0) return 0;
    return carve(nullptr, n_tok, n_traj).total +
           head_ws_bytes(n_tok, V, K, resolve_head_ctas(kernel), resolve_head_mode(kernel));
}

int awr_head_launches_per_call(int64_t n_tok, int64_t V, int64_t K, int32_t kernel) {
    const int ctas = resolve_head_ctas(kernel);
    if (ctas < 0) return AWR_ERR_PARAM;
    return 3 + head_launches(n_tok, V, K, ctas, resolve_head_mode(kernel));     // a0, a1, [F, scalars, 3 per panel], final sum
}

int awr_loss_fwd_bwd_fused_head(const awr_head_batch* b, const awr_params* p,
                                const awr_head_outputs* o, void* ws_ptr, size_t ws_bytes,
                                void* stream) {
    if (!b || !p || !o) return AWR_ERR_NULL;
    int rc = check_segments(b->n_tok, b->n_steps, b->n_traj, b->n_groups);
    if (rc) return rc;
    if (b->V <= 0 || b->K <= 0 || b->V % 8 != 0 || b->K % 64 != 0) return AWR_ERR_SHAPE;
    if (b->V > 0x7fffffffLL || b->K > 0x7fffffffLL) return AWR_ERR_SHAPE;
    if (b->w_layout != AWR_W_K_BY_V && b->w_layout != AWR_W_V_BY_K) return AWR_ERR_DTYPE;
    rc = check_params(p);
    if (rc) return rc;
    if (resolve_head_ctas(p->kernel) < 0) return AWR_ERR_PARAM;
    if (!o->loss || !o->clip_count || !o->dw_head) return AWR_ERR_NULL;
    if (b->n_tok > 0 && (!o->token_lp || !o->dhidden)) return AWR_ERR_NULL;
    if (!b->step_off || !b->traj_off || !b->group_off || !b->w_head) return AWR_ERR_NULL;
    if (b->n_tok > 0 && (!b->hidden || !b->target_ids || !b->behave_lp ||
                         (!(p->flags & AWR_FLAG_COUPLED) && !b->prox_lp))) return AWR_ERR_NULL;
    if (b->n_traj > 0 && !b->rewards) return AWR_ERR_NULL;
    if ((reinterpret_cast<uintptr_t>(b->hidden) & 15) || (reinterpret_cast<uintptr_t>(b->w_head) & 15) ||
        (reinterpret_cast<uintptr_t>(o->dhidden) & 15) || (reinterpret_cast<uintptr_t>(o->dw_head) & 15))
        return AWR_ERR_ALIGN;
    const size_t need = awr_head_workspace_bytes(b->n_tok, b->V, b->K, b->n_steps, b->n_traj, b->n_groups,
                                                 p->kernel);
    if (!ws_ptr || (reinterpret_cast<uintptr_t>(ws_ptr) & 255) || ws_bytes < need) return AWR_ERR_WORKSPACE;
    DeviceInfo info;
    if (device_info(info) != cudaSuccess) { cudaGetLastError(); return AWR_ERR_CUDA; }
    if (info.major != 10) return AWR_ERR_ARCH;

    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    Workspace w = carve(ws_ptr, b->n_tok, b->n_traj);
    uint32_t* err = o->err_word ? o->err_word : w.err;
    float* adv = o->adv ? o->adv : w.adv;
    int32_t* tok_traj = o->tok_traj ? o->tok_traj : w.tok_traj;
    float* tok_term = o->tok_term ? o->tok_term : w.tok_term;

    cudaError_t e = cudaMemsetAsync(ws_ptr, 0, w.zero_bytes, st);
    if (e == cudaSuccess && o->err_word) e = cudaMemsetAsync(o->err_word, 0, 4, st);
    if (e == cudaSuccess && o->adv && b->n_traj > 0) e = cudaMemsetAsync(o->adv, 0, (size_t)b->n_traj * 4, st);
    if (e == cudaSuccess)
        e = launch_segment_expand(b->step_off, b->traj_off, b->group_off, b->n_tok, b->n_steps,
                                  b->n_traj, b->n_groups, tok_traj, err, info.num_sms, st);
    if (e == cudaSuccess)
        e = launch_group_advantage(b->rewards, b->group_off, b->traj_off, b->n_groups, b->n_traj,
                                   p->flags, p->normalizer, p->k_norm, p->loss_scale, adv,
                                   w.traj_scale, w.err + 1, st);
    RowArgs a = {};
    a.n_tok = b->n_tok; a.V = b->V; a.ld = b->V;
    a.target_ids = b->target_ids; a.behave_lp = b->behave_lp;
    a.prox_lp = (p->flags & AWR_FLAG_COUPLED) ? b->behave_lp : b->prox_lp;
    a.tok_traj = tok_traj; a.adv = adv; a.traj_scale = w.traj_scale;
    a.token_lp = o->token_lp; a.tok_term = tok_term; a.tok_coef = o->tok_coef;
    a.target_logit = nullptr; a.tok_flag = w.tok_flag; a.err_word = err;
    a.token_entropy = o->token_entropy;
    a.clip_eps = p->clip_eps; a.stale_cap = p->stale_cap; a.dual_c = p->dual_clip_c;
    HeadCall c;
    c.hidden = b->hidden; c.w_head = b->w_head; c.w_layout = b->w_layout;
    c.n_tok = b->n_tok; c.V = b->V; c.K = b->K; c.rows = &a;
    c.dhidden = o->dhidden; c.dw_head = o->dw_head;
    c.ws = reinterpret_cast<uint8_t*>(ws_ptr) + w.total;
    c.ctas = resolve_head_ctas(p->kernel);
    c.mode = resolve_head_mode(p->kernel);
    if (e == cudaSuccess) e = launch_head(c, info.num_sms, st);
    if (e == cudaSuccess) e = launch_final_reduce(tok_term, w.tok_flag, b->n_tok, o->loss, o->clip_count,
                                                    o->dual_clip_count, st);
    if (e != cudaSuccess) { cudaGetLastError(); return AWR_ERR_CUDA; }
    return AWR_OK;
}

int awr_gemm_bf16(const void* A, int32_t a_major, int64_t lda, const void* B, int32_t b_major,
                  int64_t ldb, int64_t M, int64_t N, int64_t Kc, void* C, int64_t ldc, int32_t kernel,
                  void* stream) {
    if (!A || !B || !C) return AWR_ERR_NULL;
    const int ctas = resolve_head_ctas(kernel);
    if (ctas < 0) return AWR_ERR_PARAM;
    if (M <= 0 || N <= 0 || Kc <= 0 || M > 0x7fffffffLL || N > 0x7fffffffLL || Kc > 0x7fffffffLL) return AWR_ERR_SHAPE;
    if ((a_major != 0 && a_major != 1) || (b_major != 0 && b_major != 1)) return AWR_ERR_DTYPE;
    if (lda % 8 || ldb % 8 || ldc % 8 || N % 8) return AWR_ERR_ALIGN;
    if ((reinterpret_cast<uintptr_t>(A) & 15) || (reinterpret_cast<uintptr_t>(B) & 15) ||
        (reinterpret_cast<uintptr_t>(C) & 15)) return AWR_ERR_ALIGN;
    DeviceInfo info;
    if (device_info(info) != cudaSuccess) { cudaGetLastError(); return AWR_ERR_CUDA; }
    if (info.major != 10) return AWR_ERR_ARCH;
    cudaError_t e = launch_gemm_bf16(A, a_major, lda, B, b_major, ldb, M, N, Kc, C, ldc, info.num_sms,
                                     ctas, reinterpret_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) { cudaGetLastError(); return AWR_ERR_CUDA; }
    return AWR_OK;
}

// ------------------------------------------------------------------ a5 with HOST buffers
namespace {
struct HeadHostPlan {
    size_t hidden, w, dh, dw, tok, steps, traj, groups, rew, adv, total_small, head_ws, total;
};
HeadHostPlan head_host_plan(int64_t n_tok, int64_t V, int64_t K, int32_t n_steps, int32_t n_traj,
                            int32_t n_groups, int32_t kernel) {
    HeadHostPlan h;
    h.hidden = align_up((size_t)n_tok * K * 2, 256);
    h.w = align_up((size_t)K * V * 2, 256);
    h.dh = h.hidden;
    h.dw = h.w;
    h.tok = align_up((size_t)n_tok * 4, 256);
    h.steps = align_up((size_t)(n_steps + 1) * 4, 256);
    h.traj = align_up((size_t)(n_traj + 1) * 4, 256);
    h.groups = align_up((size_t)(n_groups + 1) * 4, 256);
    h.rew = align_up((size_t)n_traj * 4, 256);
    h.adv = h.rew;
    // ids, b, q in; lp, term, coef, tok_traj, entropy out; offsets; rewards; adv; scalars
    h.total_small = 8 * h.tok + h.steps + h.traj + h.groups + h.rew + h.adv + 256;
    h.head_ws = awr_head_workspace_bytes(n_tok, V, K, n_steps, n_traj, n_groups, kernel);
    h.total = h.hidden + h.w + h.dh + h.dw + h.total_small + h.head_ws;
    return h;
}
}  // namespace

size_t awr_head_host_workspace_bytes(int64_t n_tok, int64_t V, int64_t K, int32_t n_steps,
                                     int32_t n_traj, int32_t n_groups, int32_t kernel) {
    if (n_tok < 0 || V <= 0 || K <= 0 || n_steps < 0 || n_traj < 0 || n_groups < 0) return 0;
    if (resolve_head_ctas(kernel) < 0) return 0;
    return head_host_plan(n_tok, V, K, n_steps, n_traj, n_groups, kernel).total;
}

int awr_loss_fwd_bwd_fused_head_host(const awr_head_batch* hb, const awr_params* p,
                                     const awr_head_outputs* ho, void* dev_ws, size_t dev_ws_bytes,
                                     void* stream) {
    if (!hb || !p || !ho) return AWR_ERR_NULL;
    int rc = check_segments(hb->n_tok, hb->n_steps, hb->n_traj, hb->n_groups);
    if (rc) return rc;
    if (hb->V <= 0 || hb->K <= 0 || hb->V % 8 != 0 || hb->K % 64 != 0) return AWR_ERR_SHAPE;
    rc = check_params(p);
    if (rc) return rc;
    const bool coupled = (p->flags & AWR_FLAG_COUPLED) != 0;
    if (!ho->loss || !ho->clip_count || !ho->dw_head) return AWR_ERR_NULL;
    if (hb->n_tok > 0 && (!ho->token_lp || !ho->dhidden)) return AWR_ERR_NULL;
    if (!hb->step_off || !hb->traj_off || !hb->group_off || !hb->w_head) return AWR_ERR_NULL;
    if (hb->n_tok > 0 && (!hb->hidden || !hb->target_ids || !hb->behave_lp || (!coupled && !hb->prox_lp)))
        return AWR_ERR_NULL;
    if (hb->n_traj > 0 && !hb->rewards) return AWR_ERR_NULL;
    if (resolve_head_ctas(p->kernel) < 0) return AWR_ERR_PARAM;
    const HeadHostPlan hp = head_host_plan(hb->n_tok, hb->V, hb->K, hb->n_steps, hb->n_traj, hb->n_groups,
                                           p->kernel);
    if (!dev_ws || (reinterpret_cast<uintptr_t>(dev_ws) & 255) || dev_ws_bytes < hp.total) return AWR_ERR_WORKSPACE;

    const int64_t n = hb->n_tok;
    uint8_t* base = reinterpret_cast<uint8_t*>(dev_ws);
    size_t off = 0;
    auto take = [&](size_t bytes) { void* r = base + off; off += bytes; return r; };
    void* d_h = take(hp.hidden);
    void* d_w = take(hp.w);
    void* d_dh = take(hp.dh);
    void* d_dw = take(hp.dw);
    int32_t* d_ids = (int32_t*)take(hp.tok);
    float* d_b = (float*)take(hp.tok);
    float* d_q = (float*)take(hp.tok);
    float* d_lp = (float*)take(hp.tok);
    float* d_term = (float*)take(hp.tok);
    float* d_coef = (float*)take(hp.tok);
    int32_t* d_tt = (int32_t*)take(hp.tok);
    float* d_ent = (float*)take(hp.tok);
    int32_t* d_so = (int32_t*)take(hp.steps);
    int32_t* d_to = (int32_t*)take(hp.traj);
    int32_t* d_go = (int32_t*)take(hp.groups);
    float* d_rw = (float*)take(hp.rew);
    float* d_adv = (float*)take(hp.adv);
    uint8_t* d_scal = (uint8_t*)take(256);
    void* d_headws = base + off;

    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const cudaMemcpyKind H2D = cudaMemcpyHostToDevice, D2H = cudaMemcpyDeviceToHost;
    cudaError_t e = cudaSuccess;
#define AWR_TRY(x) do { if (e == cudaSuccess) e = (x); } while (0)
    AWR_TRY(cudaMemcpyAsync(d_w, hb->w_head, (size_t)hb->K * hb->V * 2, H2D, st));
    if (n > 0) {
        AWR_TRY(cudaMemcpyAsync(d_h, hb->hidden, (size_t)n * hb->K * 2, H2D, st));
        AWR_TRY(cudaMemcpyAsync(d_ids, hb->target_ids, (size_t)n * 4, H2D, st));
        AWR_TRY(cudaMemcpyAsync(d_b, hb->behave_lp, (size_t)n * 4, H2D, st));
        if (!coupled) AWR_TRY(cudaMemcpyAsync(d_q, hb->prox_lp, (size_t)n * 4, H2D, st));
    }
    AWR_TRY(cudaMemcpyAsync(d_so, hb->step_off, (size_t)(hb->n_steps + 1) * 4, H2D, st));
    AWR_TRY(cudaMemcpyAsync(d_to, hb->traj_off, (size_t)(hb->n_traj + 1) * 4, H2D, st));
    AWR_TRY(cudaMemcpyAsync(d_go, hb->group_off, (size_t)(hb->n_groups + 1) * 4, H2D, st));
    if (hb->n_traj > 0) AWR_TRY(cudaMemcpyAsync(d_rw, hb->rewards, (size_t)hb->n_traj * 4, H2D, st));
    if (e != cudaSuccess) { cudaGetLastError(); return AWR_ERR_CUDA; }

    awr_head_batch db = *hb;
    db.hidden = d_h; db.w_head = d_w; db.target_ids = d_ids; db.behave_lp = d_b;
    db.prox_lp = coupled ? nullptr : d_q;
    db.step_off = d_so; db.traj_off = d_to; db.group_off = d_go; db.rewards = d_rw;
    awr_head_outputs dout = {};
    dout.loss = (float*)d_scal; dout.clip_count = (int64_t*)(d_scal + 8);
    dout.err_word = (uint32_t*)(d_scal + 16); dout.dual_clip_count = (int64_t*)(d_scal + 24);
    dout.dhidden = d_dh; dout.dw_head = d_dw; dout.token_lp = d_lp;
    dout.adv = d_adv; dout.tok_traj = d_tt; dout.tok_term = d_term; dout.tok_coef = d_coef;
    dout.token_entropy = ho->token_entropy ? d_ent : nullptr;
    rc = awr_loss_fwd_bwd_fused_head(&db, p, &dout, d_headws, hp.head_ws, stream);
    if (rc != AWR_OK) { cudaStreamSynchronize(st); cudaGetLastError(); return rc; }

    AWR_TRY(cudaMemcpyAsync(ho->dw_head, d_dw, (size_t)hb->K * hb->V * 2, D2H, st));
    AWR_TRY(cudaMemcpyAsync(ho->loss, d_scal, 4, D2H, st));
    AWR_TRY(cudaMemcpyAsync(ho->clip_count, d_scal + 8, 8, D2H, st));
    if (ho->err_word) AWR_TRY(cudaMemcpyAsync(ho->err_word, d_scal + 16, 4, D2H, st));
    if (ho->dual_clip_count) AWR_TRY(cudaMemcpyAsync(ho->dual_clip_count, d_scal + 24, 8, D2H, st));
    if (n > 0) {
        AWR_TRY(cudaMemcpyAsync(ho->dhidden, d_dh, (size_t)n * hb->K * 2, D2H, st));
        AWR_TRY(cudaMemcpyAsync(ho->token_lp, d_lp, (size_t)n * 4, D2H, st));
        if (ho->tok_traj) AWR_TRY(cudaMemcpyAsync(ho->tok_traj, d_tt, (size_t)n * 4, D2H, st));
        if (ho->tok_term) AWR_TRY(cudaMemcpyAsync(ho->tok_term, d_term, (size_t)n * 4, D2H, st));
        if (ho->tok_coef) AWR_TRY(cudaMemcpyAsync(ho->tok_coef, d_coef, (size_t)n * 4, D2H, st));
        if (ho->token_entropy) AWR_TRY(cudaMemcpyAsync(ho->token_entropy, d_ent, (size_t)n * 4, D2H, st));
    }
    if (ho->adv && hb->n_traj > 0) AWR_TRY(cudaMemcpyAsync(ho->adv, d_adv, (size_t)hb->n_traj * 4, D2H, st));
    { cudaError_t e2 = cudaStreamSynchronize(st); if (e == cudaSuccess) e = e2; }
#undef AWR_TRY
    if (e != cudaSuccess) { cudaGetLastError(); return AWR_ERR_CUDA; }
    return AWR_OK;
}

// ------------------------------------------------------------------ host-buffer variant
namespace {
constexpr int kPanelBufs = 3;

struct HostPlan {
    int64_t panel_rows;
    size_t panel_bytes;   // per buffer
    size_t small_bytes;   // per-token / per-segment arrays
    size_t ws_bytes;      // awr_workspace_bytes
    size_t total;
};

HostPlan host_plan(int64_t n_tok, int64_t V, int64_t ld, int32_t dtype, int32_t n_steps,
                   int32_t n_traj, int32_t n_groups) {
    HostPlan h;
    const size_t esz = dtype == AWR_DTYPE_BF16 ? 2 : 4;
    const size_t row_bytes = (size_t)ld * esz;
    int64_t rows = (int64_t)((256u << 20) / (row_bytes ? row_bytes : 1));     // 256 MB panels
    if (rows < 64) rows = 64;
    if (rows > n_tok) rows = n_tok > 0 ? n_tok : 1;
    h.panel_rows = rows;
    h.panel_bytes = align_up((size_t)rows * row_bytes, 256);
    size_t s = 0;
    s += align_up((size_t)n_tok * 4, 256) * 4;     // target_ids, behave_lp, prox_lp, token_lp
    s += align_up((size_t)(n_steps + 1) * 4, 256) + align_up((size_t)(n_traj + 1) * 4, 256) +
         align_up((size_t)(n_groups + 1) * 4, 256) + align_up((size_t)n_traj * 4, 256);
    s += 256;                                      // loss, clip_count, err
    s += align_up((size_t)n_tok * 4, 256) * 5;     // optional tok_traj, target_logit, tok_term, tok_coef,
                                                   // token_entropy
    s += align_up((size_t)n_traj * 4, 256);        // optional adv
    h.small_bytes = s;
    h.ws_bytes = awr_workspace_bytes(n_tok, V, n_steps, n_traj, n_groups);
    h.total = h.small_bytes + h.ws_bytes + kPanelBufs * h.panel_bytes;
    return h;
}
}  // namespace

size_t awr_host_workspace_bytes(int64_t n_tok, int64_t V, int64_t ld, int32_t logits_dtype,
                                int32_t n_steps, int32_t n_traj, int32_t n_groups) {
    if (n_tok < 0 || V <= 0 || ld < V || n_steps < 0 || n_traj < 0 || n_groups < 0) return 0;
    return host_plan(n_tok, V, ld, logits_dtype, n_steps, n_traj, n_groups).total;
}

int awr_loss_fwd_bwd_host(const awr_batch* hb, const awr_params* p, const awr_outputs* ho,
                          void* dev_ws, size_t dev_ws_bytes, void* stream) {
    if (!hb || !p || !ho) return AWR_ERR_NULL;
    int rc = check_segments(hb->n_tok, hb->n_steps, hb->n_traj, hb->n_groups);
    if (rc) return rc;
    if (hb->V <= 0 || hb->ld < hb->V) return AWR_ERR_SHAPE;
    if (hb->logits_dtype != AWR_DTYPE_BF16 && hb->logits_dtype != AWR_DTYPE_F32) return AWR_ERR_DTYPE;
    rc = check_params(p);
    if (rc) return rc;
    if (!ho->loss || !ho->clip_count) return AWR_ERR_NULL;
    if (hb->n_tok > 0 && (!ho->token_lp || !ho->dlogits)) return AWR_ERR_NULL;
    if (!hb->step_off || !hb->traj_off || !hb->group_off) return AWR_ERR_NULL;
    const bool coupled = (p->flags & AWR_FLAG_COUPLED) != 0;      // prox_lp is neither read nor copied
    if (hb->n_tok > 0 && (!hb->logits || !hb->target_ids || !hb->behave_lp || (!coupled && !hb->prox_lp)))
        return AWR_ERR_NULL;
    if (hb->n_traj > 0 && !hb->rewards) return AWR_ERR_NULL;
    const size_t esz = hb->logits_dtype == AWR_DTYPE_BF16 ? 2 : 4;
    if (((size_t)hb->ld * esz) % 16) return AWR_ERR_ALIGN;
    HostPlan hp = host_plan(hb->n_tok, hb->V, hb->ld, hb->logits_dtype, hb->n_steps, hb->n_traj, hb->n_groups);
    if (!dev_ws || (reinterpret_cast<uintptr_t>(dev_ws) & 255) || dev_ws_bytes < hp.total) return AWR_ERR_WORKSPACE;
    const int kernel = resolve_kernel(p->kernel, hb->V, hb->ld, hb->logits_dtype, ho->token_entropy != nullptr);
    if (kernel < 0 || kernel == AWR_KERNEL_FWD_STREAM) return AWR_ERR_PARAM;
    DeviceInfo info;
    if (device_info(info) != cudaSuccess) { cudaGetLastError(); return AWR_ERR_CUDA; }
    if (info.major != 10) return AWR_ERR_ARCH;

    const int64_t n = hb->n_tok;
    uint8_t* base = reinterpret_cast<uint8_t*>(dev_ws);
    size_t off = 0;
    auto take = [&](size_t bytes) { void* r = base + off; off += align_up(bytes, 256); return r; };
    int32_t* d_ids = (int32_t*)take((size_t)n * 4);
    float* d_b = (float*)take((size_t)n * 4);
    float* d_q = (float*)take((size_t)n * 4);
    float* d_lp = (float*)take((size_t)n * 4);
    int32_t* d_so = (int32_t*)take((size_t)(hb->n_steps + 1) * 4);
    int32_t* d_to = (int32_t*)take((size_t)(hb->n_traj + 1) * 4);
    int32_t* d_go = (int32_t*)take((size_t)(hb->n_groups + 1) * 4);
    float* d_rw = (float*)take((size_t)hb->n_traj * 4);
    uint8_t* d_scal = (uint8_t*)take(256);
    int32_t* d_tt = (int32_t*)take((size_t)n * 4);
    float* d_tl = (float*)take((size_t)n * 4);
    float* d_term = (float*)take((size_t)n * 4);
    float* d_coef = (float*)take((size_t)n * 4);
    float* d_ent = (float*)take((size_t)n * 4);
    float* d_adv = (float*)take((size_t)hb->n_traj * 4);
    off = hp.small_bytes;
    void* d_ws = base + off; off += hp.ws_bytes;
    uint8_t* d_panel = base + off;
    float* d_loss = (float*)d_scal;
    int64_t* d_cnt = (int64_t*)(d_scal + 8);
    uint32_t* d_err = (uint32_t*)(d_scal + 16);
    int64_t* d_dual = (int64_t*)(d_scal + 24);

    cudaStream_t user = reinterpret_cast<cudaStream_t>(stream);
    cudaStream_t s_in = nullptr, s_k = nullptr, s_out = nullptr;
    cudaEvent_t ev_start = nullptr, ev_in[kPanelBufs] = {}, ev_k[kPanelBufs] = {}, ev_out[kPanelBufs] = {};
    cudaError_t e = cudaSuccess;
#define AWR_TRY(x) do { if (e == cudaSuccess) e = (x); } while (0)
    AWR_TRY(cudaStreamCreateWithFlags(&s_in, cudaStreamNonBlocking));
    AWR_TRY(cudaStreamCreateWithFlags(&s_k, cudaStreamNonBlocking));
    AWR_TRY(cudaStreamCreateWithFlags(&s_out, cudaStreamNonBlocking));
    AWR_TRY(cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming));
    for (int i = 0; i < kPanelBufs; ++i) {
        AWR_TRY(cudaEventCreateWithFlags(&ev_in[i], cudaEventDisableTiming));
        AWR_TRY(cudaEventCreateWithFlags(&ev_k[i], cudaEventDisableTiming));
        AWR_TRY(cudaEventCreateWithFlags(&ev_out[i], cudaEventDisableTiming));
    }
    AWR_TRY(cudaEventRecord(ev_start, user));
    AWR_TRY(cudaStreamWaitEvent(s_in, ev_start, 0));
    AWR_TRY(cudaStreamWaitEvent(s_k, ev_start, 0));
    AWR_TRY(cudaStreamWaitEvent(s_out, ev_start, 0));
    // small arrays + a0, a1 on the kernel stream
    const cudaMemcpyKind H2D = cudaMemcpyHostToDevice, D2H = cudaMemcpyDeviceToHost;
    if (n > 0) {
        AWR_TRY(cudaMemcpyAsync(d_ids, hb->target_ids, (size_t)n * 4, H2D, s_k));
        AWR_TRY(cudaMemcpyAsync(d_b, hb->behave_lp, (size_t)n * 4, H2D, s_k));
        if (!coupled) AWR_TRY(cudaMemcpyAsync(d_q, hb->prox_lp, (size_t)n * 4, H2D, s_k));
    }
    AWR_TRY(cudaMemcpyAsync(d_so, hb->step_off, (size_t)(hb->n_steps + 1) * 4, H2D, s_k));
    AWR_TRY(cudaMemcpyAsync(d_to, hb->traj_off, (size_t)(hb->n_traj + 1) * 4, H2D, s_k));
    AWR_TRY(cudaMemcpyAsync(d_go, hb->group_off, (size_t)(hb->n_groups + 1) * 4, H2D, s_k));
    if (hb->n_traj > 0) AWR_TRY(cudaMemcpyAsync(d_rw, hb->rewards, (size_t)hb->n_traj * 4, H2D, s_k));
    Workspace w = carve(d_ws, n, hb->n_traj);
    AWR_TRY(cudaMemsetAsync(d_ws, 0, w.zero_bytes, s_k));
    AWR_TRY(cudaMemsetAsync(d_scal, 0, 256, s_k));
    if (hb->n_traj > 0) AWR_TRY(cudaMemsetAsync(d_adv, 0, (size_t)hb->n_traj * 4, s_k));
    AWR_TRY(launch_segment_expand(d_so, d_to, d_go, n, hb->n_steps, hb->n_traj, hb->n_groups, d_tt, d_err,
                                  info.num_sms, s_k));
    AWR_TRY(launch_group_advantage(d_rw, d_go, d_to, hb->n_groups, hb->n_traj, p->flags, p->normalizer,
                                   p->k_norm, p->loss_scale, d_adv, w.traj_scale, w.err + 1, s_k));
    // row panels: H2D -> kernel (in place) -> D2H, three buffers in flight
    const size_t row_bytes = (size_t)hb->ld * esz;
    int64_t panel = 0;
    for (int64_t r0 = 0; r0 < n && e == cudaSuccess; r0 += hp.panel_rows, ++panel) {
        const int bi = (int)(panel % kPanelBufs);
        const int64_t rows = (n - r0 < hp.panel_rows) ? (n - r0) : hp.panel_rows;
        uint8_t* buf = d_panel + (size_t)bi * hp.panel_bytes;
        if (panel >= kPanelBufs) AWR_TRY(cudaStreamWaitEvent(s_in, ev_out[bi], 0));
        AWR_TRY(cudaMemcpyAsync(buf, (const uint8_t*)hb->logits + (size_t)r0 * row_bytes,
                                (size_t)rows * row_bytes, H2D, s_in));
        AWR_TRY(cudaEventRecord(ev_in[bi], s_in));
        AWR_TRY(cudaStreamWaitEvent(s_k, ev_in[bi], 0));
        RowArgs a;
        a.logits = buf; a.dlogits = buf;                 // in place on the panel
        a.n_tok = rows; a.V = hb->V; a.ld = hb->ld;
        a.target_ids = d_ids + r0; a.behave_lp = d_b + r0;
        a.prox_lp = (coupled ? d_b : d_q) + r0;
        a.tok_traj = d_tt + r0; a.adv = d_adv; a.traj_scale = w.traj_scale;
        a.token_lp = d_lp + r0; a.tok_term = d_term + r0; a.tok_coef = d_coef + r0;
        a.target_logit = d_tl + r0; a.tok_flag = w.tok_flag + r0; a.err_word = d_err;
        a.token_entropy = ho->token_entropy ? d_ent + r0 : nullptr;
        a.clip_eps = p->clip_eps; a.stale_cap = p->stale_cap; a.dual_c = p->dual_clip_c;
        AWR_TRY(launch_rows(kernel, a, hb->logits_dtype, info.num_sms, s_k));
        AWR_TRY(cudaEventRecord(ev_k[bi], s_k));
        AWR_TRY(cudaStreamWaitEvent(s_out, ev_k[bi], 0));
        AWR_TRY(cudaMemcpyAsync((uint8_t*)ho->dlogits + (size_t)r0 * row_bytes, buf,
                                (size_t)rows * row_bytes, D2H, s_out));
        AWR_TRY(cudaEventRecord(ev_out[bi], s_out));
    }
    AWR_TRY(launch_final_reduce(d_term, w.tok_flag, n, d_loss, d_cnt, d_dual, s_k));
    AWR_TRY(cudaMemcpyAsync(ho->loss, d_loss, 4, D2H, s_k));
    AWR_TRY(cudaMemcpyAsync(ho->clip_count, d_cnt, 8, D2H, s_k));
    if (ho->dual_clip_count) AWR_TRY(cudaMemcpyAsync(ho->dual_clip_count, d_dual, 8, D2H, s_k));
    if (ho->err_word) AWR_TRY(cudaMemcpyAsync(ho->err_word, d_err, 4, D2H, s_k));
    if (n > 0) {
        AWR_TRY(cudaMemcpyAsync(ho->token_lp, d_lp, (size_t)n * 4, D2H, s_k));
        if (ho->tok_traj) AWR_TRY(cudaMemcpyAsync(ho->tok_traj, d_tt, (size_t)n * 4, D2H, s_k));
        if (ho->target_logit) AWR_TRY(cudaMemcpyAsync(ho->target_logit, d_tl, (size_t)n * 4, D2H, s_k));
        if (ho->tok_term) AWR_TRY(cudaMemcpyAsync(ho->tok_term, d_term, (size_t)n * 4, D2H, s_k));
        if (ho->tok_coef) AWR_TRY(cudaMemcpyAsync(ho->tok_coef, d_coef, (size_t)n * 4, D2H, s_k));
        if (ho->token_entropy) AWR_TRY(cudaMemcpyAsync(ho->token_entropy, d_ent, (size_t)n * 4, D2H, s_k));
    }
    if (ho->adv && hb->n_traj > 0) AWR_TRY(cudaMemcpyAsync(ho->adv, d_adv, (size_t)hb->n_traj * 4, D2H, s_k));
    if (s_in) { cudaError_t e2 = cudaStreamSynchronize(s_in); if (e == cudaSuccess) e = e2; }
    if (s_k) { cudaError_t e2 = cudaStreamSynchronize(s_k); if (e == cudaSuccess) e = e2; }
    if (s_out) { cudaError_t e2 = cudaStreamSynchronize(s_out); if (e == cudaSuccess) e = e2; }
#undef AWR_TRY
    for (int i = 0; i < kPanelBufs; ++i) {
        if (ev_in[i]) cudaEventDestroy(ev_in[i]);
        if (ev_k[i]) cudaEventDestroy(ev_k[i]);
        if (ev_out[i]) cudaEventDestroy(ev_out[i]);
    }
    if (ev_start) cudaEventDestroy(ev_start);
    if (s_in) cudaStreamDestroy(s_in);
    if (s_k) cudaStreamDestroy(s_k);
    if (s_out) cudaStreamDestroy(s_out);
    if (e != cudaSuccess) { cudaGetLastError(); return AWR_ERR_CUDA; }
    return AWR_OK;
}

}  // extern "C"
