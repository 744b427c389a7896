/* awr.h - C ABI of the B200-native AsyncWebRL token-loss library (libawr.so).
 *
 * What it computes (all citations are /root/reference/PAPER.md lines; "A<n>" / "O<n>" are
 * the readings and oracle steps of SURVEY.md section 8(c), restated in DESIGN.md):
 *
 *   J(theta) = E[ 1/(G k) sum_i sum_j sum_t min( (pi_theta/pi_behave) A_i ,
 *                 (pi_prox/pi_behave) clip(pi_theta/pi_prox, 1-eps, 1+eps) A_i ) ]   Eq. (1), :57
 *   A_i = (r_i - mean(r)) / std(r) over the G rollouts of one task                    :61
 *   1/k (constant, k = 10) or the standard 1/|tau_i| (steps of rollout i)             :55, :59
 *
 * per token t of trajectory i of group g, with z_t the logits row and y_t the sampled id:
 *   l_t = z_t[y_t] - logsumexp(z_t)          r_t = exp(l_t - prox_lp_t)
 *   w_t = exp(prox_lp_t - behave_lp_t), truncated at stale_cap if 0 < stale_cap < inf (A4)
 *   u = r_t A_i ; v = clip(r_t, 1-eps, 1+eps) A_i ; trig_t = (v < u)                  (A5, A6)
 *   scale_i = loss_scale / (NG * G_g) * (1/k_norm | 1/|tau_i|)                        (A1, O6)
 *   term_t = scale_i w_t min(u, v)           loss = - sum_t term_t  (fixed order, fp64 sum)
 *   c_t = trig_t ? 0 : scale_i w_t r_t A_i   dlogits[t, v] = c_t (softmax(z_t)_v - [v = y_t])
 *   clip_count = sum_t trig_t
 *
 * Conventions
 *   - Every pointer in awr_batch / awr_outputs / awr_head_* is a DEVICE pointer owned by the
 *     caller; inputs are read-only; outputs are overwritten (never accumulated into).
 *     Only awr_loss_fwd_bwd_host takes HOST pointers (stated there).
 *   - Calls only enqueue work on `stream` (a cudaStream_t passed as void*; NULL = the legacy
 *     default stream).  No allocation, no host synchronisation; outputs are valid once the
 *     stream has been synchronised.  Graph-capturable.
 *   - Thread safety / state: entry points may be called concurrently from several host threads
 *     as long as concurrent calls use different `stream`s, different workspaces and different
 *     outputs.  The library keeps no per-call state.  What it keeps per DEVICE: cached device
 *     attributes, function attributes, and (fused head, stored-logits mode only) a pool of up to
 *     8 side streams, each with one fork / join event pair, keyed by the caller's stream - calls
 *     on different streams never share one; when all 8 are busy the call runs without the
 *     overlap.  Two calls racing on the SAME stream are ordered by whichever enqueues first, as
 *     with any CUDA work.
 *   - Return value: AWR_OK or a negative awr_status.  Host-side checks cover scalars, null
 *     pointers, alignment and workspace size only.  Data-dependent faults set bits in
 *     *err_word (AWR_ERRBIT_*) and the affected token contributes nothing.
 *   - target_ids[t] < 0 marks a masked token: zero term, zero dlogits row, token_lp = 0,
 *     never counted (A13).  target_ids[t] >= V additionally sets AWR_ERRBIT_TARGET_RANGE.
 *   - Rows: logits[t * ld + v], 0 <= v < V, ld >= V; every row start must be 16-byte aligned
 *     (base pointer 16-B aligned and ld * sizeof(element) % 16 == 0).  Columns >= V are never
 *     read or written.  dlogits has the same dtype and stride and MAY alias logits exactly
 *     (in-place); any other overlap is undefined.
 *   - The device must be compute capability 10.x (sm_100a code only): otherwise AWR_ERR_ARCH.
 *     There is no CPU or other-architecture fallback.
 */
#ifndef AWR_H_
#define AWR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define AWR_VERSION 200

#if defined(__GNUC__)
#define AWR_API __attribute__((visibility("default")))
#else
#define AWR_API
#endif

typedef enum awr_status {
    AWR_OK = 0,
    AWR_ERR_NULL = -1,      /* a required pointer is NULL */
    AWR_ERR_SHAPE = -2,     /* negative / inconsistent sizes, ld < V, counts overflowing int32 */
    AWR_ERR_DTYPE = -3,     /* unknown dtype / layout enum */
    AWR_ERR_ALIGN = -4,     /* row starts not 16-byte aligned */
    AWR_ERR_PARAM = -5,     /* k_norm <= 0, clip_eps outside [0,1), NaN scalars, bad enum */
    AWR_ERR_WORKSPACE = -6, /* workspace NULL, misaligned (256 B) or too small */
    AWR_ERR_ARCH = -7,      /* current device is not sm_100 */
    AWR_ERR_CUDA = -8,      /* a CUDA runtime call / launch failed (cudaGetLastError cleared) */
    AWR_ERR_STATIC_LIMIT = -9 /* awr_loss_fwd_bwd_static: the batch needs more scratch than
                                 AWR_STATIC_WS_BYTES; use awr_loss_fwd_bwd with a workspace */
} awr_status;

enum { AWR_DTYPE_BF16 = 0, AWR_DTYPE_F32 = 1 };
enum { AWR_NORM_CONST_K = 0,   /* n_i = 1 / k_norm   (:59) */
       AWR_NORM_PER_TRAJ = 1   /* n_i = 1 / |tau_i|  (:55) */ };
enum { AWR_FLAG_SAMPLE_STD = 1u,     /* A2: std with 1/(G-1) instead of the default 1/G */
       AWR_FLAG_SUCCESS_FILTER = 2u, /* RAFT++ baseline (:65): A_i = 1[R_i > 0], no group mean/std */
       AWR_FLAG_SKIP_UNIFORM = 8u,   /* dynamic sampling (:63): all-success / all-failure groups are
                                        skipped on the device - zero advantage, and the mean over
                                        groups runs over the mixed groups only (one extra launch) */
       AWR_FLAG_COUPLED = 4u         /* coupled-ratio ablation (:114): one pi_theta/pi_behave ratio
                                        with the clip centred on it, no staleness weight; prox_lp
                                        is not read and may be NULL */ };
enum { AWR_W_K_BY_V = 0 /* w_head[k * V + v] */, AWR_W_V_BY_K = 1 /* w_head[v * K + k] */ };
enum { AWR_KERNEL_AUTO = 0,     /* pick by shape / dtype */
       AWR_KERNEL_GENERIC = 1,  /* one CTA per row, second pass re-reads the row through L2 */
       AWR_KERNEL_CLUSTER = 2,  /* row resident in the shared memory of a 2-CTA cluster (bf16) */
       AWR_KERNEL_CLUSTER_RF = 3, /* row resident in the register files of a 2-CTA cluster (bf16,
                                    16K <= V <= 163,840); shared memory is a TMA load FIFO */
       AWR_KERNEL_CLUSTER_RF4 = 4, /* the same with a row quarter per CTA of a 4-CTA cluster and
                                    two CTAs (of different rows) resident per SM */
       /* fused-head entry points only (AUTO = AWR_KERNEL_HEAD_2CTA_ROWREF): */
       AWR_KERNEL_HEAD_1CTA = 5, /* tcgen05 cta_group::1, 128 x 256 tiles, one CTA per SM; the
                                    logits tile is recomputed for the backward (8 K V flops/token) */
       AWR_KERNEL_HEAD_2CTA = 6, /* tcgen05 cta_group::2, 256 x 256 tiles on CTA pairs; recompute */
       AWR_KERNEL_HEAD_2CTA_STORED = 7, /* CTA pairs; the fp32 logits of ONE row panel (<= 9,472
                                    rows, workspace) are kept between the forward GEMM and a
                                    streaming dS pass: 6 K V flops/token, same bits as recompute */
       /* awr_loss_fwd only (its AUTO choice for bf16 rows of >= 64 KB): */
       AWR_KERNEL_FWD_STREAM = 8, /* forward-only streaming kernel: whole rows through a ring of TMA
                                    bulk copies, one persistent CTA per SM, no row residency (bf16,
                                    V and ld multiples of 8); with awr_loss_fwd_bwd -> AWR_ERR_PARAM */
       AWR_KERNEL_HEAD_2CTA_E16 = 9 /* fused head, CTA pairs: the forward epilogue leaves E = bf16(exp(z -
                                    tile row max)) of ONE row panel (<= 9,472 rows) in the dS buffer and one
                                    in-place pass rescales it to dS: 6 K V flops/token, 2 bytes of
                                    transient per logit of the panel, no side stream */,
       AWR_KERNEL_CLUSTER_RFS = 10 /* row resident in the register files of a 2-CTA cluster, 15 data
                                    warps + one service warp per CTA: whole-slot TMA loads, gradient
                                    through shared-memory staging and TMA bulk stores, (max, sum)
                                    exchange by st.async, a3 on the service warp; rows pipelined in
                                    groups of 5 rounds, the row's (max, sum) sent for a3 BEFORE the last
                                    group's gradient is staged (its statistics taken from the ring) so
                                    that the a3 hand-over is hidden (bf16, 15,368 <= V <= 153,600; AUTO's
                                    choice for awr_loss_fwd_bwd there) */,
       AWR_KERNEL_HEAD_2CTA_ROWREF = 11 /* fused head, CTA pairs: E = bf16(exp(z - zref_t)) with a per-row
                                    reference computed before the GEMM (zref_t = the row's largest logit
                                    among the first 256 vocabulary entries: one column tile), so dS =
                                    E f_t with ONE factor per row: the dhidden GEMM scales its output rows
                                    by f_t, the dw_head GEMM reads bf16(f_t hidden_t); no pass over the
                                    panel is left.  A row with a logit more than ~88 nats above that
                                    reference (exp overflows; none on ordinary logits) is redone exactly
                                    from hidden and w_head on the CUDA cores (~2 ms per such row) */,
       AWR_KERNEL_CLUSTER_RFS_LATE = 12 /* AWR_KERNEL_CLUSTER_RFS with the row's (max, sum) sent for a3 after
                                    the last register group has been exponentiated instead of before its
                                    gradient is staged: the data warps wait ~2 k clocks per row for a3,
                                    but 25 % fewer shared-memory sweeps.  Measured (config 1): 5-8 % slower
                                    than CLUSTER_RFS in a cold burst at the boost clock, 2-3 % faster at
                                    1.6-1.8 GHz, level between dense GEMMs - DESIGN.md section 4 */ };
enum { AWR_ERRBIT_STEP_OFF = 1u, AWR_ERRBIT_TRAJ_OFF = 2u, AWR_ERRBIT_GROUP_OFF = 4u,
       AWR_ERRBIT_TARGET_RANGE = 8u };

/* One batch of response tokens (:61 "G rollouts per task, |tau_i| steps per rollout,
 * |tau_{i,j}| tokens per step"), as three CSR offset arrays.  Each offset array starts at 0,
 * is non-decreasing and ends at the count of the level below (O1); violations set
 * AWR_ERRBIT_* and give unspecified (but memory-safe) results. */
typedef struct awr_batch {
    int64_t n_tok;              /* rows of logits = response tokens in the batch */
    int64_t V;                  /* vocabulary size */
    int64_t ld;                 /* row stride in elements, >= V */
    const void* logits;         /* [n_tok, ld], dtype logits_dtype */
    const int32_t* target_ids;  /* [n_tok] sampled token y_t; < 0 = masked */
    const float* behave_lp;     /* [n_tok] log pi_behave(y_t) (:53) */
    const float* prox_lp;       /* [n_tok] log pi_prox(y_t)   (:53, :436) */
    const int32_t* step_off;    /* [n_steps + 1] token index where each step starts */
    const int32_t* traj_off;    /* [n_traj + 1]  step index where each trajectory starts */
    const int32_t* group_off;   /* [n_groups + 1] trajectory index where each group starts */
    const float* rewards;       /* [n_traj] r_i (:73 binary in the paper; any finite f32) */
    int32_t n_steps;
    int32_t n_traj;
    int32_t n_groups;
    int32_t logits_dtype;       /* AWR_DTYPE_* */
} awr_batch;

typedef struct awr_params {
    float k_norm;       /* the constant k of 1/k (:59), > 0; used when normalizer == CONST_K */
    float clip_eps;     /* eps of the decoupled clip (:57), in [0, 1); paper: 0.2 (:437) */
    float stale_cap;    /* A4: w_t <- min(w_t, cap); <= 0 or +inf = off (Eq. 1 exactly) */
    float loss_scale;   /* multiplies loss and gradient (micro-batching); 1 = Eq. 1 */
    float dual_clip_c;  /* Eq. (2) (:270-275, c = 3.0 in every GRPO run of the paper, :461): > 1 caps
                           the per-token min from below by c * A when A < 0; <= 1 = off = Eq. (1).
                           A hit (A < 0 and pi_theta/pi_prox > c) has zero gradient. */
    int32_t normalizer; /* AWR_NORM_* */
    uint32_t flags;     /* AWR_FLAG_*; unknown bits -> AWR_ERR_PARAM */
    int32_t kernel;     /* AWR_KERNEL_*; CLUSTER on an unsupported shape -> AWR_ERR_PARAM */
} awr_params;

typedef struct awr_outputs {
    float* loss;            /* [1]  -J, f32: the per-token terms summed in fp64 in a FIXED order
                               (thread-strided partial sums of 1024 threads, then a binary tree)
                               and rounded once - bit-reproducible, not token order */
    void* dlogits;          /* [n_tok, ld] same dtype/stride as logits; NULL in awr_loss_fwd */
    float* token_lp;        /* [n_tok] l_t = log pi_theta(y_t); 0 for masked tokens */
    int64_t* clip_count;    /* [1] number of tokens with trig_t */
    /* optional (NULL = not wanted) */
    float* adv;             /* [n_traj] A_i */
    int32_t* tok_traj;      /* [n_tok] trajectory index of each token */
    float* target_logit;    /* [n_tok] z_t[y_t] widened to f32 (exact); 0 for masked tokens */
    float* tok_term;        /* [n_tok] per-token contribution to J (loss = -sum) */
    float* tok_coef;        /* [n_tok] c_t */
    uint32_t* err_word;     /* [1] OR of AWR_ERRBIT_* (0 = clean) */
    int64_t* dual_clip_count; /* [1] number of tokens hit by the dual clip (:128); 0 when off */
    float* token_entropy;   /* [n_tok] optional: H_t = -sum_v p_v log p_v of softmax(z_t), the paper's
                               per-token entropy diagnostic (:232, :341), from the same streaming
                               pass; 0 for masked tokens.  Generic and register-file kernels (an
                               explicit AWR_KERNEL_CLUSTER with it -> AWR_ERR_PARAM) */
    /* optional measurement aid (both or neither; NULL = off): two cudaEvent_t created by the
     * caller with timing enabled; THIS call records them on `stream` immediately before / after
     * its row kernel (a2 + a3 + a4), so bench.py can report that kernel's own duration from
     * inside the timed region.  Per call, no library state (ignored by the host-buffer entry). */
    void* ev_row_begin;
    void* ev_row_end;
} awr_outputs;

/* a0..a4 fused: segment expansion, group advantage (:61), online log-sum-exp + target gather,
 * decoupled ratio / clip / normalizer (Eq. 1, :57-:59) and the gradient write.  4 launches. */
AWR_API int awr_loss_fwd_bwd(const awr_batch* batch, const awr_params* params, const awr_outputs* out,
                     void* workspace, size_t workspace_bytes, void* stream);

/* Forward only: loss, token_lp, clip_count (and the optional per-token outputs); out->dlogits
 * is ignored.  Reads each row once, writes no gradient.  This is the proximal log-prob
 * recomputation the trainer runs at the start of every update ("proximal logprobs
 * recomputed"; token_lp of this call is the prox_lp of the update's loss calls) and the source of
 * the per-token entropy diagnostic (:232, :341). */
AWR_API int awr_loss_fwd(const awr_batch* batch, const awr_params* params, const awr_outputs* out,
                 void* workspace, size_t workspace_bytes, void* stream);

/* Kernel 1 alone (:61).  One warp per group.  flags: AWR_FLAG_SAMPLE_STD. */
AWR_API int awr_group_advantage(const float* rewards, const int32_t* group_off, int32_t n_groups,
                        int32_t n_traj, uint32_t flags, float* adv, void* stream);

/* Bytes of device workspace awr_loss_fwd_bwd / awr_loss_fwd need (256-B aligned pointer). */
AWR_API size_t awr_workspace_bytes(int64_t n_tok, int64_t V, int32_t n_steps, int32_t n_traj,
                           int32_t n_groups);

/* awr_loss_fwd_bwd for callers that cannot allocate (code under CUDA-graph capture, serving loops,
 * harnesses that forbid cudaMalloc): the same checks, kernels and results, with the workspace in
 * a fixed device array inside the library instead of a caller buffer.  The call itself never
 * allocates: no cudaMalloc / cudaFree / allocating library routine; inputs and outputs are still
 * the caller's.
 *   Limit: awr_workspace_bytes(n_tok, V, n_steps, n_traj, n_groups) <= AWR_STATIC_WS_BYTES
 *   (1 MiB: 8 + 8 bytes per trajectory and 9 bytes per token, each array rounded up to 256 B -
 *   e.g. 110,000 tokens with 1,024 trajectories); a larger batch returns AWR_ERR_STATIC_LIMIT and
 *   nothing is launched.  The array costs 1 MiB of device memory on every GPU that loads the
 *   library, until the process exits.
 *   Sharing: every call on a device uses the SAME array, and it keeps the previous call's
 *   contents; the part that must start at zero (error word, advantages, trajectory scales) is
 *   cleared on `stream` at the start of every call.  Two calls that overlap on one GPU (different
 *   streams, or several host threads) RACE on it: order them on one stream or with events.
 *   Back-to-back calls on one stream are safe. */
#define AWR_STATIC_WS_BYTES ((size_t)1 << 20)
AWR_API int awr_loss_fwd_bwd_static(const awr_batch* batch, const awr_params* params,
                                    const awr_outputs* out, void* stream);

/* Same path with HOST buffers: every pointer in `batch` and `out` is a host pointer (pinned
 * memory gives full PCIe speed; pageable works).  Rows are staged through `dev_workspace` in
 * panels: H2D copy, the same kernels in place on the panel, D2H copy of the gradient panel, on
 * three internal non-blocking streams ordered after `stream`; the call returns after the
 * results are in the host buffers (it synchronises).  dev_workspace: device pointer of at
 * least awr_host_workspace_bytes(...) bytes. */
AWR_API int awr_loss_fwd_bwd_host(const awr_batch* host_batch, const awr_params* params,
                          const awr_outputs* host_out, void* dev_workspace,
                          size_t dev_workspace_bytes, void* stream);
AWR_API size_t awr_host_workspace_bytes(int64_t n_tok, int64_t V, int64_t ld, int32_t logits_dtype,
                                int32_t n_steps, int32_t n_traj, int32_t n_groups);

/* a5 (BASELINE.json config 4): hidden states + LM head instead of logits.  logits = hidden
 * [n_tok, K] x w_head are produced tile by tile in tensor memory and fed from there to the
 * log-sum-exp with fp32 accumulation (A17); the full [n_tok, V] matrix never exists.  What the modes
 * keep, for ONE row panel (<= 9,472 rows) at a time, between the panel's forward GEMM and its backward
 * GEMMs:  ROWREF (AUTO): E = bf16(exp(z - zref_t)), 2 bytes per logit of the panel, zref_t the row's
 * largest logit among the first 256 vocabulary entries, computed before the GEMM; dS = E f_t is never formed (the row factor is
 * applied by the dhidden epilogue and folded into the hidden operand of the dw_head GEMM);
 * E16: bf16(exp(z - tile row max)) in the dS buffer, rescaled to dS by one in-place pass;
 * STORED: the fp32 logits of the panel (two buffers, a side stream);  HEAD_1CTA / HEAD_2CTA: nothing
 * (the tile is recomputed, 8 K V instead of 6 K V flops per token).  awr_head_workspace_bytes()
 * gives the bytes per mode.  Outputs dhidden = dS W^T and dw_head = H^T dS (bf16, overwritten). */
typedef struct awr_head_batch {
    int64_t n_tok;
    int64_t V;
    int64_t K;                  /* hidden size; multiple of 64 (V: multiple of 8) */
    const void* hidden;         /* bf16 [n_tok, K] row-major */
    const void* w_head;         /* bf16, layout w_layout */
    const int32_t* target_ids;
    const float* behave_lp;
    const float* prox_lp;
    const int32_t* step_off;
    const int32_t* traj_off;
    const int32_t* group_off;
    const float* rewards;
    int32_t n_steps;
    int32_t n_traj;
    int32_t n_groups;
    int32_t w_layout;           /* AWR_W_* */
} awr_head_batch;

typedef struct awr_head_outputs {
    float* loss;
    void* dhidden;          /* bf16 [n_tok, K] */
    void* dw_head;          /* bf16, same layout as w_head */
    float* token_lp;
    int64_t* clip_count;
    float* adv;             /* optional */
    int32_t* tok_traj;      /* optional */
    float* tok_term;        /* optional */
    float* tok_coef;        /* optional */
    uint32_t* err_word;     /* optional */
    int64_t* dual_clip_count; /* optional */
    float* token_entropy;   /* optional [n_tok], as in awr_outputs (a third per-tile partial) */
} awr_head_outputs;

AWR_API int awr_loss_fwd_bwd_fused_head(const awr_head_batch* batch, const awr_params* params,
                                const awr_head_outputs* out, void* workspace,
                                size_t workspace_bytes, void* stream);
/* Workspace of the fused head for `kernel` (an AWR_KERNEL_HEAD_* id or AUTO); the modes differ:
 * config 4 (32,768 x 2048 x 151,936) needs 4.4 GB with ROWREF (AUTO) or E16, 15.9 GB with
 * HEAD_2CTA_STORED. */
AWR_API size_t awr_head_workspace_bytes(int64_t n_tok, int64_t V, int64_t K, int32_t n_steps,
                                int32_t n_traj, int32_t n_groups, int32_t kernel);

/* a5 with HOST buffers (the `e2e` leg of bench.py --config 4): every pointer in `host_batch` and
 * `host_out` is a host pointer (pinned memory gives full PCIe speed).  hidden, w_head and the
 * per-token arrays are copied to `dev_workspace`, awr_loss_fwd_bwd_fused_head runs there, and
 * dhidden, dw_head, loss, token_lp and the optional outputs are copied back, all on `stream`; the
 * call returns after the results are in the host buffers (it synchronises `stream`). */
AWR_API int awr_loss_fwd_bwd_fused_head_host(const awr_head_batch* host_batch, const awr_params* params,
                                     const awr_head_outputs* host_out, void* dev_workspace,
                                     size_t dev_workspace_bytes, void* stream);
AWR_API size_t awr_head_host_workspace_bytes(int64_t n_tok, int64_t V, int64_t K, int32_t n_steps,
                                     int32_t n_traj, int32_t n_groups, int32_t kernel);

/* Note: only AWR_KERNEL_HEAD_2CTA_STORED uses a side stream: it forks the dS pass of each row panel
 * onto a library-owned side stream (pool keyed by the caller's stream, see "Thread safety / state")
 * and joins it back before the panel's dhidden GEMM; from the caller's point of view all work is
 * still ordered on `stream`, and the call can be captured into a CUDA graph.
 *
 * Kernel launches one awr_loss_fwd_bwd_fused_head call enqueues for this shape. */
AWR_API int awr_head_launches_per_call(int64_t n_tok, int64_t V, int64_t K, int32_t kernel);

/* The tensor-core engine of a5 on its own (tests, benchmarks): C[M, N] = A B, bf16 operands,
 * fp32 accumulation in tensor memory, bf16 row-major result C[m * ldc + n].  A is [M, Kc] and B
 * is [Kc, N] as matrices; *_major says which index is contiguous in memory:
 *   a_major 0: A[m * lda + k]   a_major 1: A[k * lda + m]
 *   b_major 0: B[n * ldb + k]   b_major 1: B[k * ldb + n]
 * lda, ldb, ldc and N multiples of 8; pointers 16-byte aligned; device pointers.
 * kernel: AWR_KERNEL_AUTO, AWR_KERNEL_HEAD_1CTA or AWR_KERNEL_HEAD_2CTA. */
AWR_API int awr_gemm_bf16(const void* A, int32_t a_major, int64_t lda, const void* B, int32_t b_major,
                  int64_t ldb, int64_t M, int64_t N, int64_t Kc, void* C, int64_t ldc,
                  int32_t kernel, void* stream);

AWR_API const char* awr_status_string(int status);
AWR_API int awr_version(void);

/* Introspection for benchmarks and tests: which row kernel AWR_KERNEL_AUTO resolves to for
 * this shape in awr_loss_fwd_bwd (AWR_KERNEL_GENERIC, AWR_KERNEL_CLUSTER, AWR_KERNEL_CLUSTER_RF or
 * AWR_KERNEL_CLUSTER_RFS), and the number of kernel launches one
 * awr_loss_fwd_bwd call enqueues. */
AWR_API int awr_select_kernel(int64_t V, int64_t ld, int32_t logits_dtype);
AWR_API int awr_launches_per_call(void);

#ifdef __cplusplus
}
#endif
#endif /* AWR_H_ */
