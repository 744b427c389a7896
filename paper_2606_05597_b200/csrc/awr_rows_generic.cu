// Generic row kernel: a2 (online log-sum-exp + target gather), a3 (ratio / clip / normalizer)
// and a4 (dlogits write) for any V, any row stride and both dtypes.  One CTA per row; the
// gradient pass re-reads the row, which at one row per CTA is an L2 hit (<= 148*8 rows of
// <= 300 KB in flight against 126 MB of L2), so HBM sees one read and one write per element.
// Plain (coherent) loads: dlogits may alias logits exactly.
// This is the correctness-first kernel and the path for fp32 logits / small or odd V; large
// bf16 rows go to the cluster kernel (awr_rows_cluster.cu).
// PAPER.md:57 (Eq. 1), :435 (token-level IS); gradient: SURVEY.md 8(c) O8.
#include "awr_common.cuh"
#include "awr_kernels.h"

namespace awr {

constexpr int kGenericThreads = 256;

template <typename T> struct Elem;
template <> struct Elem<float> {
    static constexpr int kPerVec = 4;
    static __device__ __forceinline__ void unpack(const uint4& v, float* x) {
        x[0] = __uint_as_float(v.x); x[1] = __uint_as_float(v.y);
        x[2] = __uint_as_float(v.z); x[3] = __uint_as_float(v.w);
    }
    static __device__ __forceinline__ uint4 pack(const float* x) {
        return make_uint4(__float_as_uint(x[0]), __float_as_uint(x[1]), __float_as_uint(x[2]),
                          __float_as_uint(x[3]));
    }
    static __device__ __forceinline__ float load(const float* p) { return *p; }
    static __device__ __forceinline__ void store(float* p, float v) { *p = v; }
};
template <> struct Elem<__nv_bfloat16> {
    static constexpr int kPerVec = 8;
    static __device__ __forceinline__ void unpack(const uint4& v, float* x) {
        x[0] = bf16_lo(v.x); x[1] = bf16_hi(v.x); x[2] = bf16_lo(v.y); x[3] = bf16_hi(v.y);
        x[4] = bf16_lo(v.z); x[5] = bf16_hi(v.z); x[6] = bf16_lo(v.w); x[7] = bf16_hi(v.w);
    }
    static __device__ __forceinline__ uint4 pack(const float* x) {
        return make_uint4(pack_bf16x2(x[0], x[1]), pack_bf16x2(x[2], x[3]),
                          pack_bf16x2(x[4], x[5]), pack_bf16x2(x[6], x[7]));
    }
    static __device__ __forceinline__ float load(const __nv_bfloat16* p) {
        return __bfloat162float(*p);
    }
    static __device__ __forceinline__ void store(__nv_bfloat16* p, float v) {
        *p = __float2bfloat16_rn(v);
    }
};

template <typename T, bool ENT>
__global__ void __launch_bounds__(kGenericThreads)
rows_generic_kernel(RowArgs a) {
    using E = Elem<T>;
    constexpr int EPV = E::kPerVec;
    __shared__ MaxSum s_red[kGenericThreads / 32];
    __shared__ float s_redz[kGenericThreads / 32];
    constexpr bool want_ent = ENT;        // token_entropy output: its own instantiation
    __shared__ float s_coef, s_lse, s_gy;
    __shared__ int s_y;
    const int tid = threadIdx.x;
    const int64_t nvec = a.V / EPV;
    const int64_t tail0 = nvec * EPV;

    for (int64_t row = blockIdx.x; row < a.n_tok; row += gridDim.x) {
        const T* z = reinterpret_cast<const T*>(a.logits) + row * a.ld;
        RowHeader h;
        bool valid = false;
        if (tid == 0) h = load_row_header(a, row, valid, sizeof(T) == 2);
        // every thread knows the target column: it is left out of the (max, sum) state, so
        // that l_t and 1 - p_y come from lse_rest without cancellation (token_scalars)
        const int yt = a.target_ids[row];
        const int64_t ycol = (yt >= 0 && yt < a.V) ? (int64_t)yt : (int64_t)-1;
        const int64_t yvec = ycol >= 0 ? ycol / EPV : (int64_t)-1;

        // ---- a2: one streaming pass, per-thread online (max, sum)
        MaxSum ms{-INFINITY, 0.f};
        float sz = 0.f;                    // sum e^{x - m} x alongside ms (entropy, optional)
        const uint4* zv = reinterpret_cast<const uint4*>(z);
        for (int64_t i = tid; i < nvec; i += kGenericThreads) {
            uint4 v = zv[i];
            float x[EPV];
            E::unpack(v, x);
            if (i == yvec) {
                const int yk = (int)(ycol - i * EPV);
#pragma unroll
                for (int k = 0; k < EPV; ++k) x[k] = (k == yk) ? -INFINITY : x[k];
            }
            float cm = x[0];
#pragma unroll
            for (int k = 1; k < EPV; ++k) cm = fmaxf(cm, x[k]);
            if (cm > ms.m) {
                const float sc = ex2_approx((ms.m - cm) * kLog2e);
                ms.s *= sc;
                if (want_ent) sz *= sc;
                ms.m = cm;
            }
            float ml = (ms.m == -INFINITY) ? 0.f : ms.m * kLog2e;   // all -inf so far: no NaN
            float acc = 0.f;
            if (want_ent) {
#pragma unroll
                for (int k = 0; k < EPV; ++k) {
                    const float e = ex2_approx(fmaf(x[k], kLog2e, -ml));
                    acc += e;
                    sz = fmaf(e, fmaxf(x[k], kZFloor), sz);
                }
            } else {
#pragma unroll
                for (int k = 0; k < EPV; ++k) acc += ex2_approx(fmaf(x[k], kLog2e, -ml));
            }
            ms.s += acc;
        }
        for (int64_t i = tail0 + tid; i < a.V; i += kGenericThreads) {
            float x = (i == ycol) ? -INFINITY : E::load(z + i);
            if (x > ms.m) {
                const float sc = ex2_approx((ms.m - x) * kLog2e);
                ms.s *= sc;
                if (want_ent) sz *= sc;
                ms.m = x;
            }
            if (ms.m != -INFINITY) {
                const float e = ex2_approx((x - ms.m) * kLog2e);
                ms.s += e;
                if (want_ent) sz = fmaf(e, fmaxf(x, kZFloor), sz);
            }
        }
        if (want_ent) {
            // bring this thread's sz to the warp's max before the (max, sum) state is merged
            float wm = ms.m;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) wm = fmaxf(wm, __shfl_xor_sync(kFull, wm, o));
            sz = (ms.m == -INFINITY) ? 0.f : sz * ex2_approx((ms.m - wm) * kLog2e);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) sz += __shfl_xor_sync(kFull, sz, o);
        }
        ms = warp_combine(ms);
        if ((tid & 31) == 0) { s_red[tid >> 5] = ms; s_redz[tid >> 5] = sz; }
        __syncthreads();
        if (tid == 0) {
            MaxSum tot = s_red[0];
#pragma unroll
            for (int w = 1; w < kGenericThreads / 32; ++w) tot = combine(tot, s_red[w]);
            float lse_rest = tot.m + logf(tot.s);   // -inf when the row has no other entry
            // ---- a3
            TokenScalars ts = token_scalars(h, lse_rest, valid, a.clip_eps, a.stale_cap, a.dual_c);
            store_token_outputs(a, row, h, ts, valid);
            if (want_ent) {
                float szt = 0.f;
#pragma unroll
                for (int w = 0; w < kGenericThreads / 32; ++w)
                    if (s_red[w].m != -INFINITY) szt += s_redz[w] * ex2_approx((s_red[w].m - tot.m) * kLog2e);
                a.token_entropy[row] = valid ? row_entropy(ts.lse, tot.m, szt, ts.lp, h.zy) : 0.f;
            }
            s_coef = ts.coef;
            s_lse = ts.lse;
            s_y = valid ? h.y : -1;
            s_gy = ts.gy;                           // c_t (p_y - 1)
        }
        __syncthreads();

        // ---- a4
        if (a.dlogits != nullptr) {
            T* g = reinterpret_cast<T*>(a.dlogits) + row * a.ld;
            uint4* gv = reinterpret_cast<uint4*>(g);
            const float coef = s_coef;
            const int y = s_y;
            if (coef == 0.f) {
                const uint4 zero = make_uint4(0, 0, 0, 0);
                for (int64_t i = tid; i < nvec; i += kGenericThreads) gv[i] = zero;
                for (int64_t i = tail0 + tid; i < a.V; i += kGenericThreads) E::store(g + i, 0.f);
            } else {
                const float nl = -s_lse * kLog2e;
                const float gy = s_gy;
                for (int64_t i = tid; i < nvec; i += kGenericThreads) {
                    uint4 v = zv[i];
                    float x[EPV];
                    E::unpack(v, x);
#pragma unroll
                    for (int k = 0; k < EPV; ++k) x[k] = coef * ex2_approx(fmaf(x[k], kLog2e, nl));
                    int64_t base = i * EPV;
                    if (y >= base && y < base + EPV) x[y - base] = gy;
                    gv[i] = E::pack(x);
                }
                for (int64_t i = tail0 + tid; i < a.V; i += kGenericThreads) {
                    float x = E::load(z + i);
                    float gval = (i == y) ? gy : coef * ex2_approx(fmaf(x, kLog2e, nl));
                    E::store(g + i, gval);
                }
            }
        }
        __syncthreads();
    }
}

cudaError_t launch_rows_generic(const RowArgs& a, int dtype, int num_sms, cudaStream_t st) {
    if (a.n_tok <= 0) return cudaSuccess;
    int64_t blocks = a.n_tok;
    int64_t cap = (int64_t)num_sms * 8;
    if (blocks > cap) blocks = cap;
    const bool ent = a.token_entropy != nullptr;
    if (dtype == AWR_DTYPE_BF16) {
        if (ent) rows_generic_kernel<__nv_bfloat16, true><<<(int)blocks, kGenericThreads, 0, st>>>(a);
        else rows_generic_kernel<__nv_bfloat16, false><<<(int)blocks, kGenericThreads, 0, st>>>(a);
    } else {
        if (ent) rows_generic_kernel<float, true><<<(int)blocks, kGenericThreads, 0, st>>>(a);
        else rows_generic_kernel<float, false><<<(int)blocks, kGenericThreads, 0, st>>>(a);
    }
    return cudaGetLastError();
}

}  // namespace awr
