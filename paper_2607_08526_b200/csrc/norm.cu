// norm.cu -- NEXT-2: the normalisation in front of QKV / MLP-up fused with the S1 activation
// quantiser ("quantizing activations alongside weights"; the DiT blocks of L71 / L278).  An
// unfused block stores the normalised tensor (2 MK bytes), reads it back in the S1 pass and writes the codes;
// here one pass reads X once and writes only the int8 codes and the per-token scales (the normalised
// tensor itself is written only if the caller asks for it: residual paths, tests).  HBM bound:
// algorithmic bytes per element = sizeof(x) + 1 (+ sizeof(x) with Xn) + 8/K.
//   kind 0 LayerNorm: mu = mean x; var = mean (x - mu)^2 (two-pass, biased); n = (x - mu) rstd gamma + beta
//   kind 1 RMSNorm:   n = x rstd gamma + beta,  rstd = 1 / sqrt(mean x^2 + eps)
// n is rounded ONCE to the activation dtype (the value an unfused norm kernel would store, R20)
// and S1 (include/aria.h) runs on that rounded value with the exact division-free rounding of quant_dev.cuh,
// so codes and scales are bit-identical to aria_quantize_act_int8 applied to Xn.
// One row per group of RW warps (RW = 1: shuffle reductions only; RW = 8: the whole CTA, via shared memory);
// every lane issues all its 16-byte loads up front and the row stays in registers for all three sweeps.
#include "internal.cuh"
#include "quant_dev.cuh"

namespace aria {

template <typename T> __device__ __forceinline__ float round_to(float v);
template <> __device__ __forceinline__ float round_to<float>(float v) { return v; }
template <> __device__ __forceinline__ float round_to<__nv_bfloat16>(float v) {
    return __bfloat162float(__float2bfloat16_rn(v));
}
__device__ __forceinline__ void store8(float* p, const float (&v)[8]) {
    *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
    *reinterpret_cast<float4*>(p + 4) = make_float4(v[4], v[5], v[6], v[7]);
}
__device__ __forceinline__ void store8(__nv_bfloat16* p, const float (&v)[8]) {   // v already holds bf16 values
    uint4 o;
    o.x = (__float_as_uint(v[0]) >> 16) | (__float_as_uint(v[1]) & 0xFFFF0000u);
    o.y = (__float_as_uint(v[2]) >> 16) | (__float_as_uint(v[3]) & 0xFFFF0000u);
    o.z = (__float_as_uint(v[4]) >> 16) | (__float_as_uint(v[5]) & 0xFFFF0000u);
    o.w = (__float_as_uint(v[6]) >> 16) | (__float_as_uint(v[7]) & 0xFFFF0000u);
    *reinterpret_cast<uint4*>(p) = o;
}

// sum (MAX = false) or max (MAX = true) over the RW warps that share a row
template <int RW, bool MAX>
__device__ __forceinline__ float row_reduce(float v, float* red, int lane, int warp) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float t = __shfl_xor_sync(0xffffffffu, v, o);
        v = MAX ? fmaxf(v, t) : v + t;
    }
    if (RW == 1) return v;
    __syncthreads();                      // `red` may still be read from the previous reduction
    if (lane == 0) red[warp] = v;
    __syncthreads();
    float r = red[0];
#pragma unroll
    for (int w = 1; w < RW; ++w) r = MAX ? fmaxf(r, red[w]) : r + red[w];   // fixed order: deterministic
    return r;
}

template <typename T, int VPL, int RW>
__global__ void __launch_bounds__(256)
norm_quant_rows_kernel(const T* __restrict__ X, int M, int K, const float* __restrict__ gamma,
                       const float* __restrict__ beta, int kind, float eps, T* __restrict__ Xn,
                       int8_t* __restrict__ Xq, float* __restrict__ scale) {
    __shared__ float red[8];
    pdl_wait_prior_grid();
    pdl_launch_dependents();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t row = RW == 1 ? static_cast<int64_t>(blockIdx.x) * 8 + warp : blockIdx.x;
    const bool live = row < M;            // RW == 1 only: whole warps of the last CTA may be idle
    const int64_t r = live ? row : 0;
    const T* x = X + r * K;
    const int nvec = K >> 3;
    const int v0 = RW == 1 ? lane : threadIdx.x;
    constexpr int STEP = 32 * RW;
    Raw8<T> raw[VPL];
#pragma unroll
    for (int i = 0; i < VPL; ++i)
        if (v0 + STEP * i < nvec) load_raw(x + 8 * (v0 + STEP * i), raw[i]);
    const float inv_k = 1.0f / static_cast<float>(K);
    float mu = 0.0f;
    if (kind == ARIA_NORM_LAYER) {
        float s = 0.0f;
#pragma unroll
        for (int i = 0; i < VPL; ++i)
            if (v0 + STEP * i < nvec) {
                float v[8];
                unpack8(raw[i], v);
#pragma unroll
                for (int j = 0; j < 8; ++j) s += v[j];
            }
        mu = row_reduce<RW, false>(s, red, lane, warp) * inv_k;
    }
    float ss = 0.0f;
#pragma unroll
    for (int i = 0; i < VPL; ++i)
        if (v0 + STEP * i < nvec) {
            float v[8];
            unpack8(raw[i], v);
#pragma unroll
            for (int j = 0; j < 8; ++j) ss = fmaf(v[j] - mu, v[j] - mu, ss);
        }
    const float var = row_reduce<RW, false>(ss, red, lane, warp) * inv_k;
    const float rstd = __fdiv_rn(1.0f, __fsqrt_rn(var + eps));
    // normalise, round to the activation dtype, keep the rounded values (packed as the input was)
    float a = 0.0f;
#pragma unroll
    for (int i = 0; i < VPL; ++i) {
        const int idx = v0 + STEP * i;
        if (idx < nvec) {
            float v[8], g[8], b[8];
            unpack8(raw[i], v);
            load8<float>(gamma + 8 * idx, g);
            if (beta) load8<float>(beta + 8 * idx, b);
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                v[j] = round_to<T>(fmaf((v[j] - mu) * rstd, g[j], beta ? b[j] : 0.0f));
                a = fmaxf(a, fabsf(v[j]));
            }
            if (Xn && live) store8(Xn + r * K + 8 * idx, v);
            if constexpr (sizeof(T) == 2) {
                raw[i].a.x = (__float_as_uint(v[0]) >> 16) | (__float_as_uint(v[1]) & 0xFFFF0000u);
                raw[i].a.y = (__float_as_uint(v[2]) >> 16) | (__float_as_uint(v[3]) & 0xFFFF0000u);
                raw[i].a.z = (__float_as_uint(v[4]) >> 16) | (__float_as_uint(v[5]) & 0xFFFF0000u);
                raw[i].a.w = (__float_as_uint(v[6]) >> 16) | (__float_as_uint(v[7]) & 0xFFFF0000u);
            } else {
                raw[i].a = make_float4(v[0], v[1], v[2], v[3]);
                raw[i].b = make_float4(v[4], v[5], v[6], v[7]);
            }
        }
    }
    a = row_reduce<RW, true>(a, red, lane, warp);
    const float s = a > 0.0f ? __fdiv_rn(a, 127.0f) : 1.0f;
    if (v0 == 0 && live) scale[row] = s;
    const FastQ f = make_fastq(s);
#pragma unroll
    for (int i = 0; i < VPL; ++i) {
        const int idx = v0 + STEP * i;
        if (idx < nvec && live) {
            float v[8];
            unpack8(raw[i], v);
            uint2 o;
            if (!f.ok || !quant8_fast(v, f, o)) o = quant8_i8(v, s);
            *reinterpret_cast<uint2*>(Xq + r * K + 8 * idx) = o;
        }
    }
}

// ---- bf16 rows up to 8192 elements (the DiT widths): `tpr` threads per row, VPT 16-byte vectors per thread, fp32
// arithmetic on pairs (add / fma .f32x2), ~10 instructions per element; see quant_rows_bf16_kernel for the why.
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) {
    uint64_t d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ uint64_t bf16x2_to_f2(uint32_t w) {
    return pack_f2(__uint_as_float(w << 16), __uint_as_float(w & 0xFFFF0000u));
}
__device__ __forceinline__ float hsum2(uint64_t v) {
    float lo, hi;
    unpack_f2(v, lo, hi);
    return lo + hi;
}
// reduce over the tpr threads of a row; `red` is this reduction's own 8 floats
template <bool MAX>
__device__ __forceinline__ float group_reduce(float v, float* red, int tpr, int lane, int warp) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float t = __shfl_xor_sync(0xffffffffu, v, o);
        v = MAX ? fmaxf(v, t) : v + t;
    }
    if (tpr > 32) {
        if (lane == 0) red[warp] = v;
        __syncthreads();
        const int wpr = tpr >> 5, w0 = (warp / wpr) * wpr;
        v = red[w0];
        for (int w = 1; w < wpr; ++w) v = MAX ? fmaxf(v, red[w0 + w]) : v + red[w0 + w];   // fixed order
    }
    return v;
}

template <int VPT>
__global__ void __launch_bounds__(256)
norm_quant_bf16_kernel(const __nv_bfloat16* __restrict__ X, int M, int K, int tpr, const float* __restrict__ gamma,
                       const float* __restrict__ beta, int kind, float eps, __nv_bfloat16* __restrict__ Xn,
                       int8_t* __restrict__ Xq, float* __restrict__ scale) {
    __shared__ float red[3][8];
    pdl_wait_prior_grid();
    pdl_launch_dependents();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int t = threadIdx.x & (tpr - 1);
    const int64_t row = static_cast<int64_t>(blockIdx.x) * (256 / tpr) + threadIdx.x / tpr;
    const bool live = row < M;
    const int nvec = K >> 3;
    const int64_t roff = (live ? row : 0) * K;
    uint4 raw[VPT];
#pragma unroll
    for (int i = 0; i < VPT; ++i) {
        const int idx = t + tpr * i;
        raw[i] = (live && idx < nvec) ? ld_global_v4(X + roff + 8 * idx) : make_uint4(0, 0, 0, 0);
    }
    const float inv_k = 1.0f / static_cast<float>(K);
    float mu = 0.0f;
    if (kind == ARIA_NORM_LAYER) {
        uint64_t s2 = 0;                       // (0.0f, 0.0f); absent vectors are zeros
#pragma unroll
        for (int i = 0; i < VPT; ++i) {
            s2 = add2(s2, add2(bf16x2_to_f2(raw[i].x), bf16x2_to_f2(raw[i].y)));
            s2 = add2(s2, add2(bf16x2_to_f2(raw[i].z), bf16x2_to_f2(raw[i].w)));
        }
        mu = group_reduce<false>(hsum2(s2), red[0], tpr, lane, warp) * inv_k;
    }
    const uint64_t nmu2 = pack_f2(-mu, -mu);
    uint64_t ss2 = 0;
#pragma unroll
    for (int i = 0; i < VPT; ++i)
        if (t + tpr * i < nvec) {
            const uint32_t w[4] = {raw[i].x, raw[i].y, raw[i].z, raw[i].w};
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint64_t d = add2(bf16x2_to_f2(w[j]), nmu2);
                ss2 = fma2(d, d, ss2);
            }
        }
    const float var = group_reduce<false>(hsum2(ss2), red[1], tpr, lane, warp) * inv_k;
    const float rstd = __fdiv_rn(1.0f, __fsqrt_rn(var + eps));
    const uint64_t rstd2 = pack_f2(rstd, rstd);
    uint32_t amax = 0;
#pragma unroll
    for (int i = 0; i < VPT; ++i) {
        const int idx = t + tpr * i;
        if (idx < nvec) {
            const float4 g0 = ld_global_f4(gamma + 8 * idx), g1 = ld_global_f4(gamma + 8 * idx + 4);
            float4 b0 = make_float4(0, 0, 0, 0), b1 = b0;
            if (beta) { b0 = ld_global_f4(beta + 8 * idx); b1 = ld_global_f4(beta + 8 * idx + 4); }
            const uint64_t g[4] = {pack_f2(g0.x, g0.y), pack_f2(g0.z, g0.w), pack_f2(g1.x, g1.y), pack_f2(g1.z, g1.w)};
            const uint64_t b[4] = {pack_f2(b0.x, b0.y), pack_f2(b0.z, b0.w), pack_f2(b1.x, b1.y), pack_f2(b1.z, b1.w)};
            const uint32_t w[4] = {raw[i].x, raw[i].y, raw[i].z, raw[i].w};
            uint32_t o[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint64_t d = add2(bf16x2_to_f2(w[j]), nmu2);
                const uint64_t n = fma2(mul2(d, rstd2), g[j], b[j]);
                float lo, hi;
                unpack_f2(n, lo, hi);
                asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(o[j]) : "f"(hi), "f"(lo));
                amax = __vmaxu2(o[j] & 0x7FFF7FFFu, amax);
            }
            raw[i] = make_uint4(o[0], o[1], o[2], o[3]);
            if (Xn && live) *reinterpret_cast<uint4*>(Xn + roff + 8 * idx) = raw[i];
        }
    }
    const float a = group_reduce<true>(absmax_bf16x2_to_f32(amax), red[2], tpr, lane, warp);
    const float s = a > 0.0f ? __fdiv_rn(a, 127.0f) : 1.0f;
    if (t == 0 && live) scale[row] = s;
    const FastQ2 f = make_fastq2(s);
#pragma unroll
    for (int i = 0; i < VPT; ++i) {
        const int idx = t + tpr * i;
        if (live && idx < nvec) {
            uint2 o;
            if (!f.ok || !quant8_fast_bf16(raw[i], f, o)) {
                float v[8];
                Raw8<__nv_bfloat16> r8;
                r8.a = raw[i];
                unpack8(r8, v);
                o = quant8_i8(v, s);
            }
            *reinterpret_cast<uint2*>(Xq + roff + 8 * idx) = o;
        }
    }
}

template <typename T, int VPL, int RW>
static cudaError_t launch_nq(const void* X, int M, int K, const float* gamma, const float* beta, int kind, float eps,
                             void* Xn, int8_t* q, float* s, cudaLaunchConfig_t& cfg) {
    cfg.blockDim = dim3(256);
    cfg.gridDim = dim3(RW == 1 ? (M + 7) / 8 : M);
    return cudaLaunchKernelEx(&cfg, norm_quant_rows_kernel<T, VPL, RW>, static_cast<const T*>(X), M, K, gamma, beta, kind,
                              eps, static_cast<T*>(Xn), q, s);
}

template <typename T>
static cudaError_t dispatch_nq(const void* X, int M, int K, const float* gamma, const float* beta, int kind, float eps,
                               void* Xn, int8_t* q, float* s, cudaLaunchConfig_t& cfg, bool* ok) {
    const int nvec = K / 8;
    *ok = true;
    if (nvec <= 64) return launch_nq<T, 2, 1>(X, M, K, gamma, beta, kind, eps, Xn, q, s, cfg);
    if (nvec <= 192) return launch_nq<T, 6, 1>(X, M, K, gamma, beta, kind, eps, Xn, q, s, cfg);     // d_model 1024 / 1536
    if (nvec <= 1024) return launch_nq<T, 4, 8>(X, M, K, gamma, beta, kind, eps, Xn, q, s, cfg);    // up to 8192
    if (nvec <= 3072) return launch_nq<T, 12, 8>(X, M, K, gamma, beta, kind, eps, Xn, q, s, cfg);   // up to 24576
    *ok = false;
    return cudaSuccess;
}

int launch_norm_quant(const void* X, int xt, int M, int K, const float* gamma, const float* beta, int kind, float eps,
                      void* Xn, int8_t* q, float* s, cudaStream_t st, bool pdl) {
    cudaLaunchConfig_t cfg = {};
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl ? 1 : 0;
    const int nvec = K / 8;
    if (xt == ARIA_BF16 && nvec <= 1024) {
        int tpr = 32;
        while (tpr < 256 && tpr * 3 < nvec) tpr *= 2;
        const int vpt = (nvec + tpr - 1) / tpr;
        cfg.blockDim = dim3(256);
        const int rpc = 256 / tpr;
        cfg.gridDim = dim3((M + rpc - 1) / rpc);
        const __nv_bfloat16* x = static_cast<const __nv_bfloat16*>(X);
        __nv_bfloat16* xn = static_cast<__nv_bfloat16*>(Xn);
        cudaError_t e;
        if (vpt == 1) e = cudaLaunchKernelEx(&cfg, norm_quant_bf16_kernel<1>, x, M, K, tpr, gamma, beta, kind, eps, xn, q, s);
        else if (vpt == 2) e = cudaLaunchKernelEx(&cfg, norm_quant_bf16_kernel<2>, x, M, K, tpr, gamma, beta, kind, eps, xn, q, s);
        else if (vpt == 3) e = cudaLaunchKernelEx(&cfg, norm_quant_bf16_kernel<3>, x, M, K, tpr, gamma, beta, kind, eps, xn, q, s);
        else e = cudaLaunchKernelEx(&cfg, norm_quant_bf16_kernel<4>, x, M, K, tpr, gamma, beta, kind, eps, xn, q, s);
        return e == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
    }
    bool ok = false;
    const cudaError_t e = xt == ARIA_BF16
                              ? dispatch_nq<__nv_bfloat16>(X, M, K, gamma, beta, kind, eps, Xn, q, s, cfg, &ok)
                              : dispatch_nq<float>(X, M, K, gamma, beta, kind, eps, Xn, q, s, cfg, &ok);
    if (!ok) return ARIA_ERR_SHAPE;
    return e == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
}

}  // namespace aria
