// quant.cu -- S0 / S1: symmetric int8 row quantisation and int4 group quantisation.
// HBM-bound scans: 128-bit loads, warp-shuffle + smem block reduction for the absmax, one
// pass over DRAM (the row is kept in registers between the absmax and the rounding).
// Arithmetic (include/aria.h, R2-R4, R7): IEEE fp32 division (__fdiv_rn), round
// half to even (__float2int_rn), clamp; never a reciprocal or fast-math shortcut, so codes and
// scales are bit-identical to the definition.
#include "internal.cuh"
#include "quant_dev.cuh"

namespace aria {

constexpr int QROW_MAX_THREADS = 256;
constexpr int QROW_CACHE = 4;  // 8-element vectors kept in registers per thread

// One CTA per row.  R1..R4: a = max|x|; s = a > 0 ? a/127 : 1; q = clamp(rint(x/s), +-127).
template <typename T>
__global__ void __launch_bounds__(QROW_MAX_THREADS)
quant_rows_i8_kernel(const T* __restrict__ X, int K, int8_t* __restrict__ Xq,
                     float* __restrict__ scale, const float* known_absmax, float* zero_absmax) {
    __shared__ float red[QROW_MAX_THREADS / 32];
    pdl_wait_prior_grid();
    const int64_t row = blockIdx.x;
    const T* x = X + row * K;
    int8_t* q = Xq + row * K;
    const int nvec = K >> 3;
    const int tid = threadIdx.x, nthr = blockDim.x;

    float v[QROW_CACHE][8];
    float a = 0.0f;
#pragma unroll
    for (int i = 0; i < QROW_CACHE; ++i) {
        const int idx = tid + i * nthr;
        if (idx < nvec) {
            load8<T>(x + 8 * idx, v[i]);
            a = absmax8(v[i], a);
        }
    }
    for (int idx = tid + QROW_CACHE * nthr; idx < nvec; idx += nthr) {  // K > 8*CACHE*threads
        float t[8];
        load8<T>(x + 8 * idx, t);
        a = absmax8(t, a);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a = fmaxf(a, __shfl_xor_sync(0xffffffffu, a, o));
    if ((tid & 31) == 0) red[tid >> 5] = a;
    __syncthreads();
    const int nwarp = nthr >> 5;
    a = red[0];
    for (int w = 1; w < nwarp; ++w) a = fmaxf(a, red[w]);
    // fused S1: the producing epilogue already reduced this row (same value, taken after the wait above).
    // `wrong`: the supplied maximum is below the row's own (a stale or foreign buffer) or not a number --
    // the division-free rounding would wrap instead of saturating, so the row takes the clamping path.
    bool wrong = false;
    if (known_absmax) {
        const float own = a;
        asm volatile("ld.global.f32 %0, [%1];" : "=f"(a) : "l"(known_absmax + row) : "memory");
        wrong = !(own <= a);
    }

    const float s = a > 0.0f ? __fdiv_rn(a, 127.0f) : 1.0f;
    if (known_absmax && zero_absmax == known_absmax) __syncthreads();   // every thread has read it before it is cleared
    if (tid == 0) {
        scale[row] = s;
        if (zero_absmax) zero_absmax[row] = 0.0f;
    }
    pdl_launch_dependents();
    const FastQ f = make_fastq(s);
#pragma unroll
    for (int i = 0; i < QROW_CACHE; ++i) {
        const int idx = tid + i * nthr;
        if (idx < nvec) {
            uint2 o;
            if (!f.ok || wrong || !quant8_fast(v[i], f, o)) o = quant8_i8(v[i], s);
            *reinterpret_cast<uint2*>(q + 8 * idx) = o;
        }
    }
    for (int idx = tid + QROW_CACHE * nthr; idx < nvec; idx += nthr) {
        float t[8];
        load8<T>(x + 8 * idx, t);
        uint2 o;
        if (!f.ok || wrong || !quant8_fast(t, f, o)) o = quant8_i8(t, s);
        *reinterpret_cast<uint2*>(q + 8 * idx) = o;
    }
}

// One WARP per row (K <= 8 * 32 * VPL): every lane issues all its 16-byte loads up front, the
// absmax is a pure shuffle reduction, no shared memory and no block barrier.
template <typename T, int VPL>
__global__ void __launch_bounds__(256)
quant_rows_i8_warp_kernel(const T* __restrict__ X, int R, int K, int8_t* __restrict__ Xq,
                          float* __restrict__ scale, const float* known_absmax, float* zero_absmax) {
    pdl_wait_prior_grid();
    pdl_launch_dependents();
    const int lane = threadIdx.x & 31;
    const int64_t row = static_cast<int64_t>(blockIdx.x) * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= R) return;
    const T* x = X + row * K;
    int8_t* q = Xq + row * K;
    const int nvec = K >> 3;
    Raw8<T> raw[VPL];
#pragma unroll
    for (int i = 0; i < VPL; ++i) {
        const int idx = lane + 32 * i;
        if (idx < nvec) load_raw(x + 8 * idx, raw[i]);
    }
    float a = 0.0f;
#pragma unroll
    for (int i = 0; i < VPL; ++i) {
        if (lane + 32 * i < nvec) {
            float v[8];
            unpack8(raw[i], v);
            a = absmax8(v, a);
        }
    }
    bool wrong = false;   // this lane holds a value above the supplied maximum (or that is NaN): clamp, see above
    if (known_absmax) {   // fused S1: reduced by the producing epilogue (warp-uniform branch)
        const float own = a;
        asm volatile("ld.global.f32 %0, [%1];" : "=f"(a) : "l"(known_absmax + row) : "memory");
        wrong = !(own <= a);
        __syncwarp();     // every lane has read absmax[row] before lane 0 may clear it below
    } else {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) a = fmaxf(a, __shfl_xor_sync(0xffffffffu, a, o));
    }
    const float s = a > 0.0f ? __fdiv_rn(a, 127.0f) : 1.0f;
    if (lane == 0) {
        scale[row] = s;
        if (zero_absmax) zero_absmax[row] = 0.0f;
    }
    const FastQ f = make_fastq(s);
#pragma unroll
    for (int i = 0; i < VPL; ++i) {
        const int idx = lane + 32 * i;
        if (idx < nvec) {
            float v[8];
            unpack8(raw[i], v);
            uint2 o;
            if (!f.ok || wrong || !quant8_fast(v, f, o)) o = quant8_i8(v, s);
            *reinterpret_cast<uint2*>(q + 8 * idx) = o;
        }
    }
}

// int4, group 32 along K: 4 threads per group, 8 elements each (R3, R4, R7, R8).
template <typename T>
__global__ void __launch_bounds__(256)
quant_groups_i4_kernel(const T* __restrict__ W, int64_t n_vec, uint8_t* __restrict__ Wq4,
                       uint16_t* __restrict__ g_scale) {
    const int64_t idx = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    const bool live = idx < n_vec;  // n_vec is a multiple of 4, so a group is never split
    float v[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    if (live) load8<T>(W + 8 * idx, v);
    float a = absmax8(v, 0.0f);
    a = fmaxf(a, __shfl_xor_sync(0xffffffffu, a, 1));
    a = fmaxf(a, __shfl_xor_sync(0xffffffffu, a, 2));
    const __half h = __float2half_rn(__fdiv_rn(a, 7.0f));
    const float sg = __half2float(h);
    uint32_t packed = 0;
    if (sg != 0.0f) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            packed |= (static_cast<uint32_t>(quant1(v[i], sg, 7)) & 0xFu) << (4 * i);
    }
    if (live) {
        reinterpret_cast<uint32_t*>(Wq4)[idx] = packed;  // codes 8idx..8idx+7: low nibble = even k
        if ((idx & 3) == 0) g_scale[idx >> 2] = __half_as_ushort(h);
    }
}

// bf16 rows up to 8192 elements: `tpr` threads per row (32..256, a power of two; 256 / tpr rows per CTA), each
// holding VPT 16-byte vectors, everything packed: the absmax runs on bf16x2 (HMNMX2), the rounding on fp32
// pairs (FFMA2), ~5 instructions per element instead of ~20 -- these passes were bound by instruction issue
// at one warp per row (ncu r1c / r2a: 17 % of HBM bandwidth, 18-20 % warps active), not by memory.
template <int VPT>
__global__ void __launch_bounds__(256)
quant_rows_bf16_kernel(const __nv_bfloat16* __restrict__ X, int R, int K, int tpr, int8_t* __restrict__ Xq,
                       float* __restrict__ scale, const float* known_absmax, float* zero_absmax, int check_known) {
    __shared__ float red[8];
    pdl_wait_prior_grid();
    pdl_launch_dependents();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int t = threadIdx.x & (tpr - 1);
    const int64_t row = static_cast<int64_t>(blockIdx.x) * (256 / tpr) + threadIdx.x / tpr;
    const bool live = row < R;
    const int nvec = K >> 3;
    const __nv_bfloat16* x = X + (live ? row : 0) * K;
    uint4 raw[VPT];
#pragma unroll
    for (int i = 0; i < VPT; ++i) {
        const int idx = t + tpr * i;
        raw[i] = (live && idx < nvec) ? ld_global_v4(x + 8 * idx) : make_uint4(0, 0, 0, 0);
    }
    float a;
    bool wrong = false;
    if (known_absmax) {            // fused S1: reduced by the producing epilogue
        a = 0.0f;
        if (live) asm volatile("ld.global.f32 %0, [%1];" : "=f"(a) : "l"(known_absmax + row) : "memory");
        if (zero_absmax == known_absmax) {   // all of the row's threads have read it before thread 0 clears it
            if (tpr > 32) __syncthreads();
            else __syncwarp();
        }
        // check_known (a maximum supplied through the public aria_round_act_int8, not by this library's own
        // epilogues): a thread holding a value above it, or a NaN maximum, takes the clamping path
        if (check_known) {
            uint32_t acc = 0;
#pragma unroll
            for (int i = 0; i < VPT; ++i) acc = absmax8_bf16(raw[i], acc);
            wrong = !(absmax_bf16x2_to_f32(acc) <= a);
        }
    } else {
        uint32_t acc = 0;
#pragma unroll
        for (int i = 0; i < VPT; ++i) acc = absmax8_bf16(raw[i], acc);
        a = absmax_bf16x2_to_f32(acc);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) a = fmaxf(a, __shfl_xor_sync(0xffffffffu, a, o));
        if (tpr > 32) {
            if (lane == 0) red[warp] = a;
            __syncthreads();
            const int wpr = tpr >> 5, w0 = (warp / wpr) * wpr;
            a = red[w0];
            for (int w = 1; w < wpr; ++w) a = fmaxf(a, red[w0 + w]);
        }
    }
    const float s = a > 0.0f ? __fdiv_rn(a, 127.0f) : 1.0f;
    if (t == 0 && live) {
        scale[row] = s;
        if (zero_absmax) zero_absmax[row] = 0.0f;
    }
    const FastQ2 f = make_fastq2(s);
    int8_t* q = Xq + (live ? row : 0) * K;
#pragma unroll
    for (int i = 0; i < VPT; ++i) {
        const int idx = t + tpr * i;
        if (live && idx < nvec) {
            uint2 o;
            if (!f.ok || wrong || !quant8_fast_bf16(raw[i], f, o)) {
                float v[8];
                Raw8<__nv_bfloat16> r8;
                r8.a = raw[i];
                unpack8(r8, v);
                o = quant8_i8(v, s);
            }
            *reinterpret_cast<uint2*>(q + 8 * idx) = o;
        }
    }
}

template <typename T, int VPL>
static cudaError_t launch_warp_rows(const void* X, int R, int C, int8_t* q, float* s,
                                    cudaLaunchConfig_t& cfg, const float* known, float* zero) {
    constexpr int WARPS = 8;
    cfg.blockDim = dim3(32 * WARPS);
    cfg.gridDim = dim3((R + WARPS - 1) / WARPS);
    return cudaLaunchKernelEx(&cfg, quant_rows_i8_warp_kernel<T, VPL>, static_cast<const T*>(X), R, C, q, s, known, zero);
}

int launch_quant_rows_i8(const void* X, int xt, int R, int C, int8_t* q, float* s, cudaStream_t st,
                         bool pdl, const float* known, float* zero, bool check_known) {
    const int ck = check_known ? 1 : 0;
    const int nvec = C / 8;
    if (xt == ARIA_BF16 && nvec <= 1024) {
        int tpr = 32;
        while (tpr < 256 && tpr * 3 < nvec) tpr *= 2;
        const int vpt = (nvec + tpr - 1) / tpr;
        cudaLaunchConfig_t cfg = {};
        cfg.stream = st;
        cfg.blockDim = dim3(256);
        const int rpc = 256 / tpr;
        cfg.gridDim = dim3((R + rpc - 1) / rpc);
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at;
        cfg.numAttrs = pdl ? 1 : 0;
        const __nv_bfloat16* x = static_cast<const __nv_bfloat16*>(X);
        cudaError_t e;
        if (vpt == 1) e = cudaLaunchKernelEx(&cfg, quant_rows_bf16_kernel<1>, x, R, C, tpr, q, s, known, zero, ck);
        else if (vpt == 2) e = cudaLaunchKernelEx(&cfg, quant_rows_bf16_kernel<2>, x, R, C, tpr, q, s, known, zero, ck);
        else if (vpt == 3) e = cudaLaunchKernelEx(&cfg, quant_rows_bf16_kernel<3>, x, R, C, tpr, q, s, known, zero, ck);
        else e = cudaLaunchKernelEx(&cfg, quant_rows_bf16_kernel<4>, x, R, C, tpr, q, s, known, zero, ck);
        return e == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
    }
    {   // warp-per-row variants (fp32 rows, and bf16 rows wider than 8192 elements): rows up to 3072 elements (wider rows: one CTA per row, below; a 24-vector
        // warp-per-row variant for 6144-element bf16 rows was measured slower: 2.18 vs 2.08 ms per C5 step)
        cudaLaunchConfig_t cfg = {};
        cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at;
        cfg.numAttrs = pdl ? 1 : 0;
        const int vpl = (nvec + 31) / 32;
        cudaError_t e = cudaErrorInvalidValue;
        bool done = true;
        if (xt == ARIA_BF16) {
            if (vpl <= 2) e = launch_warp_rows<__nv_bfloat16, 2>(X, R, C, q, s, cfg, known, zero);
            else if (vpl <= 6) e = launch_warp_rows<__nv_bfloat16, 6>(X, R, C, q, s, cfg, known, zero);
            else if (vpl <= 12) e = launch_warp_rows<__nv_bfloat16, 12>(X, R, C, q, s, cfg, known, zero);
            else done = false;
        } else {
            if (vpl <= 2) e = launch_warp_rows<float, 2>(X, R, C, q, s, cfg, known, zero);
            else if (vpl <= 6) e = launch_warp_rows<float, 6>(X, R, C, q, s, cfg, known, zero);
            else if (vpl <= 12) e = launch_warp_rows<float, 12>(X, R, C, q, s, cfg, known, zero);
            else done = false;
        }
        if (done) return e == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
    }
    int threads = ((nvec + 31) / 32) * 32;
    threads = threads > QROW_MAX_THREADS ? QROW_MAX_THREADS : threads;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(R);
    cfg.blockDim = dim3(threads);
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl ? 1 : 0;
    cudaError_t e;
    if (xt == ARIA_F32)
        e = cudaLaunchKernelEx(&cfg, quant_rows_i8_kernel<float>, static_cast<const float*>(X), C, q, s, known, zero);
    else
        e = cudaLaunchKernelEx(&cfg, quant_rows_i8_kernel<__nv_bfloat16>,
                               static_cast<const __nv_bfloat16*>(X), C, q, s, known, zero);
    return e == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
}

int launch_quant_groups_i4(const void* W, int wt, int N, int K, uint8_t* q4, uint16_t* sg,
                           cudaStream_t st) {
    const int64_t n_vec = static_cast<int64_t>(N) * K / 8;
    const int threads = 256;
    const unsigned blocks = static_cast<unsigned>((n_vec + threads - 1) / threads);
    if (wt == ARIA_F32)
        quant_groups_i4_kernel<float><<<blocks, threads, 0, st>>>(static_cast<const float*>(W), n_vec, q4, sg);
    else
        quant_groups_i4_kernel<__nv_bfloat16><<<blocks, threads, 0, st>>>(
            static_cast<const __nv_bfloat16*>(W), n_vec, q4, sg);
    return cudaGetLastError() == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
}

}  // namespace aria
