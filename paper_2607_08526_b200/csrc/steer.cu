// steer.cu -- NEXT-3: in-graph activation steering of the residual stream (eq. 2,
// projection variant L192 / L248).  One warp per token row; the strength is read from DEVICE memory on
// every launch, so a captured graph is replayed with a new strength without re-capture (L77: "reads a
// strength value refreshed each step ... enabling it triggers no re-capture"), and strength == 0 returns
// before any store: the output is bit-identical to the unsteered pass (L77, L98).
//   op 0 (add):      h[t,:] += alpha * hbar_norm * d[:]                      (eq. 2)
//   op 1 (project):  c_t = sum_j h[t,j] d[j];  h[t,:] += beta * c_t * d[:]   (L192)
// fp32 arithmetic: one multiply for the row's coefficient, one FMA per element, one rounding to the
// storage type.  HBM bound: reads and writes the [M, D] tensor once (the projection reads it twice, the
// second time from L1/L2).
#include "internal.cuh"

namespace aria {

__device__ __forceinline__ void ld8(const float* p, float (&v)[8]) {
    const float4 a = *reinterpret_cast<const float4*>(p), b = *reinterpret_cast<const float4*>(p + 4);
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
}
__device__ __forceinline__ void ld8(const __nv_bfloat16* p, float (&v)[8]) {
    const uint4 a = *reinterpret_cast<const uint4*>(p);
    const uint32_t w[4] = {a.x, a.y, a.z, a.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        v[2 * i] = __uint_as_float(w[i] << 16);
        v[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    }
}
__device__ __forceinline__ void st8(float* p, const float (&v)[8]) {
    *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
    *reinterpret_cast<float4*>(p + 4) = make_float4(v[4], v[5], v[6], v[7]);
}
__device__ __forceinline__ void st8(__nv_bfloat16* p, const float (&v)[8]) {
    uint32_t w[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        __nv_bfloat162 t = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]);
        w[i] = *reinterpret_cast<uint32_t*>(&t);
    }
    *reinterpret_cast<uint4*>(p) = make_uint4(w[0], w[1], w[2], w[3]);
}

template <typename T>
__global__ void __launch_bounds__(256) steer_kernel(T* __restrict__ H, int M, int D, const float* __restrict__ d,
                                                    const float* __restrict__ strength, float hbar_norm, int op) {
    const float s = *strength;                 // device scalar, refreshed by the host between replays
    if (s == 0.0f) return;                     // bit-identical to the base model
    const int lane = threadIdx.x & 31;
    const int row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= M) return;
    T* h = H + static_cast<size_t>(row) * D;
    const int nvec = D >> 3;
    float coef = s * hbar_norm;
    if (op == 1) {
        float c = 0.0f;
        for (int i = lane; i < nvec; i += 32) {
            float hv[8], dv[8];
            ld8(h + 8 * i, hv);
            ld8(d + 8 * i, dv);
#pragma unroll
            for (int j = 0; j < 8; ++j) c = fmaf(hv[j], dv[j], c);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
        coef = s * c;
    }
    for (int i = lane; i < nvec; i += 32) {
        float hv[8], dv[8];
        ld8(h + 8 * i, hv);
        ld8(d + 8 * i, dv);
#pragma unroll
        for (int j = 0; j < 8; ++j) hv[j] = fmaf(coef, dv[j], hv[j]);
        st8(h + 8 * i, hv);
    }
}

int launch_steer(void* H, int ht, int M, int D, const float* d, const float* strength, float hbar_norm, int op,
                 cudaStream_t st) {
    const int rows_per_cta = 8;
    const unsigned grid = static_cast<unsigned>((M + rows_per_cta - 1) / rows_per_cta);
    if (ht == ARIA_F32)
        steer_kernel<float><<<grid, 32 * rows_per_cta, 0, st>>>(static_cast<float*>(H), M, D, d, strength, hbar_norm, op);
    else
        steer_kernel<__nv_bfloat16><<<grid, 32 * rows_per_cta, 0, st>>>(static_cast<__nv_bfloat16*>(H), M, D, d, strength,
                                                                      hbar_norm, op);
    return cudaGetLastError() == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
}

}  // namespace aria
