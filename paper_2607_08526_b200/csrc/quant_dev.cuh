// quant_dev.cuh -- device helpers of the symmetric int8 row quantiser (S0 int8, S1), shared by the
// stand-alone quantiser kernels (quant.cu) and the quantiser side job inside the W8A8 GEMM kernel
// (gemm_w8a8.cu).  Arithmetic: include/aria.h, R2-R4.
#pragma once
#include "ptx.cuh"

namespace aria {

// 16-byte global loads that stay BELOW griddepcontrol.wait: a non-coherent (ld.global.nc) load is a
// pure value to the compiler, which hoisted it above the wait of the quantiser kernels -- under
// programmatic dependent launch the previous grid is still writing X at that point.
__device__ __forceinline__ uint4 ld_global_v4(const void* p) {
    uint4 v;
    asm volatile("ld.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ float4 ld_global_f4(const void* p) {
    const uint4 v = ld_global_v4(p);
    return make_float4(__uint_as_float(v.x), __uint_as_float(v.y), __uint_as_float(v.z), __uint_as_float(v.w));
}
template <typename T>
__device__ __forceinline__ void load8(const T* p, float (&v)[8]);

template <>
__device__ __forceinline__ void load8<float>(const float* p, float (&v)[8]) {
    const float4 a = ld_global_f4(p);
    const float4 b = ld_global_f4(p + 4);
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
    v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
}
template <>
__device__ __forceinline__ void load8<__nv_bfloat16>(const __nv_bfloat16* p, float (&v)[8]) {
    const uint4 a = ld_global_v4(p);
    const uint32_t w[4] = {a.x, a.y, a.z, a.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        v[2 * i] = __uint_as_float(w[i] << 16);
        v[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    }
}

// Raw (still packed) 8-element vectors: what the warp-per-row kernel keeps in registers.
template <typename T> struct Raw8;
template <> struct Raw8<float> { float4 a, b; };
template <> struct Raw8<__nv_bfloat16> { uint4 a; };
__device__ __forceinline__ void load_raw(const float* p, Raw8<float>& r) {
    r.a = ld_global_f4(p);
    r.b = ld_global_f4(p + 4);
}
__device__ __forceinline__ void load_raw(const __nv_bfloat16* p, Raw8<__nv_bfloat16>& r) {
    r.a = ld_global_v4(p);
}
__device__ __forceinline__ void unpack8(const Raw8<float>& r, float (&v)[8]) {
    v[0] = r.a.x; v[1] = r.a.y; v[2] = r.a.z; v[3] = r.a.w;
    v[4] = r.b.x; v[5] = r.b.y; v[6] = r.b.z; v[7] = r.b.w;
}
__device__ __forceinline__ void unpack8(const Raw8<__nv_bfloat16>& r, float (&v)[8]) {
    const uint32_t w[4] = {r.a.x, r.a.y, r.a.z, r.a.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        v[2 * i] = __uint_as_float(w[i] << 16);
        v[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    }
}

__device__ __forceinline__ float absmax8(const float (&v)[8], float a) {
#pragma unroll
    for (int i = 0; i < 8; ++i) a = fmaxf(a, fabsf(v[i]));
    return a;
}

__device__ __forceinline__ int quant1(float x, float s, int lim) {
    int q = __float2int_rn(__fdiv_rn(x, s));
    return max(-lim, min(lim, q));
}

// Exact rint(fl32(x / s)) without a division per element.  With r = RN(1/s), r_lo = r (1 - 2^-20) and
// r_hi = r (1 + 2^-20) bracket 1/s by far more than the rounding of r, so for every x the exact
// quotient AND its fp32 rounding lie between x*r_lo and x*r_hi.  fma(x, r_*, 1.5*2^23) rounds the
// exact product to an integer (ties to even) in the low mantissa bits; rint is monotone, so if both
// ends give the same integer, rint(fl32(x/s)) is that integer (a tie strictly inside the bracket
// would separate the two ends).  Otherwise (|x/s| within ~1e-4 of a .5 boundary, probability ~2e-4)
// the caller falls back to the IEEE division.  |x/s| <= 127 (1 + 2^-23): no clamp is needed.
struct FastQ {
    float r_lo, r_hi;
    bool ok;  // false: s is outside the range where r is finite and normal -> always divide
};
__device__ __forceinline__ FastQ make_fastq(float s) {
    FastQ f;
    const float r = __frcp_rn(s);
    f.r_lo = r * 0.99999904632568359375f;   // 1 - 2^-20
    f.r_hi = r * 1.00000095367431640625f;   // 1 + 2^-20
    f.ok = (s > 1e-30f) && (s < 1e30f);
    return f;
}
constexpr float QMAGIC = 12582912.0f;  // 1.5 * 2^23: float bits 0x4B400000 + q

// Quantise 8 values; returns false if any needs the exact-division path.
__device__ __forceinline__ bool quant8_fast(const float (&v)[8], const FastQ& f, uint2& out) {
    uint32_t y[8];
    bool same = true;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const uint32_t a = __float_as_uint(fmaf(v[i], f.r_lo, QMAGIC));
        const uint32_t b = __float_as_uint(fmaf(v[i], f.r_hi, QMAGIC));
        same = same && (a == b);
        y[i] = a;
    }
    // low byte of each y is the two's-complement code
    out.x = __byte_perm(__byte_perm(y[0], y[1], 0x0040), __byte_perm(y[2], y[3], 0x0040), 0x5410);
    out.y = __byte_perm(__byte_perm(y[4], y[5], 0x0040), __byte_perm(y[6], y[7], 0x0040), 0x5410);
    return same;
}

__device__ __forceinline__ uint2 quant8_i8(const float (&v)[8], float s) {
    uint32_t lo = 0, hi = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        lo |= (static_cast<uint32_t>(quant1(v[i], s, 127)) & 0xFFu) << (8 * i);
        hi |= (static_cast<uint32_t>(quant1(v[4 + i], s, 127)) & 0xFFu) << (8 * i);
    }
    return make_uint2(lo, hi);
}

// ------------------------------------------------------------------ packed bf16 fast path
// The same exact rounding as quant8_fast, on 8 bf16 values still packed in a uint4, with two fp32 FMAs per
// instruction (fma.rn.f32x2 is IEEE per lane): per element 1 unpack + 1 FFMA2 + 1 LOP3 + 3/4 PRMT.
struct FastQ2 {
    uint64_t r_lo, r_hi, magic;
    bool ok;
};
__device__ __forceinline__ FastQ2 make_fastq2(float s) {
    const FastQ f = make_fastq(s);
    FastQ2 g;
    g.r_lo = pack_f2(f.r_lo, f.r_lo);
    g.r_hi = pack_f2(f.r_hi, f.r_hi);
    g.magic = pack_f2(QMAGIC, QMAGIC);
    g.ok = f.ok;
    return g;
}
// acc | (a ^ b)
__device__ __forceinline__ uint32_t lop_or_xor(uint32_t acc, uint32_t a, uint32_t b) {
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0xF6;" : "=r"(r) : "r"(acc), "r"(a), "r"(b));   // a | (b ^ c)
    return r;
}
__device__ __forceinline__ bool quant8_fast_bf16(const uint4& raw, const FastQ2& f, uint2& out) {
    const uint32_t w[4] = {raw.x, raw.y, raw.z, raw.w};
    uint32_t y[8];
    uint32_t diff = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        uint32_t a0, a1, b0, b1;
        const uint32_t lo = w[i] << 16, hi = w[i] & 0xFFFF0000u;
        asm("{\n\t.reg .b64 x, a, b;\n\t"
            "mov.b64 x, {%4, %5};\n\t"
            "fma.rn.f32x2 a, x, %6, %8;\n\t"
            "fma.rn.f32x2 b, x, %7, %8;\n\t"
            "mov.b64 {%0, %1}, a;\n\t"
            "mov.b64 {%2, %3}, b;\n\t}"
            : "=r"(a0), "=r"(a1), "=r"(b0), "=r"(b1)
            : "r"(lo), "r"(hi), "l"(f.r_lo), "l"(f.r_hi), "l"(f.magic));
        y[2 * i] = a0;
        y[2 * i + 1] = a1;
        diff |= (a0 ^ b0) | (a1 ^ b1);
    }
    out.x = __byte_perm(__byte_perm(y[0], y[1], 0x0040), __byte_perm(y[2], y[3], 0x0040), 0x5410);
    out.y = __byte_perm(__byte_perm(y[4], y[5], 0x0040), __byte_perm(y[6], y[7], 0x0040), 0x5410);
    return diff == 0;
}
// max |.| of 8 packed bf16 as a packed bf16x2 running maximum (exact: max and abs do not round)
__device__ __forceinline__ uint32_t absmax8_bf16(const uint4& raw, uint32_t acc) {
    const uint32_t w[4] = {raw.x, raw.y, raw.z, raw.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        acc = __vmaxu2(w[i] & 0x7FFF7FFFu, acc);     // |x| of finite bf16 orders like its bit pattern
    }
    return acc;
}
__device__ __forceinline__ float absmax_bf16x2_to_f32(uint32_t acc) {
    return fmaxf(__uint_as_float(acc << 16), __uint_as_float(acc & 0xFFFF0000u));
}

}  // namespace aria
