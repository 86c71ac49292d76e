// gemm_w4a16.cu -- S4: W4A16 linear.  int4 group-32 weights are dequantised ON CHIP to bf16 and
// fed to tcgen05.mma kind::f16 (bf16 x bf16, fp32 accumulators in TMEM).
//
// "Swap-AB": the weight tile is the MMA's M operand (128 output channels on the 128 TMEM lanes)
// and the token tile is the MMA's N operand (TT = 32..256 tokens), so a 32-token batch is a legal
// N = 32 instruction and each dequantised weight feeds TT MACs.
//
// Persistent, warp-specialised, one CTA per SM, 14 warps:
//   warp 0       TMA producer: per k-block the packed int4 tile [128 rows x BK/2 bytes] (32/64-byte
//                swizzle) and the X tile [TT x BK] bf16 (128-byte swizzle) into a ring.
//   warp 1       MMA issuer (one thread): BK/16 tcgen05.mma per k-block, A = dequantised weights,
//                B = X, into one of two TMEM accumulators.
//   warps 2..5   epilogue: tcgen05.ld -> (+bias, GELU, cast) -> Y, or split-K partials.
//   warps 6..13  dequantisers (256 threads, thread = weight row x chunk parity): LDS 16 B (32 codes,
//                one group) -> 32 exact fp32 products q*sg -> cvt.rn.bf16x2 -> STS into the
//                128-byte-swizzled K-major A tile; fence.proxy.async; arrive on `a_full`.
// Exactness of w^ = bf16_rne(q*sg): the nibble n is placed (XOR 8 = offset binary u = q+8) at
// mantissa bit pos in {8,12,16} of 1.0f, giving x = 1 + u*2^(pos-23); one FFMA
// x * (2^(23-pos) sg) - (2^(23-pos)+8) sg has exactly representable addends and the exactly
// representable result q*sg, so fp32 holds q*sg exactly and one cvt.rn rounds it to bf16.
//
// Split-K (small M): a work unit is (tile, k-range); units of a tile write fp32 partials to the
// workspace, the last to arrive (per 32-channel quarter, atomic counter) sums them in split order
// -- deterministic -- and finishes the epilogue.
#include "internal.cuh"

namespace aria {

constexpr int W4_BN = 128;      // output channels per tile = MMA M
constexpr int W4_THREADS = 448;
constexpr int W4_DEQ_WARP0 = 6;
constexpr int W4_DEQ_THREADS = 256;
constexpr int W4_DEQ_WARPS = W4_DEQ_THREADS / 32;

template <int TT, int BK>
struct W4Cfg {
    static constexpr int P_ROW = BK / 2;                       // packed bytes per row per k-block
    static constexpr int P_BYTES = W4_BN * P_ROW;              // 4 or 8 KB
    static constexpr int X_SUB = TT * 128;                     // one 64-column bf16 sub-tile
    static constexpr int X_BYTES = X_SUB * (BK / 64);
    static constexpr int STAGE_BYTES = X_BYTES + P_BYTES;
    static constexpr int A_SUB = W4_BN * 128;                  // 16 KB: 128 rows x 64 bf16
    static constexpr int A_BYTES = A_SUB * (BK / 64);
    static constexpr int NA = BK == 64 ? 3 : 2;                // dequantised A buffers
    static constexpr int STAGES_RAW = (196 * 1024 - NA * A_BYTES) / STAGE_BYTES;
    static constexpr int STAGES = STAGES_RAW > 8 ? 8 : STAGES_RAW;
    static constexpr int ACC_STRIDE = TT;
    static constexpr int TMEM_COLS = 2 * TT < 32 ? 32 : 2 * TT;
    static constexpr int BAR_BYTES = (2 * STAGES + 2 * NA + 4) * 8 + 16;
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + NA * A_BYTES + BAR_BYTES + 1024;
    static_assert(TT == 32 || TT == 64 || TT == 128 || TT == 256, "TT");
    static_assert(BK == 64 || BK == 128, "BK");
    static_assert(STAGES >= 2, "ring too shallow");
    static_assert(SMEM_BYTES <= 227 * 1024, "shared memory");
};

struct W4Params {
    const uint16_t* g_scale;  // fp16 bits [N, K/32]
    const void* bias;         // bf16 [N] or nullptr
    void* Y;
    float* partials;          // [splits, M, N] fp32 (split-K only)
    unsigned* counters;       // [num_tiles * 4], zero between launches (self-resetting)
    int act, out_t;
    int M, N, K;
    int splits;
};

__device__ __forceinline__ uint32_t cvt_bf16x2(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}
__device__ __forceinline__ uint32_t lop_and_xor(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0x6A;" : "=r"(r) : "r"(a), "r"(b), "r"(c));  // (a & b) ^ c
    return r;
}

// 8 codes of one 32-bit word -> 8 exact fp32 products q*sg -> 4 packed bf16x2 (k ascending).
struct GroupConst {
    float s8, c8, s12, c12, s16, c16;
};
__device__ __forceinline__ GroupConst group_const(float sg) {
    GroupConst g;
    g.s8 = sg * 32768.0f;  g.c8 = -(sg * 32776.0f);   // 2^15, 2^15 + 8
    g.s12 = sg * 2048.0f;  g.c12 = -(sg * 2056.0f);   // 2^11, 2^11 + 8
    g.s16 = sg * 128.0f;   g.c16 = -(sg * 136.0f);    // 2^7,  2^7  + 8
    return g;
}
__device__ __forceinline__ uint4 dequant_word(uint32_t w, const GroupConst& g) {
    const uint32_t wa = w << 8, wb = w >> 12;
    const uint32_t M8 = 0x00000F00u, M12 = 0x0000F000u, M16 = 0x000F0000u;
    const uint32_t X8 = 0x3F800800u, X12 = 0x3F808000u, X16 = 0x3F880000u;  // 1.0f | (8 << pos)
    const float e0 = fmaf(__uint_as_float(lop_and_xor(wa, M8, X8)), g.s8, g.c8);
    const float e1 = fmaf(__uint_as_float(lop_and_xor(wa, M12, X12)), g.s12, g.c12);
    const float e2 = fmaf(__uint_as_float(lop_and_xor(wa, M16, X16)), g.s16, g.c16);
    const float e3 = fmaf(__uint_as_float(lop_and_xor(w, M12, X12)), g.s12, g.c12);
    const float e4 = fmaf(__uint_as_float(lop_and_xor(w, M16, X16)), g.s16, g.c16);
    const float e5 = fmaf(__uint_as_float(lop_and_xor(wb, M8, X8)), g.s8, g.c8);
    const float e6 = fmaf(__uint_as_float(lop_and_xor(wb, M12, X12)), g.s12, g.c12);
    const float e7 = fmaf(__uint_as_float(lop_and_xor(wb, M16, X16)), g.s16, g.c16);
    return make_uint4(cvt_bf16x2(e0, e1), cvt_bf16x2(e2, e3), cvt_bf16x2(e4, e5), cvt_bf16x2(e6, e7));
}

__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, const uint4& v) {
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z),
                 "r"(v.w)
                 : "memory");
}

__device__ __forceinline__ float w4_finish(float y, int act) {
    return act == ARIA_ACT_GELU_ERF ? gelu_erf(y) : y;
}
__device__ __forceinline__ void w4_store(void* Y, int out_t, int64_t idx, float y) {
    if (out_t == ARIA_F32)
        static_cast<float*>(Y)[idx] = y;
    else
        static_cast<__nv_bfloat16*>(Y)[idx] = __float2bfloat16_rn(y);
}

template <int TT, int BK>
__global__ void __launch_bounds__(W4_THREADS, 1)
w4a16_gemm_kernel(const __grid_constant__ CUtensorMap tmP, const __grid_constant__ CUtensorMap tmX,
                  const W4Params p) {
    using Cfg = W4Cfg<TT, BK>;
    constexpr int STAGES = Cfg::STAGES, NA = Cfg::NA;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    uint8_t* gbase = smem_raw + (base - raw);
    const uint32_t sStage = base;                                   // [STAGES][X | P]
    const uint32_t sA = base + STAGES * Cfg::STAGE_BYTES;           // [NA][A]
    const uint32_t bars = sA + NA * Cfg::A_BYTES;
    const uint32_t full0 = bars, empty0 = full0 + 8 * STAGES;
    const uint32_t afull0 = empty0 + 8 * STAGES, aempty0 = afull0 + 8 * NA;
    const uint32_t tfull0 = aempty0 + 8 * NA, tempty0 = tfull0 + 16;
    const uint32_t tmem_slot = tempty0 + 16;
    volatile uint32_t* tmem_slot_g = reinterpret_cast<volatile uint32_t*>(
        gbase + STAGES * Cfg::STAGE_BYTES + NA * Cfg::A_BYTES + (2 * STAGES + 2 * NA + 4) * 8);

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int num_n = (p.N + W4_BN - 1) / W4_BN;
    const int num_t = (p.M + TT - 1) / TT;
    const int num_kb = (p.K + BK - 1) / BK;
    const int S = p.splits;
    const int num_units = num_n * num_t * S;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmP);
        tma_prefetch_desc(&tmX);
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, W4_DEQ_WARPS + 1);  // dequantiser warps (packed) + MMA commit (X)
        }
        for (int a = 0; a < NA; ++a) {
            mbar_init(afull0 + 8 * a, W4_DEQ_WARPS);
            mbar_init(aempty0 + 8 * a, 1);
        }
        for (int a = 0; a < 2; ++a) {
            mbar_init(tfull0 + 8 * a, 1);
            mbar_init(tempty0 + 8 * a, 4);
        }
        fence_mbar_init();
    }
    if (warp == 1) {
        tmem_alloc(tmem_slot, Cfg::TMEM_COLS);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_g;

    pdl_wait_prior_grid();

    if (warp == 0) {
        // ------------------------------------------------------------ TMA producer
        if (lane == 0) {
            const uint64_t pol_w = policy_evict_first();  // weights are streamed once per launch
            int stage = 0;
            uint32_t phase = 0;
            for (int u = blockIdx.x; u < num_units; u += gridDim.x) {
                const int tile = u / S, sp = u % S;
                const int n0 = (tile % num_n) * W4_BN, t0 = (tile / num_n) * TT;
                const int kb0 = (sp * num_kb) / S, kb1 = ((sp + 1) * num_kb) / S;
                for (int kb = kb0; kb < kb1; ++kb) {
                    mbar_wait(empty0 + 8 * stage, phase ^ 1);
                    const uint32_t st = sStage + stage * Cfg::STAGE_BYTES;
                    mbar_arrive_expect_tx(full0 + 8 * stage, Cfg::STAGE_BYTES);
#pragma unroll
                    for (int j = 0; j < BK / 64; ++j)
                        tma_load_2d(st + j * Cfg::X_SUB, &tmX, kb * BK + j * 64, t0, full0 + 8 * stage);
                    tma_load_2d_hint(st + Cfg::X_BYTES, &tmP, kb * (BK / 2), n0, full0 + 8 * stage, pol_w);
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------ MMA issuer
        if (lane == 0) {
            constexpr uint32_t idesc = idesc_bf16(W4_BN, TT);
            int stage = 0, ab = 0, acc = 0;
            uint32_t phase = 0, aphase = 0, acc_phase = 0;
            for (int u = blockIdx.x; u < num_units; u += gridDim.x) {
                const int sp = u % S;
                const int kb0 = (sp * num_kb) / S, kb1 = ((sp + 1) * num_kb) / S;
                mbar_wait(tempty0 + 8 * acc, acc_phase ^ 1);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + acc * Cfg::ACC_STRIDE;
                for (int kb = kb0; kb < kb1; ++kb) {
                    mbar_wait(full0 + 8 * stage, phase);    // X landed
                    mbar_wait(afull0 + 8 * ab, aphase);     // weights dequantised
                    tc_fence_after();
                    const uint32_t xs = sStage + stage * Cfg::STAGE_BYTES;
                    const uint32_t as = sA + ab * Cfg::A_BYTES;
#pragma unroll
                    for (int j = 0; j < BK / 64; ++j) {
                        const uint64_t a_desc = make_smem_desc_sw128(as + j * Cfg::A_SUB);
                        const uint64_t b_desc = make_smem_desc_sw128(xs + j * Cfg::X_SUB);
#pragma unroll
                        for (int k = 0; k < 4; ++k)  // 4 x (K = 16 bf16 = 32 bytes) per 64-column sub-tile
                            mma_f16_ss(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc,
                                       (kb != kb0 || j != 0 || k != 0) ? 1u : 0u);
                    }
                    tc_commit(empty0 + 8 * stage);
                    tc_commit(aempty0 + 8 * ab);
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                    if (++ab == NA) { ab = 0; aphase ^= 1; }
                }
                tc_commit(tfull0 + 8 * acc);
                if (++acc == 2) { acc = 0; acc_phase ^= 1; }
            }
        }
    } else if (warp >= W4_DEQ_WARP0) {
        // ------------------------------------------------------------ dequantisers
        const int dt = threadIdx.x - W4_DEQ_WARP0 * 32;
        const int r = dt & 127;        // weight row inside the tile
        const int par = dt >> 7;       // chunk parity handled by this thread
        constexpr int NCH = BK / 32;   // 16-byte chunks (= groups) per row per k-block
        constexpr uint32_t SWM = Cfg::P_ROW / 16 - 1;
        const int gpr = p.K >> 5;      // groups per weight row
        int stage = 0, ab = 0;
        uint32_t phase = 0, aphase = 0;
        for (int u = blockIdx.x; u < num_units; u += gridDim.x) {
            const int tile = u / S, sp = u % S;
            const int n0 = (tile % num_n) * W4_BN;
            const int kb0 = (sp * num_kb) / S, kb1 = ((sp + 1) * num_kb) / S;
            const bool row_ok = n0 + r < p.N;
            const uint16_t* srow = p.g_scale + static_cast<int64_t>(row_ok ? n0 + r : 0) * gpr;
            for (int kb = kb0; kb < kb1; ++kb) {
                uint16_t sbits[NCH / 2];
#pragma unroll
                for (int i = 0; i < NCH / 2; ++i) {
                    const int g = kb * NCH + par + 2 * i;
                    sbits[i] = (row_ok && g < gpr) ? __ldg(srow + g) : static_cast<uint16_t>(0);
                }
                mbar_wait(full0 + 8 * stage, phase);
                const uint32_t ps = sStage + stage * Cfg::STAGE_BYTES + Cfg::X_BYTES;
                uint4 pk[NCH / 2];
#pragma unroll
                for (int i = 0; i < NCH / 2; ++i) {
                    const uint32_t off = r * Cfg::P_ROW + (par + 2 * i) * 16;
                    pk[i] = lds128(ps + (off ^ (((off >> 7) & SWM) << 4)));
                }
                mbar_wait(aempty0 + 8 * ab, aphase ^ 1);   // MMAs that read this A buffer retired
                const uint32_t as = sA + ab * Cfg::A_BYTES;
#pragma unroll
                for (int i = 0; i < NCH / 2; ++i) {
                    const int c = par + 2 * i;
                    const GroupConst gc = group_const(__half2float(__ushort_as_half(sbits[i])));
                    const uint32_t rowb = as + (c >> 1) * Cfg::A_SUB + (r >> 3) * 1024 + (r & 7) * 128;
                    const uint32_t words[4] = {pk[i].x, pk[i].y, pk[i].z, pk[i].w};
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const uint32_t chunk = static_cast<uint32_t>((c & 1) * 4 + j) ^ (r & 7);
                        sts128(rowb + chunk * 16, dequant_word(words[j], gc));
                    }
                }
                fence_proxy_async_smem();                  // generic-proxy writes -> async proxy (MMA)
                __syncwarp();
                if (lane == 0) {                           // one arrival per warp, not per thread
                    mbar_arrive(afull0 + 8 * ab);
                    mbar_arrive(empty0 + 8 * stage);       // packed bytes consumed
                }
                if (++stage == STAGES) { stage = 0; phase ^= 1; }
                if (++ab == NA) { ab = 0; aphase ^= 1; }
            }
        }
    } else {
        // ------------------------------------------------------------ epilogue (warps 2..5)
        const int q = warp & 3;
        int acc = 0;
        uint32_t acc_phase = 0;
        for (int u = blockIdx.x; u < num_units; u += gridDim.x) {
            const int tile = u / S, sp = u % S;
            const int n0 = (tile % num_n) * W4_BN, t0 = (tile / num_n) * TT;
            const int n = n0 + q * 32 + lane;
            const bool n_ok = n < p.N;
            float bv = 0.0f;
            if (p.bias && n_ok) bv = __bfloat162float(static_cast<const __nv_bfloat16*>(p.bias)[n]);
            mbar_wait(tfull0 + 8 * acc, acc_phase);
            tc_fence_after();
            const uint32_t t_addr = tmem_base + acc * Cfg::ACC_STRIDE + (static_cast<uint32_t>(q * 32) << 16);
            if (S == 1) {
#pragma unroll 1
                for (int c = 0; c < TT / 32; ++c) {
                    uint32_t v[32];
                    tmem_ld_32x32b_x32(t_addr + c * 32, v);
                    tmem_wait_ld();
#pragma unroll
                    for (int j = 0; j < 32; ++j) {
                        const int tok = t0 + c * 32 + j;
                        if (n_ok && tok < p.M)
                            w4_store(p.Y, p.out_t, static_cast<int64_t>(tok) * p.N + n,
                                     w4_finish(__uint_as_float(v[j]) + bv, p.act));
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tempty0 + 8 * acc);
            } else {
                float* part = p.partials + static_cast<int64_t>(sp) * p.M * p.N;
#pragma unroll 1
                for (int c = 0; c < TT / 32; ++c) {
                    uint32_t v[32];
                    tmem_ld_32x32b_x32(t_addr + c * 32, v);
                    tmem_wait_ld();
#pragma unroll
                    for (int j = 0; j < 32; ++j) {
                        const int tok = t0 + c * 32 + j;
                        if (n_ok && tok < p.M)
                            __stcg(part + static_cast<int64_t>(tok) * p.N + n, __uint_as_float(v[j]));
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tempty0 + 8 * acc);
                // last arriver of this (tile, quarter) reduces in split order
                __threadfence();
                __syncwarp();
                unsigned old = 0;
                if (lane == 0) old = atomicAdd(p.counters + tile * 4 + q, 1u);
                old = __shfl_sync(0xffffffffu, old, 0);
                if (old == static_cast<unsigned>(S - 1)) {
                    __threadfence();
                    const int tmax = min(TT, p.M - t0);
                    const int64_t sstride = static_cast<int64_t>(p.M) * p.N;
                    for (int j0 = 0; j0 < tmax; j0 += 8) {   // 8 tokens x S loads in flight
                        float y[8];
#pragma unroll
                        for (int j = 0; j < 8; ++j) y[j] = 0.0f;
                        for (int s = 0; s < S; ++s) {        // fixed split order: deterministic sum
#pragma unroll
                            for (int j = 0; j < 8; ++j) {
                                const int64_t idx = static_cast<int64_t>(t0 + j0 + j) * p.N + n;
                                if (n_ok && j0 + j < tmax) y[j] += __ldcg(p.partials + s * sstride + idx);
                            }
                        }
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const int64_t idx = static_cast<int64_t>(t0 + j0 + j) * p.N + n;
                            if (n_ok && j0 + j < tmax) w4_store(p.Y, p.out_t, idx, w4_finish(y[j] + bv, p.act));
                        }
                    }
                    if (lane == 0) p.counters[tile * 4 + q] = 0;  // ready for the next launch
                }
            }
            if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        }
    }

    pdl_launch_dependents();
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
    }
}

template <int TT, int BK>
static int launch_w4(const void* X, int M, int K, const uint8_t* Wq4, int N, const W4Params& p,
                     int grid, cudaStream_t st, bool pdl) {
    using Cfg = W4Cfg<TT, BK>;
    static bool attr_set = false;
    auto kern = w4a16_gemm_kernel<TT, BK>;
    if (!attr_set) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES) !=
            cudaSuccess)
            return ARIA_ERR_CUDA;
        attr_set = true;
    }
    CUtensorMap tmP, tmX;
    int rc = make_tmap_2d(&tmP, Wq4, 1, N, K / 2, W4_BN, Cfg::P_ROW, Cfg::P_ROW);
    if (rc != ARIA_OK) return rc;
    rc = make_tmap_2d(&tmX, X, 2, M, K, TT, 64, 128);
    if (rc != ARIA_OK) return rc;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(W4_THREADS);
    cfg.dynamicSmemBytes = Cfg::SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, tmP, tmX, p) == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
}

// Split-K plan shared by the launcher and aria_workspace_bytes.
void w4_plan(int M, int N, int K, int sms, int* tt_out, int* bk_out, int* splits_out) {
    const int tt = M <= 32 ? 32 : M <= 64 ? 64 : M <= 128 ? 128 : 256;
    const int bk = tt <= 64 ? 128 : 64;
    const int tiles = ((N + W4_BN - 1) / W4_BN) * ((M + tt - 1) / tt);
    const int num_kb = (K + bk - 1) / bk;
    int s = 1;
    if (tiles * 2 <= sms) {  // less than half the machine busy: split K
        s = sms / tiles;
        if (s > num_kb) s = num_kb;
        if (s > 16) s = 16;
        if (s < 1) s = 1;
    }
    *tt_out = tt; *bk_out = bk; *splits_out = s;
}

size_t w4_workspace_bytes(int M, int N, int K, int sms) {
    int tt, bk, s;
    w4_plan(M, N, K, sms, &tt, &bk, &s);
    const size_t tiles = static_cast<size_t>((N + W4_BN - 1) / W4_BN) * ((M + tt - 1) / tt);
    size_t counters = (tiles * 4 * sizeof(unsigned) + 255) / 256 * 256;
    size_t partials = s > 1 ? static_cast<size_t>(s) * M * N * sizeof(float) : 0;
    return counters + (partials + 255) / 256 * 256;
}

int launch_gemm_w4a16(const void* X, int M, int K, const uint8_t* Wq4, const uint16_t* g_scale,
                      int N, const void* bias, int act, void* Y, int yt, void* ws, size_t ws_bytes,
                      cudaStream_t st, bool pdl) {
    const int sms = num_sms();
    if (sms <= 0) return ARIA_ERR_CUDA;
    int tt, bk, s;
    w4_plan(M, N, K, sms, &tt, &bk, &s);
    if (s > 1 && (ws == nullptr || ws_bytes < w4_workspace_bytes(M, N, K, sms))) s = 1;
    W4Params p;
    p.g_scale = g_scale; p.bias = bias; p.Y = Y;
    p.act = act; p.out_t = yt; p.M = M; p.N = N; p.K = K; p.splits = s;
    const size_t tiles = static_cast<size_t>((N + W4_BN - 1) / W4_BN) * ((M + tt - 1) / tt);
    p.counters = static_cast<unsigned*>(ws);
    p.partials = s > 1 ? reinterpret_cast<float*>(static_cast<uint8_t*>(ws) +
                                                  (tiles * 4 * sizeof(unsigned) + 255) / 256 * 256)
                       : nullptr;
    const int units = static_cast<int>(tiles) * s;
    const int grid = units < sms ? units : sms;
    if (s > 1 && cudaMemsetAsync(p.counters, 0, tiles * 4 * sizeof(unsigned), st) != cudaSuccess)
        return ARIA_ERR_CUDA;
    if (tt == 32) return launch_w4<32, 128>(X, M, K, Wq4, N, p, grid, st, pdl);
    if (tt == 64) return launch_w4<64, 128>(X, M, K, Wq4, N, p, grid, st, pdl);
    if (tt == 128) return launch_w4<128, 64>(X, M, K, Wq4, N, p, grid, st, pdl);
    return launch_w4<256, 64>(X, M, K, Wq4, N, p, grid, st, pdl);
}

}  // namespace aria
