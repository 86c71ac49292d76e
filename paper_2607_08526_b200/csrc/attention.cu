// attention.cu -- NEXT-2: fused full self-attention between the QKV projection and the
// out-projection ("the transformer's full self-attention ... a fused attention kernel
// (FlashAttention-class) behind a build flag is the open lever"; L224).  include/aria.h: aria_attention.
//
//   per (sequence b, head h, query i):  s_j = scale q_i . k_j;  p = softmax_j(s);  o_i = sum_j p_j v_j
//
// One CTA = one tile of 128 queries of one (b, h); two CTAs are resident per SM (80 KB of shared memory,
// 256 tensor-memory columns each), so one CTA's exponentials overlap the other's MMAs.  192 threads:
//   warp 0      TMA producer: the Q tile once, then K and V tiles of 128 keys ([128 x 64] bf16, 128-byte
//               swizzle) straight out of the [B*S, 3*H*64] QKV tensor through ONE 3-D tensor map
//               (columns, token, sequence: rows past the end of a sequence are zero-filled, never the next
//               sequence's) into two 2-stage rings.
//   warp 1      MMA issuer (one thread).  S = Q K^T: 4 x tcgen05.mma 128x128x16, both operands K-major in
//               shared memory, fp32 scores in tensor memory.  O += P V: 8 x tcgen05.mma 128x64x16 with
//               A = P read from TENSOR MEMORY (bf16, written there by the softmax warps -- P never touches
//               shared memory) and B = the V tile as it lies in shared memory, described MN-major (the
//               head dimension is contiguous), so V needs no transposition.  Q K^T of tile j+1 is issued as
//               soon as the softmax warps have pulled S_j into registers, i.e. it runs under exp(S_j).
//   warps 2..5  softmax, thread = query row (= tensor-memory lane): tcgen05.ld of the 128 scores, row
//               maximum, p = exp2(s c - m) with c = scale log2 e, bf16 P back into tensor memory, running
//               sum.  The running maximum is LAZY: m only moves when the tile maximum exceeds it by more
//               than 8 (log2 units), so the O accumulator in tensor memory is rescaled (ld, mul, st) on few
//               tiles; p <= 2^8 meanwhile, harmless in bf16 / fp32, and O / l is unchanged mathematically.
//               Epilogue: O / l -> bf16 -> 128 contiguous bytes per thread to global memory; optionally the
//               per-token max |o| is reduced across heads with atomicMax (first half of a fused S1 for a
//               W8A8 out-projection).
// Roofline: per (query tile, key tile) 640 cycles of tensor work (an N = 64 tcgen05.mma costs 48 cycles, not 32)
// against 1024 cycles of the SM's 16 ex2 lanes -- the exponential unit is the kernel's ceiling.
// Measured (debug-build role timings): 2990 cycles per key tile per CTA, of which ~650 are the
// exponentials and ~560 barrier waits of the softmax warp; without exponentials at all the kernel is only 16 %
// faster, so today it is bound by the per-tile chain of dependent phases, not by that ceiling.
#include "internal.cuh"

namespace aria {

constexpr int AT_BM = 128;                 // queries per CTA
constexpr int AT_BN = 128;                 // keys per tile
constexpr int AT_D = 64;                   // head dimension
constexpr int AT_ST = 2;                   // K / V ring depth
constexpr int AT_TILE = AT_BN * AT_D * 2;  // 16 KB
constexpr int AT_Q_OFF = 0;
constexpr int AT_K_OFF = AT_TILE;
constexpr int AT_V_OFF = AT_K_OFF + AT_ST * AT_TILE;
constexpr int AT_BAR_OFF = AT_V_OFF + AT_ST * AT_TILE;
constexpr int AT_NBAR = 1 + 4 * AT_ST + 4;
constexpr int AT_SMEM = AT_BAR_OFF + AT_NBAR * 8 + 16 + 1024;
constexpr int AT_S_COL = 0, AT_P_COL = 128, AT_O_COL = 192, AT_TMEM_COLS = 256;
constexpr float AT_LAZY = 8.0f;

struct AttParams {
    __nv_bfloat16* O;       // [B*S, H*64]
    float* row_absmax;      // [B*S] or nullptr
    int S, H;
    float c;                // scale * log2(e)
#ifdef ARIA_DEBUG
    long long* prof;        // per-CTA role timings (debug builds), or nullptr
#endif
};

#ifdef ARIA_DEBUG
static long long* g_att_prof = nullptr;
void att_set_profile_buffer(long long* p) { g_att_prof = p; }
#define AT_TIMED(acc, stmt) do { const long long t_ = clock64(); stmt; acc += clock64() - t_; } while (0)
#else
#define AT_TIMED(acc, stmt) do { stmt; } while (0)
#endif

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* m, int c0, int c1, int c2, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes"
        " [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(dst),
        "l"(reinterpret_cast<uint64_t>(m)), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}
__device__ __forceinline__ float ex2(float x) {
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ uint32_t bf16x2(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}

__global__ void __launch_bounds__(192, 2)
attention_kernel(const __grid_constant__ CUtensorMap tmQKV, const AttParams p) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    uint8_t* gbase = smem_raw + (base - raw);
    const uint32_t sQ = base + AT_Q_OFF, sK = base + AT_K_OFF, sV = base + AT_V_OFF;
    const uint32_t bars = base + AT_BAR_OFF;
    const uint32_t qfull = bars, kfull0 = qfull + 8, kempty0 = kfull0 + 8 * AT_ST, vfull0 = kempty0 + 8 * AT_ST,
                   vempty0 = vfull0 + 8 * AT_ST, sfull = vempty0 + 8 * AT_ST, sfree = sfull + 8, pfull = sfree + 8,
                   pvdone = pfull + 8, tmem_slot = pvdone + 8;
    volatile uint32_t* tmem_slot_g = reinterpret_cast<volatile uint32_t*>(gbase + AT_BAR_OFF + AT_NBAR * 8);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int qt = blockIdx.x, h = blockIdx.y, b = blockIdx.z;
    const int nkv = (p.S + AT_BN - 1) / AT_BN;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmQKV);
        mbar_init(qfull, 1);
        for (int s = 0; s < AT_ST; ++s) {
            mbar_init(kfull0 + 8 * s, 1);
            mbar_init(kempty0 + 8 * s, 1);
            mbar_init(vfull0 + 8 * s, 1);
            mbar_init(vempty0 + 8 * s, 1);
        }
        mbar_init(sfull, 1);
        mbar_init(sfree, 4);
        mbar_init(pfull, 4);
        mbar_init(pvdone, 1);
        fence_mbar_init();
    }
    if (warp == 1) {
        tmem_alloc(tmem_slot, AT_TMEM_COLS);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_g;
    pdl_launch_dependents();

    if (warp == 0) {
        // ------------------------------------------------------------ TMA producer
        pdl_wait_prior_grid();
        if (elect_one()) {
            mbar_arrive_expect_tx(qfull, AT_TILE);
            tma_load_3d(sQ, &tmQKV, h * AT_D, qt * AT_BM, b, qfull);
        }
        __syncwarp();
        for (int j = 0; j < nkv; ++j) {
            const int st = j % AT_ST;
            const uint32_t ph = (j / AT_ST) & 1;
            mbar_wait(kempty0 + 8 * st, ph ^ 1);
            if (elect_one()) {
                mbar_arrive_expect_tx(kfull0 + 8 * st, AT_TILE);
                tma_load_3d(sK + st * AT_TILE, &tmQKV, (p.H + h) * AT_D, j * AT_BN, b, kfull0 + 8 * st);
            }
            __syncwarp();
            mbar_wait(vempty0 + 8 * st, ph ^ 1);
            if (elect_one()) {
                mbar_arrive_expect_tx(vfull0 + 8 * st, AT_TILE);
                tma_load_3d(sV + st * AT_TILE, &tmQKV, (2 * p.H + h) * AT_D, j * AT_BN, b, vfull0 + 8 * st);
            }
            __syncwarp();
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------ MMA issuer
        constexpr uint32_t idesc_qk = idesc_bf16(AT_BM, AT_BN);
        constexpr uint32_t idesc_pv = idesc_bf16(AT_BM, AT_D) | (1u << 16);   // B (= V) is MN-major
        const uint64_t desc_hi = make_smem_desc_sw128(0);
        const uint64_t q_desc = desc_hi | ((sQ & 0x3FFFF) >> 4);
        const uint32_t s_tmem = tmem_base + AT_S_COL, p_tmem = tmem_base + AT_P_COL, o_tmem = tmem_base + AT_O_COL;
        long long m_p = 0, m_v = 0, m_k = 0, m_s = 0;
        const long long m_t0 = clock64();
        auto issue_pv = [&](int j) {
            const int st = j % AT_ST;
            AT_TIMED(m_p, mbar_wait(pfull, j & 1));              // P_j in tensor memory, O rescaled
            AT_TIMED(m_v, mbar_wait(vfull0 + 8 * st, (j / AT_ST) & 1));
            tc_fence_after();
            if (elect_one()) {
                // V tile: 128 keys x 128 bytes; 8 keys = one 1024-byte swizzle atom, K = 16 keys = 2 atoms
                const uint64_t v_desc = desc_hi | (((sV + st * AT_TILE) & 0x3FFFF) >> 4);
#pragma unroll
                for (int k = 0; k < AT_BN / 16; ++k)
                    mma_f16_ts(o_tmem, p_tmem + 8 * k, v_desc + static_cast<uint64_t>(k) * (2048 >> 4), idesc_pv,
                               (j > 0 || k > 0) ? 1u : 0u);
                tc_commit(pvdone);
                tc_commit(vempty0 + 8 * st);
            }
            __syncwarp();
        };
        mbar_wait(qfull, 0);
        for (int j = 0; j < nkv; ++j) {
            const int st = j % AT_ST;
            AT_TIMED(m_k, mbar_wait(kfull0 + 8 * st, (j / AT_ST) & 1));
            if (j > 0) AT_TIMED(m_s, mbar_wait(sfree, (j - 1) & 1));   // S_{j-1} is in the softmax warps' registers
            tc_fence_after();
            if (elect_one()) {
                const uint64_t k_desc = desc_hi | (((sK + st * AT_TILE) & 0x3FFFF) >> 4);
#pragma unroll
                for (int k = 0; k < AT_D / 16; ++k)
                    mma_f16_ss(s_tmem, q_desc + 2 * k, k_desc + 2 * k, idesc_qk, k > 0 ? 1u : 0u);
                tc_commit(sfull);
                tc_commit(kempty0 + 8 * st);
            }
            __syncwarp();
            if (j > 0) issue_pv(j - 1);
        }
        issue_pv(nkv - 1);
#ifdef ARIA_DEBUG
        if (p.prof && lane == 0) {
            long long* q = p.prof + (static_cast<size_t>(blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x) * 16;
            q[0] = m_k; q[1] = m_s; q[2] = m_p; q[3] = m_v; q[4] = clock64() - m_t0;
        }
#else
        (void)m_p; (void)m_v; (void)m_k; (void)m_s; (void)m_t0;
#endif
    } else {
        // ------------------------------------------------------------ softmax + epilogue (warps 2..5)
        const int quarter = warp & 3;                            // tensor-memory lane quarter of this warp
        const int row = quarter * 32 + lane;
        const uint32_t lane_off = static_cast<uint32_t>(quarter * 32) << 16;
        const uint32_t s_addr = tmem_base + AT_S_COL + lane_off, p_addr = tmem_base + AT_P_COL + lane_off,
                       o_addr = tmem_base + AT_O_COL + lane_off;
        const float c = p.c;
        float m = 0.0f, l = 0.0f;
        long long s_w = 0, s_ld = 0, s_pv = 0, s_st = 0;
        const long long s_t0 = clock64();
        for (int j = 0; j < nkv; ++j) {
            AT_TIMED(s_w, mbar_wait(sfull, j & 1));
            const long long t_ld_ = clock64();
            tc_fence_after();
            uint32_t v[4][32];
#pragma unroll
            for (int i = 0; i < 4; ++i) tmem_ld_32x32b_x32(s_addr + 32 * i, v[i]);
            tmem_wait_ld();
            s_ld += clock64() - t_ld_;
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(sfree);
            if (j == nkv - 1 && (p.S % AT_BN) != 0) {             // keys past the end of the sequence
                const int valid = p.S - j * AT_BN;
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int k = 0; k < 32; ++k)
                        if (32 * i + k >= valid) v[i][k] = 0xFF800000u;   // -inf
            }
            float mx4[4];                                        // four independent chains (latency, not count)
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                mx4[i] = __uint_as_float(v[i][0]);
#pragma unroll
                for (int k = 1; k < 32; ++k) mx4[i] = fmaxf(mx4[i], __uint_as_float(v[i][k]));
            }
            const float mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3]));
            const float ms = mx * c;
            const bool move = (j == 0) || (ms > m + AT_LAZY);
            const float m_new = move ? ms : m;
            const float alpha = ex2(m - m_new);                  // 1 when the maximum stays
            float sum4[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int k = 0; k < 32; k += 2) {
                    const float p0 = ex2(fmaf(__uint_as_float(v[i][k]), c, -m_new));
                    const float p1 = ex2(fmaf(__uint_as_float(v[i][k + 1]), c, -m_new));
                    sum4[(k >> 1) & 3] += p0 + p1;
                    v[i >> 1][(i & 1) * 16 + (k >> 1)] = bf16x2(p0, p1);   // in place: slot index <= source index
                }
            const float sum = (sum4[0] + sum4[1]) + (sum4[2] + sum4[3]);
            if (j > 0) {
                AT_TIMED(s_pv, mbar_wait(pvdone, (j - 1) & 1));  // P_{j-1} consumed, O up to date
                tc_fence_after();
                if (__any_sync(0xffffffffu, move)) {             // rare after the first tiles
                    uint32_t o[2][32];
                    tmem_ld_32x32b_x32(o_addr, o[0]);
                    tmem_ld_32x32b_x32(o_addr + 32, o[1]);
                    tmem_wait_ld();
#pragma unroll
                    for (int i = 0; i < 2; ++i)
#pragma unroll
                        for (int k = 0; k < 32; ++k) o[i][k] = __float_as_uint(__uint_as_float(o[i][k]) * alpha);
                    tmem_st_32x32b_x32(o_addr, o[0]);
                    tmem_st_32x32b_x32(o_addr + 32, o[1]);
                }
                l *= alpha;
            }
            l += sum;
            m = m_new;
            const long long t_st_ = clock64();
            tmem_st_32x32b_x32(p_addr, v[0]);
            tmem_st_32x32b_x32(p_addr + 32, v[1]);
            tmem_wait_st();
            s_st += clock64() - t_st_;
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(pfull);
        }
        AT_TIMED(s_pv, mbar_wait(pvdone, (nkv - 1) & 1));
#ifdef ARIA_DEBUG
        if (p.prof && warp == 2 && lane == 0) {
            long long* q = p.prof + (static_cast<size_t>(blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x) * 16;
            q[8] = s_w; q[9] = s_ld; q[10] = s_pv; q[11] = s_st; q[12] = clock64() - s_t0;
        }
#else
        (void)s_w; (void)s_ld; (void)s_pv; (void)s_st; (void)s_t0;
#endif
        tc_fence_after();
        uint32_t o[2][32];
        tmem_ld_32x32b_x32(o_addr, o[0]);
        tmem_ld_32x32b_x32(o_addr + 32, o[1]);
        tmem_wait_ld();
        const float inv = 1.0f / l;
        const int tok = qt * AT_BM + row;
        if (tok < p.S) {
            const int64_t grow = static_cast<int64_t>(b) * p.S + tok;
            uint4* dst = reinterpret_cast<uint4*>(p.O + grow * (static_cast<int64_t>(p.H) * AT_D) + h * AT_D);
            float amax = 0.0f;
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int k = 0; k < 32; k += 8) {
                    uint32_t w[4];
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        w[e] = bf16x2(__uint_as_float(o[i][k + 2 * e]) * inv, __uint_as_float(o[i][k + 2 * e + 1]) * inv);
                        amax = fmaxf(amax, fmaxf(fabsf(__uint_as_float(w[e] << 16)), fabsf(__uint_as_float(w[e] & 0xFFFF0000u))));
                    }
                    dst[i * 4 + (k >> 3)] = make_uint4(w[0], w[1], w[2], w[3]);
                }
            if (p.row_absmax) atomicMax(reinterpret_cast<unsigned*>(p.row_absmax) + grow, __float_as_uint(amax));
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, AT_TMEM_COLS);
    }
}

int launch_attention(const void* QKV, int B, int S, int H, float scale, void* O, float* row_absmax, cudaStream_t st,
                     bool pdl) {
    static std::atomic<uint64_t> attr_mask{0};
    if (!ensure_dyn_smem(attention_kernel, AT_SMEM, attr_mask)) return ARIA_ERR_CUDA;
    CUtensorMap tm;
    const uint64_t ld = 3ull * H * AT_D;
    int rc = make_tmap_3d(&tm, QKV, 2, ld, static_cast<uint64_t>(S), static_cast<uint64_t>(B), ld * 2, ld * 2 * S, AT_D,
                          AT_BN, 1, 128);
    if (rc != ARIA_OK) return rc;
    AttParams p;
    p.O = static_cast<__nv_bfloat16*>(O);
    p.row_absmax = row_absmax;
    p.S = S; p.H = H;
    p.c = scale * 1.4426950408889634f;
#ifdef ARIA_DEBUG
    p.prof = g_att_prof;
#endif
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((S + AT_BM - 1) / AT_BM, H, B);
    cfg.blockDim = dim3(192);
    cfg.dynamicSmemBytes = AT_SMEM;
    if (const char* e = dbg_env("ARIA_ATT_ONE_CTA")) {          // debug builds only: one CTA per SM (timing experiment)
        (void)e;
        cfg.dynamicSmemBytes = 120 * 1024;
        cudaFuncSetAttribute(attention_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 120 * 1024);
    }
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, attention_kernel, tm, p) == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
}

}  // namespace aria
