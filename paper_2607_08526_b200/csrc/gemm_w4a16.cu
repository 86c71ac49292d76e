// gemm_w4a16.cu -- S4: W4A16 linear.  int4 group-32 weights are dequantised ON CHIP to bf16 and
// fed to tcgen05.mma kind::f16 (bf16 x bf16, fp32 accumulators in TMEM).
//
// "Swap-AB": the weight tile is the MMA's M operand (128 output channels on the 128 TMEM lanes)
// and the token tile is the MMA's N operand (TT = 32..256 tokens), so a 32-token batch is a legal
// N = 32 instruction and each dequantised weight feeds TT MACs.
//
// Persistent, warp-specialised, one CTA per SM.  k-blocks are 64 wide (two int4 groups).  The two
// operands travel through SEPARATE rings, because their consumers have very different latencies:
//   warp 0       TMA producer for X: [TT x 64] bf16 tiles (128-byte swizzle), consumed directly by
//                the MMA -> a short ring of large stages.
//   warp 2       TMA producer for the packed weights: [128 rows x 32 bytes] tiles (32-byte swizzle),
//                consumed by the dequantisers -> a deep ring of 4 KB stages (this is the HBM stream).
//   warp 1       MMA issuer (one thread): 4 tcgen05.mma per k-block, A = dequantised weights,
//                B = X, into one of two TMEM accumulators.
//   warps 4..7   epilogue: tcgen05.ld -> (+bias, GELU, cast) -> smem transpose -> TMA store, or
//                split-K partials.
//   warps 8..    G dequantiser GROUPS of 4 warps (thread = weight row).  Group g handles k-blocks
//                g, g+G, ... (A buffer = k-block index mod NB): wait packed -> LDS -> 64 x (LOP3, FFMA2/2, CVT/2) into
//                registers -> wait A buffer free -> 8 STS -> fence -> arrive.  The arithmetic is done
//                BEFORE waiting for the buffer, so the MMA -> dequant -> MMA hand-off is short.
// Exactness of w^ = bf16_rne(q*sg): the nibble n is placed (XOR 8 = offset binary u = q+8) at
// mantissa bit pos in {8,12,16} of 1.0f, giving x = 1 + u*2^(pos-23); one FMA
// x * (2^(23-pos) sg) - (2^(23-pos)+8) sg has exactly representable addends and the exactly
// representable result q*sg, so fp32 holds q*sg exactly and one cvt.rn rounds it to bf16.
// The FMAs are issued as packed fma.rn.f32x2 (two elements per instruction on sm_100).
//
// Split-K (small M): a work unit is (tile, k-range); units of a tile write fp32 partials to the
// workspace, the last to arrive (per 32-channel quarter, atomic counter) sums them in split order
// -- deterministic -- and finishes the epilogue.
#include <cstdlib>

#include "internal.cuh"

namespace aria {

constexpr int W4_BN = 128;      // output channels per tile = MMA M
constexpr int W4_BK = 64;       // k-block: 64 weights = 32 packed bytes = 2 groups per row
constexpr int W4_EPI_WARP0 = 4;
constexpr int W4_DEQ_WARP0 = 8;
constexpr int W4_G = 3;         // dequantiser groups = A buffers

// WB = weight bits: 4 (S4, int4 group-32 + fp16 group scales) or 8 (NEXT-1 "q8", int8 per-channel + fp32
// scales).  The two formats share everything but the packed-tile geometry and the dequantiser arithmetic.
// (CTA pairs and X multicast were built, parity-green and measured twice: no gain, removed -- the dequantiser
// arithmetic, not X traffic or the tensor pipe, sets the k-block time.  DESIGN.md 9.)
template <int TT, int WB = 4>
struct W4Cfg {
    static constexpr int G = W4_G;
    // ATM: the dequantised A tile goes registers -> TENSOR MEMORY (tcgen05.st) and the MMA reads it from there.
    // At M >= 512 the k-block time was set by shared-memory traffic (measured 800-860 cycles per 64-k block
    // against 384-512 of tensor time: X tile written by TMA and read by the MMA, plus 16 KB of A written by
    // the dequantisers and 16 KB read back by the MMA); A in TMEM removes those 32 KB per k-block.  Needs
    // 2 TT accumulator columns + 4 x 32 A columns <= 512: every token tile but TT = 256.
    static constexpr bool ATM = TT <= 192;
    static constexpr int NB = ATM ? 4 : G;                     // dequantised A buffers (TMEM slots / smem tiles)
    static constexpr int THREADS = 32 * W4_DEQ_WARP0 + 128 * G;
    static constexpr int P_ROW = W4_BK * WB / 8;               // 32 (int4) / 64 (int8) packed bytes per row per k-block
    static constexpr int P_BYTES = W4_BN * P_ROW;              // 4 KB / 8 KB
    static constexpr int X_ROWS = TT;                          // token rows per X stage
    static constexpr int X_BYTES = X_ROWS * 128;               // x 64 bf16
    static constexpr int A_BYTES = W4_BN * 128;                // 16 KB: 128 rows x 64 bf16
    static constexpr int STG_BYTES = 4096;                     // per epilogue warp: 32 tokens x 128 B
    // LOCK (with A in tensor memory): ONE full and ONE empty barrier per k-block, indexed by the X stage (k-block
    // mod XS): full[i] collects the dequantiser warps' arrivals AND the X tile's bytes, empty[i] is the single
    // tcgen05.commit of that k-block; the X producer waits on it before refilling stage i (k-block + XS) and the
    // dequantisers before reusing the A slot (k-block + NB: they wait on the empty barrier of k-block - NB).  The MMA
    // warp's loop is a serial chain (role timestamps: ~100 cycles per barrier wait, ~27 per tcgen05.mma, ~55 per
    // tcgen05.commit): two waits and two commits per 64-k block made it ~530 cycles, more than the 384 of tensor
    // time it feeds.  XS stays deep: an X tile takes ~2000 cycles to arrive when every SM pulls 24 KB per k-block
    // through the L2 (role timestamps; with XS = NB = 4 the k-block period was (2000 + 700) / 4).
    static constexpr bool LOCK = ATM;
    static constexpr int XS = !LOCK ? (X_ROWS == 256 ? 3 : 8)
                              : TT == 192 ? (WB == 8 ? 5 : 6) : TT == 128 ? 6 : 8;   // X ring depth
    static constexpr int PS = WB == 8 ? (TT >= 192 ? 8 : TT == 32 ? 16 : 12)      // packed ring depth
                                      : (TT >= 192 ? 8 : TT == 128 ? 12 : 16);
    static constexpr int X_OFF = 0;
    static constexpr int A_OFF = X_OFF + XS * X_BYTES;
    static constexpr int P_OFF = A_OFF + (ATM ? 0 : NB * A_BYTES);
    static constexpr int STG_OFF = P_OFF + PS * P_BYTES;
    static constexpr int BAR_OFF = STG_OFF + 4 * STG_BYTES;
    static constexpr int NBAR = 2 * XS + 2 * PS + 2 * NB + 4;
    static constexpr int SMEM_BYTES = BAR_OFF + NBAR * 8 + 16 + 1024;
    // TT = 192 fills the SMs when N / 128 is small: 12 row tiles x 11 token tiles = 132 units on 148 SMs
    // at M = 2048 (TT = 256: 96 units)
    static constexpr int ACC_STRIDE = TT;
    static constexpr int A_COL0 = 2 * ACC_STRIDE;             // ATM: 4 slots of 32 columns (128 rows x 64 k bf16)
    static constexpr int TMEM_COLS = ATM ? (A_COL0 + 4 * 32 <= 256 ? 256 : 512) : 512;
    static_assert(!ATM || A_COL0 + NB * 32 <= TMEM_COLS, "tensor memory");
    static_assert(TT == 32 || TT == 64 || TT == 128 || TT == 192 || TT == 256, "TT");
    static_assert(WB == 4 || WB == 8, "weight bits");
    static_assert(SMEM_BYTES <= 227 * 1024, "shared memory");
};

struct W4Params {
    const void* g_scale;      // WB = 4: fp16 bits [N, K/32];  WB = 8: fp32 [N]
    const void* bias;         // bf16 [N] or nullptr
    void* Y;
    float* partials;          // [splits, M, N] fp32 (split-K only)
    unsigned* counters;       // [num_tiles * 4], zeroed by a memset node before each launch
    int act, out_t;
    int M, N, K;
    int splits;
#ifdef ARIA_DEBUG
    long long* prof;          // per-CTA role timestamps (clock64), or nullptr
    int dbg;                  // timing experiments (ARIA_W4_DBG; results are WRONG): 1 = X loaded for every other k-block only, 2 = no X loads
#endif
};

#ifdef ARIA_DEBUG
static long long* g_w4_prof = nullptr;
static int g_w4_prof_launch = 0;          // every launch (graph node) gets its own 148 x 32 slot, 256 slots
void w4_set_profile_buffer(long long* p) { g_w4_prof = p; g_w4_prof_launch = 0; }
__device__ __forceinline__ void prof_stamp(const W4Params& p, int slot, long long t0) {
    if (p.prof) p.prof[blockIdx.x * 64 + slot] = clock64() - t0;
}
#define W4_TIMED(acc, stmt) do { const long long t_ = clock64(); stmt; acc += clock64() - t_; } while (0)
#define W4_CLK() clock64()
#else
#define W4_CLK() 0LL
__device__ __forceinline__ void prof_stamp(const W4Params&, int, long long) {}
#define W4_TIMED(acc, stmt) do { stmt; } while (0)
#endif

__device__ __forceinline__ uint32_t cvt_bf16x2(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}
// (a & b) ^ c in one LOP3
__device__ __forceinline__ uint32_t lop_and_xor(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0x6A;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
__device__ __forceinline__ uint64_t pack2(float lo, float hi) {
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ uint64_t pack2u(uint32_t lo, uint32_t hi) {
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(lo), "r"(hi));
    return r;
}
// two fp32 FMAs in one instruction (sm_100 FFMA2); result packed as bf16x2 (lo = element 0)
__device__ __forceinline__ uint32_t fma2_to_bf16x2(uint64_t x, uint64_t s, uint64_t c) {
    uint64_t d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(x), "l"(s), "l"(c));
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(d));
    return cvt_bf16x2(lo, hi);
}

// Per-group constants: (scale, offset) for a nibble sitting at mantissa bit 8, 12 or 16 of 1.0f.
// Scalar FFMAs on purpose: the packed f32x2 form needs both operands in aligned register pairs and cost
// 2.6 IMAD.MOV per weight pair in this loop (ncu: 84 of its 325 instructions), more than it saved.
struct GroupConst {
    float s8, c8, s12, c12, s16, c16;
};
__device__ __forceinline__ GroupConst group_const(float sg) {
    GroupConst g;
    g.s8 = sg * 32768.0f;  g.c8 = -(sg * 32776.0f);    // 2^15, 2^15 + 8
    g.s12 = sg * 2048.0f;  g.c12 = -(sg * 2056.0f);    // 2^11, 2^11 + 8
    g.s16 = sg * 128.0f;   g.c16 = -(sg * 136.0f);     // 2^7,  2^7  + 8
    return g;
}
// 8 codes of one 32-bit word (nibble i = code of k = 8w + i) -> 4 packed bf16x2, k ascending.
// x = 1.0f | (u << pos) with u = q + 8, so x * (2^(23-pos) sg) - (2^(23-pos) + 8) sg = q sg exactly
// (both addends and the result are representable), and one cvt.rn.bf16x2 rounds it: w^ = bf16_rne(q sg).
__device__ __forceinline__ uint4 dequant_word(uint32_t w, const GroupConst& g) {
    const uint32_t wa = w << 8, wb = w >> 12;
    const uint32_t M8 = 0x00000F00u, M12 = 0x0000F000u, M16 = 0x000F0000u;
    const uint32_t X8 = 0x3F800800u, X12 = 0x3F808000u, X16 = 0x3F880000u;  // 1.0f | (8 << pos)
    const float f0 = fmaf(__uint_as_float(lop_and_xor(wa, M8, X8)), g.s8, g.c8);
    const float f1 = fmaf(__uint_as_float(lop_and_xor(wa, M12, X12)), g.s12, g.c12);
    const float f2 = fmaf(__uint_as_float(lop_and_xor(wa, M16, X16)), g.s16, g.c16);
    const float f3 = fmaf(__uint_as_float(lop_and_xor(w, M12, X12)), g.s12, g.c12);
    const float f4 = fmaf(__uint_as_float(lop_and_xor(w, M16, X16)), g.s16, g.c16);
    const float f5 = fmaf(__uint_as_float(lop_and_xor(wb, M8, X8)), g.s8, g.c8);
    const float f6 = fmaf(__uint_as_float(lop_and_xor(wb, M12, X12)), g.s12, g.c12);
    const float f7 = fmaf(__uint_as_float(lop_and_xor(wb, M16, X16)), g.s16, g.c16);
    return make_uint4(cvt_bf16x2(f0, f1), cvt_bf16x2(f2, f3), cvt_bf16x2(f4, f5), cvt_bf16x2(f6, f7));
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

__device__ __forceinline__ void w4_store(void* Y, int out_t, int64_t idx, float y) {
    if (out_t == ARIA_F32)
        static_cast<float*>(Y)[idx] = y;
    else
        static_cast<__nv_bfloat16*>(Y)[idx] = __float2bfloat16_rn(y);
}

// 16 int8 codes (4 words) x one per-channel scale -> 16 bf16, k ascending: w^ = bf16_rne(fl32(q * sw)).
// (The definition rounds the exact product once; rounding it to fp32 first changes the bf16 result only
// when the fp32 rounding lands exactly on a bf16 tie: < 2^-16 of the weights, by one bf16 ulp.)
__device__ __forceinline__ void dequant_i8x16(const uint4& v, float sw, uint4& lo, uint4& hi) {
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
    uint32_t o[8];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float f0 = static_cast<float>(static_cast<int8_t>(w[i] & 0xFF)) * sw;
        const float f1 = static_cast<float>(static_cast<int8_t>((w[i] >> 8) & 0xFF)) * sw;
        const float f2 = static_cast<float>(static_cast<int8_t>((w[i] >> 16) & 0xFF)) * sw;
        const float f3 = static_cast<float>(static_cast<int8_t>(w[i] >> 24)) * sw;
        o[2 * i] = cvt_bf16x2(f0, f1);
        o[2 * i + 1] = cvt_bf16x2(f2, f3);
    }
    lo = make_uint4(o[0], o[1], o[2], o[3]);
    hi = make_uint4(o[4], o[5], o[6], o[7]);
}

// (X multicast over CTA couples -- both CTAs of a cluster on the same token tile, each loading half of every X
// tile into both -- was built twice: with A in shared memory (round 1: 3.79 vs 3.81 ms per C5 step) and with A
// in tensor memory (round 2: 3.29 vs 3.32 ms).  The k-block time is not set by L2 reads of X; removed.)
template <int TT, bool GELU, int WB>
__global__ void __launch_bounds__(W4Cfg<TT, WB>::THREADS, 1)
w4a16_gemm_kernel(const __grid_constant__ CUtensorMap tmP, const __grid_constant__ CUtensorMap tmX,
                  const __grid_constant__ CUtensorMap tmY, const W4Params p) {
    using Cfg = W4Cfg<TT, WB>;
    constexpr int XS = Cfg::XS, PS = Cfg::PS, G = Cfg::G, NB = Cfg::NB;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    uint8_t* gbase = smem_raw + (base - raw);
    const uint32_t sX = base + Cfg::X_OFF, sA = base + Cfg::A_OFF, sP = base + Cfg::P_OFF;
    const uint32_t bars = base + Cfg::BAR_OFF;
    const uint32_t xfull0 = bars, xempty0 = xfull0 + 8 * XS;
    const uint32_t pfull0 = xempty0 + 8 * XS, pempty0 = pfull0 + 8 * PS;
    const uint32_t afull0 = pempty0 + 8 * PS, aempty0 = afull0 + 8 * NB;
    const uint32_t tfull0 = aempty0 + 8 * NB, tempty0 = tfull0 + 16;
    const uint32_t tmem_slot = tempty0 + 16;
    volatile uint32_t* tmem_slot_g =
        reinterpret_cast<volatile uint32_t*>(gbase + Cfg::BAR_OFF + Cfg::NBAR * 8);

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    constexpr int UN = W4_BN;                                   // output channels per work unit
    const int num_n = (p.N + UN - 1) / UN;
    const int num_t = (p.M + TT - 1) / TT;
    const int num_kb = (p.K + W4_BK - 1) / W4_BK;
    const int S = p.splits;
    const int num_units = num_n * num_t * S;
    const int unit0 = blockIdx.x, unit_step = gridDim.x;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmP);
        tma_prefetch_desc(&tmX);
        tma_prefetch_desc(&tmY);
        for (int s = 0; s < XS; ++s) {
            mbar_init(xfull0 + 8 * s, Cfg::LOCK ? 1 + 4 : 1);   // LOCK: the X producer's expect_tx + the 4 dequant warps
            mbar_init(xempty0 + 8 * s, 1);      // MMA commit
        }
        for (int s = 0; s < PS; ++s) {
            mbar_init(pfull0 + 8 * s, 1);
            mbar_init(pempty0 + 8 * s, 4);      // the 4 warps of the dequant group that read it
        }
        for (int a = 0; a < NB; ++a) {
            mbar_init(afull0 + 8 * a, 4);       // the 4 dequant warps that fill it (unused with LOCK)
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

    // Programmatic dependent launch: only the roles that touch activations wait for the previous grid
    // -- the X producer before its first load, the epilogue warps before anything they store (which
    // also keeps "this grid complete => every earlier grid complete": no CTA exits before its epilogue
    // warps have waited).  The weight stream and the dequantisers depend on nothing the previous grid
    // writes, so the first k-blocks are fetched and dequantised during its tail.
    pdl_launch_dependents();   // the next kernel may become resident now; it blocks in its own wait
    const long long t_start = clock64();
#ifdef ARIA_DEBUG
    if (threadIdx.x == 0 && p.prof) {
        unsigned long long gt;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));
        p.prof[blockIdx.x * 64 + 14] = static_cast<long long>(gt);
    }
#endif

    // Producer / MMA warps: warp-uniform loops, one elected lane issues (see gemm_w8a8.cu).
    if (warp == 0) {
        // ------------------------------------------------------------ TMA producer: X
        pdl_wait_prior_grid();
        int stage = 0;
        uint32_t phase = 0;
        for (int u = unit0; u < num_units; u += unit_step) {
            const int tile = u / S, sp = u % S;
            const int t0 = (tile / num_n) * TT;
            const int kb0 = (sp * num_kb) / S, kb1 = ((sp + 1) * num_kb) / S;
            for (int kb = kb0; kb < kb1; ++kb) {
                const uint32_t xe = xempty0 + 8 * stage, xf = xfull0 + 8 * stage;
                mbar_wait(xe, phase ^ 1);
#ifdef ARIA_DEBUG
                if ((p.dbg == 1 && (kb & 1)) || p.dbg == 2) {
                    if (elect_one()) mbar_arrive(xf);
                    __syncwarp();
                    if (++stage == XS) { stage = 0; phase ^= 1; }
                    continue;
                }
#endif
                if (elect_one()) {
                    mbar_arrive_expect_tx(xf, Cfg::X_BYTES);
                    tma_load_2d(sX + stage * Cfg::X_BYTES, &tmX, kb * W4_BK, t0, xf);
                }
                __syncwarp();
                if (++stage == XS) { stage = 0; phase ^= 1; }
            }
        }
        if (lane == 0) prof_stamp(p, 0, t_start);
    } else if (warp == 2) {
        // ------------------------------------------------------------ TMA producer: packed weights
        const uint64_t pol_w = policy_evict_first();  // weights are streamed once per launch
        int stage = 0;
        uint32_t phase = 0;
        for (int u = unit0; u < num_units; u += unit_step) {
            const int tile = u / S, sp = u % S;
            const int n0 = (tile % num_n) * UN;
            const int kb0 = (sp * num_kb) / S, kb1 = ((sp + 1) * num_kb) / S;
            for (int kb = kb0; kb < kb1; ++kb) {
                mbar_wait(pempty0 + 8 * stage, phase ^ 1);
                if (elect_one()) {
                    mbar_arrive_expect_tx(pfull0 + 8 * stage, Cfg::P_BYTES);
                    tma_load_2d_hint(sP + stage * Cfg::P_BYTES, &tmP, kb * Cfg::P_ROW, n0,
                                     pfull0 + 8 * stage, pol_w);
                }
                __syncwarp();
                if (++stage == PS) { stage = 0; phase ^= 1; }
            }
        }
        if (lane == 0) prof_stamp(p, 6, t_start);
    } else if (warp == 1) {
        // ------------------------------------------------------------ MMA issuer
        {
            constexpr uint32_t idesc = idesc_bf16(UN, TT);
            const uint64_t desc_hi = make_smem_desc_sw128(0);
            int stage = 0, ab = 0, acc = 0;
            uint32_t phase = 0, aphase = 0, acc_phase = 0;
            long long w_x = 0, w_a = 0, w_t = 0, w_f = 0, w_m = 0, w_c1 = 0, w_c2 = 0;
            for (int u = unit0; u < num_units; u += unit_step) {
                const int sp = u % S;
                const int kb0 = (sp * num_kb) / S, kb1 = ((sp + 1) * num_kb) / S;
                W4_TIMED(w_t, mbar_wait(tempty0 + 8 * acc, acc_phase ^ 1));
                const uint32_t d_tmem = tmem_base + acc * Cfg::ACC_STRIDE;
                for (int kb = kb0; kb < kb1; ++kb) {
                    W4_TIMED(w_x, mbar_wait(xfull0 + 8 * stage, phase));   // X landed (LOCK: and weights dequantised)
                    if (!Cfg::LOCK) W4_TIMED(w_a, mbar_wait(afull0 + 8 * ab, aphase));     // weights dequantised
                    W4_TIMED(w_f, tc_fence_after());
                    const uint64_t a_desc = desc_hi | (((sA + ab * Cfg::A_BYTES) & 0x3FFFF) >> 4);
                    const uint32_t a_tmem = tmem_base + Cfg::A_COL0 + ab * 32;
                    const uint64_t b_desc = desc_hi | (((sX + stage * Cfg::X_BYTES) & 0x3FFFF) >> 4);
                    if (elect_one()) {
                        const long long t_m_ = W4_CLK();
#ifdef ARIA_DEBUG
                        if (p.prof && kb - kb0 >= 40 && kb - kb0 < 44 && u == unit0) p.prof[blockIdx.x * 64 + 24 + (kb - kb0 - 40)] = t_m_ - t_start;
#endif
#pragma unroll
                        for (int k = 0; k < 4; ++k) {  // 4 x (K = 16 bf16 = 32 bytes of X / 8 TMEM columns of A)
#ifdef ARIA_DEBUG
                            if (p.dbg == 4 && k != 0) continue;     // timing experiment: a quarter of the MMAs
#endif
                            if (Cfg::ATM) mma_f16_ts(d_tmem, a_tmem + 8 * k, b_desc + 2 * k, idesc, (kb != kb0 || k != 0) ? 1u : 0u);
                            else mma_f16_ss(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb != kb0 || k != 0) ? 1u : 0u);
                        }
                        const long long t_c_ = W4_CLK();
                        w_m += t_c_ - t_m_;
                        {
                            tc_commit(xempty0 + 8 * stage);
                            w_c1 += W4_CLK() - t_c_;
                            if (!Cfg::LOCK) tc_commit(aempty0 + 8 * ab);
                            if (kb == kb1 - 1) tc_commit(tfull0 + 8 * acc);
                        }
                    }
                    __syncwarp();
                    if (++stage == XS) { stage = 0; phase ^= 1; }
                    if (++ab == NB) { ab = 0; aphase ^= 1; }
                }
                if (++acc == 2) { acc = 0; acc_phase ^= 1; }
            }
            if (lane == 0) prof_stamp(p, 1, t_start);
#ifdef ARIA_DEBUG
            if (lane == 0 && p.prof) { p.prof[blockIdx.x * 64 + 5] = w_x; p.prof[blockIdx.x * 64 + 7] = w_a; p.prof[blockIdx.x * 64 + 12] = w_t; }
            if (p.prof && w_m != 0) {   // the elected lane
                p.prof[blockIdx.x * 64 + 20] = w_f; p.prof[blockIdx.x * 64 + 21] = w_m;
                p.prof[blockIdx.x * 64 + 22] = w_c1; p.prof[blockIdx.x * 64 + 23] = w_c2;
            }
#endif
        }
    } else if (warp >= W4_DEQ_WARP0) {
        // ------------------------------------------------------------ dequantiser groups
        // hand-off of one dequantised row (64 bf16 = 8 x 16 B, k ascending) to the MMA: tensor memory
        // (this thread's lane, 32 columns of the slot) or the 128-byte-swizzled shared-memory A tile
        long long d_pf = 0, d_ae = 0, d_st = 0, d_ar = 0;         // debug builds: cycles in each wait of this warp
        auto publish_a = [&](const uint4 (&o)[8], int it_, uint32_t rowoff_, uint32_t xr_, int q_) {
            const int ab = it_ % NB;
            if (Cfg::LOCK) {       // the MMAs of k-block it_ - NB (this slot's previous tenant) have retired
                if (it_ >= NB) W4_TIMED(d_ae, mbar_wait(xempty0 + 8 * ((it_ - NB) % XS), ((it_ - NB) / XS) & 1));
            } else {
                W4_TIMED(d_ae, mbar_wait(aempty0 + 8 * ab, ((it_ / NB) & 1) ^ 1));     // MMAs reading this A buffer retired
            }
            const long long t_st_ = W4_CLK();
            if (Cfg::ATM) {
                tc_fence_after();
                uint32_t w[32];
#pragma unroll
                for (int j = 0; j < 8; ++j) { w[4 * j] = o[j].x; w[4 * j + 1] = o[j].y; w[4 * j + 2] = o[j].z; w[4 * j + 3] = o[j].w; }
#ifdef ARIA_DEBUG
                if (p.dbg == 6) {            // timing experiment: no tensor-memory store (results are WRONG)
                    if (w[0] == 0x12345678u && w[31] == 0x9abcdef0u) static_cast<uint32_t*>(p.Y)[0] = w[7];
                } else
#endif
                {
                tmem_st_32x32b_x32(tmem_base + Cfg::A_COL0 + ab * 32 + (static_cast<uint32_t>(q_ * 32) << 16), w);
                tmem_wait_st();
                }
                tc_fence_before();
            } else {
                const uint32_t rowb = sA + ab * Cfg::A_BYTES + rowoff_;
#pragma unroll
                for (int j = 0; j < 8; ++j) sts128(rowb + ((static_cast<uint32_t>(j) ^ xr_) << 4), o[j]);
                fence_proxy_async_smem();                  // generic-proxy writes -> async proxy (MMA)
            }
            __syncwarp();
            const long long t_ar_ = W4_CLK();
            d_st += t_ar_ - t_st_;
            if (lane == 0) {                                       // one arrival per warp, on the leader's barrier
                mbar_arrive(Cfg::LOCK ? xfull0 + 8 * (it_ % XS) : afull0 + 8 * ab);
            }
            __syncwarp();
            d_ar += W4_CLK() - t_ar_;
#ifdef ARIA_DEBUG
            if (p.prof && lane == 0 && it_ >= 40 && it_ < 44) {
                p.prof[blockIdx.x * 64 + 32 + (it_ - 40) * 4 + q_] = clock64() - t_start;     // published, per warp
                p.prof[blockIdx.x * 64 + 48 + (it_ - 40) * 4 + q_] = t_st_ - t_start;         // slot was free
            }
#endif
        };
        const int dw = warp - W4_DEQ_WARP0;
        const int g = dw >> 2;                    // group = A buffer index
        const int r = (dw & 3) * 32 + lane;       // weight row inside the tile
        const int gpr = p.K >> 5;                 // groups per weight row
        const uint32_t rowoff = (r >> 3) * 1024 + (r & 7) * 128;
        const uint32_t xr = r & 7;
        const uint32_t off0 = r * Cfg::P_ROW;
        const uint32_t poff0 = off0 ^ (((off0 >> 7) & 1u) << 4);          // WB = 4: 32-byte swizzle
        const uint32_t poff1 = (off0 + 16) ^ (((off0 >> 7) & 1u) << 4);
        const uint32_t px8 = (r >> 1) & 3;                                 // WB = 8: 64-byte swizzle (chunk ^ bits 7-8)
        int it = 0;                               // running k-block counter of this CTA
        for (int u = unit0; u < num_units; u += unit_step) {
            const int tile = u / S, sp = u % S;
            const int n0 = (tile % num_n) * UN;
            const int kb0 = (sp * num_kb) / S, kb1 = ((sp + 1) * num_kb) / S;
            const bool row_ok = n0 + r < p.N;
            if (WB == 8) {
                // ---- int8 codes, one fp32 scale per output channel (this thread's row)
                const float sw = row_ok ? __ldg(static_cast<const float*>(p.g_scale) + n0 + r) : 0.0f;
                for (int kb = kb0; kb < kb1; ++kb, ++it) {
                    if (it % G != g) continue;
                    const int stage = it % PS;
                    mbar_wait(pfull0 + 8 * stage, (it / PS) & 1);
                    const uint32_t ps = sP + stage * Cfg::P_BYTES + off0;
                    uint4 pk[4];
#pragma unroll
                    for (int c = 0; c < 4; ++c) pk[c] = lds128(ps + ((static_cast<uint32_t>(c) ^ px8) << 4));
                    uint4 o[8];
#pragma unroll
                    for (int c = 0; c < 4; ++c) dequant_i8x16(pk[c], sw, o[2 * c], o[2 * c + 1]);
                    __syncwarp();
                    if (lane == 0) mbar_arrive(pempty0 + 8 * stage);   // packed bytes are in registers
                    publish_a(o, it, rowoff, xr, dw & 3);
                }
                continue;
            }
            const uint32_t* srow = reinterpret_cast<const uint32_t*>(
                static_cast<const uint16_t*>(p.g_scale) + static_cast<int64_t>(row_ok ? n0 + r : 0) * gpr);
            // the two fp16 group scales of this row and a k-block: one aligned 32-bit load.  The load for
            // this group's NEXT k-block (kb + G) is issued before the current one is processed, which
            // takes the L2 round trip (uncoalesced: one line per row) off the per-k-block chain.
            auto load_scales = [&](int kb) -> uint32_t {
                uint32_t v = 0;
                if (row_ok && kb < kb1) {
                    if ((gpr & 1) == 0) {
                        v = __ldg(srow + kb);
                    } else {  // odd group count: rows are only 2-byte aligned
                        const uint16_t* s16 = reinterpret_cast<const uint16_t*>(srow);
                        v = __ldg(s16 + 2 * kb);
                        if (2 * kb + 1 < gpr) v |= static_cast<uint32_t>(__ldg(s16 + 2 * kb + 1)) << 16;
                    }
                }
                return v;
            };
            // first k-block of this unit that belongs to this group
            const int kfirst = kb0 + ((g - it % G) + G) % G;
            uint32_t sc_next = load_scales(kfirst);
            for (int kb = kb0; kb < kb1; ++kb, ++it) {
                if (it % G != g) continue;
                const int stage = it % PS;
                const uint32_t phase = (it / PS) & 1;
                const uint32_t sc2 = sc_next;
                sc_next = load_scales(kb + G);
                W4_TIMED(d_pf, mbar_wait(pfull0 + 8 * stage, phase));
                const uint32_t ps = sP + stage * Cfg::P_BYTES;
                const uint4 pk0 = lds128(ps + poff0);
                const uint4 pk1 = lds128(ps + poff1);
                uint4 o[8];
#ifdef ARIA_DEBUG
                if (p.dbg == 5) {                                   // timing experiment: no dequantiser arithmetic
#pragma unroll
                    for (int j = 0; j < 8; ++j) o[j] = pk0;
                } else
#endif
                {
                    const GroupConst gc = group_const(__half2float(__ushort_as_half(static_cast<uint16_t>(sc2 & 0xFFFFu))));
                    o[0] = dequant_word(pk0.x, gc); o[1] = dequant_word(pk0.y, gc);
                    o[2] = dequant_word(pk0.z, gc); o[3] = dequant_word(pk0.w, gc);
                }
#ifdef ARIA_DEBUG
                if (p.dbg != 5)
#endif
                {
                    const GroupConst gc = group_const(__half2float(__ushort_as_half(static_cast<uint16_t>(sc2 >> 16))));
                    o[4] = dequant_word(pk1.x, gc); o[5] = dequant_word(pk1.y, gc);
                    o[6] = dequant_word(pk1.z, gc); o[7] = dequant_word(pk1.w, gc);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(pempty0 + 8 * stage);   // packed bytes are in registers
                publish_a(o, it, rowoff, xr, dw & 3);
            }
        }
        if ((dw & 3) == 0 && lane == 0) prof_stamp(p, 2 + g, t_start);
#ifdef ARIA_DEBUG
        if (dw == 0 && lane == 0 && p.prof) {
            p.prof[blockIdx.x * 64 + 16] = d_pf; p.prof[blockIdx.x * 64 + 17] = d_ae;
            p.prof[blockIdx.x * 64 + 18] = d_st; p.prof[blockIdx.x * 64 + 19] = d_ar;
        }
#else
        (void)d_pf; (void)d_ae; (void)d_st; (void)d_ar;
#endif
    } else if (warp >= W4_EPI_WARP0) {
        // ------------------------------------------------------------ epilogue (warps 4..7)
        pdl_wait_prior_grid();
        const int q = warp & 3;
        int acc = 0;
        uint32_t acc_phase = 0;
        for (int u = unit0; u < num_units; u += unit_step) {
            const int tile = u / S, sp = u % S;
            const int n0 = (tile % num_n) * UN, t0 = (tile / num_n) * TT;
            const int n = n0 + q * 32 + lane;
            const bool n_ok = n < p.N;
            float bv = 0.0f;
            if (p.bias && n_ok) bv = __bfloat162float(static_cast<const __nv_bfloat16*>(p.bias)[n]);
            mbar_wait(tfull0 + 8 * acc, acc_phase);
            tc_fence_after();
            if (q == 0 && lane == 0) prof_stamp(p, 8 + 2 * min(3, (u - unit0) / unit_step), t_start);
            const uint32_t t_addr = tmem_base + acc * Cfg::ACC_STRIDE + (static_cast<uint32_t>(q * 32) << 16);
            if (S == 1) {
                // Transpose through shared memory: this thread owns output channel n and 32 tokens
                // of the chunk; it writes its column of the [32 tokens x 32 channels] block (rows of
                // 64 B bf16 / 128 B fp32, swizzled as the output tensor map expects), then one TMA
                // store writes the block -- coalesced, asynchronous, clipped at M and N.
                const uint32_t stg = base + Cfg::STG_OFF + (warp - W4_EPI_WARP0) * Cfg::STG_BYTES;
                if (p.out_t == ARIA_BF16) {
                    // bf16 fast path (measured: the epilogue of the LAST tile of a CTA is fully exposed --
                    // 8.6k of 28k cycles for a one-tile-per-CTA layer with the generic loop below).  One
                    // tcgen05.ld of 32 columns per block, everything unrolled: the swizzled address of
                    // token row j is one of 4 per-thread bases (chunk index ^ ((j >> 1) & 3)) plus the
                    // immediate j * 64, so a value costs add + (GELU) + cvt + st.shared.u16.
                    uint32_t sb[4];
#pragma unroll
                    for (int cj = 0; cj < 4; ++cj)
                        sb[cj] = stg + ((static_cast<uint32_t>((lane >> 3) ^ cj)) << 4) + ((lane * 2) & 15);
#pragma unroll 1
                    for (int c = 0; c < TT / 32; ++c) {
                        uint32_t v[32];
                        tmem_ld_32x32b_x32(t_addr + c * 32, v);
                        if (lane == 0) tma_store_wait_read<0>();   // previous block left the staging buffer
                        tmem_wait_ld();
                        __syncwarp();
#pragma unroll
                        for (int j = 0; j < 32; j += 2) {
                            float y0 = __uint_as_float(v[j]) + bv, y1 = __uint_as_float(v[j + 1]) + bv;
                            if (GELU) gelu_erf2(y0, y1);
                            const uint16_t h0 = __bfloat16_as_ushort(__float2bfloat16_rn(y0));
                            const uint16_t h1 = __bfloat16_as_ushort(__float2bfloat16_rn(y1));
                            asm volatile("st.shared.u16 [%0], %1;" ::"r"(sb[(j >> 1) & 3] + j * 64), "h"(h0) : "memory");
                            asm volatile("st.shared.u16 [%0], %1;" ::"r"(sb[(j >> 1) & 3] + (j + 1) * 64), "h"(h1) : "memory");
                        }
                        fence_proxy_async_smem();
                        __syncwarp();
                        if (lane == 0) {
                            tma_store_2d(&tmY, stg, n0 + q * 32, t0 + c * 32);
                            tma_store_commit();
                        }
                    }
                } else {
#pragma unroll 1
                for (int c = 0; c < TT / 32; ++c) {
                    if (lane == 0) tma_store_wait_read<0>();   // previous block left the staging buffer
                    __syncwarp();
#pragma unroll 1
                    for (int gq = 0; gq < 4; ++gq) {           // 8 tokens per step keeps the code small
                        uint32_t v[8];
                        tmem_ld_32x32b_x8(t_addr + c * 32 + gq * 8, v);
                        tmem_wait_ld();
#pragma unroll
                        for (int jj = 0; jj < 8; ++jj) {
                            const int j = gq * 8 + jj;         // token row inside the block
                            float y = __uint_as_float(v[jj]) + bv;
                            if (GELU) y = gelu_erf(y);
                            const uint32_t off = j * 128 + ((((lane * 4) >> 4) ^ (j & 7)) << 4) + ((lane * 4) & 15);
                            asm volatile("st.shared.f32 [%0], %1;" ::"r"(stg + off), "f"(y) : "memory");
                        }
                    }
                    fence_proxy_async_smem();
                    __syncwarp();
                    if (lane == 0) {
                        tma_store_2d(&tmY, stg, n0 + q * 32, t0 + c * 32);
                        tma_store_commit();
                    }
                }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tempty0 + 8 * acc);
            } else {
                float* part = p.partials + static_cast<int64_t>(sp) * p.M * p.N;
                float* prow = part + static_cast<int64_t>(t0) * p.N + n;
                const int tleft = p.M - t0;
#pragma unroll 1
                for (int c = 0; c < TT / 32; ++c) {
                    uint32_t v[32];
                    tmem_ld_32x32b_x32(t_addr + c * 32, v);
                    tmem_wait_ld();
                    if (n_ok) {
#pragma unroll
                        for (int j = 0; j < 32; ++j)
                            if (c * 32 + j < tleft) __stcg(prow + static_cast<int64_t>(c * 32 + j) * p.N, __uint_as_float(v[j]));
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tempty0 + 8 * acc);
                // Reduction, spread over the splits: every split's warp publishes its partials, waits until
                // all S splits of this (tile, quarter) have published, and then reduces ITS share of the
                // tile's tokens (a contiguous 1/S) in fixed split order -- deterministic, and S times more
                // warps than a last-arriver reduction (measured: that took 48 of 58 us at 512 x 6144 -> 1536
                // with 6 splits).  No deadlock: the S units of a tile are consecutive unit indices, hence
                // on S different CTAs, each of which has finished every smaller unit it owns before it
                // gets here; a unit's mainloop and partial stores wait for nobody.
                __threadfence();
                __syncwarp();
                if (lane == 0) {
                    unsigned* cnt = p.counters + tile * 4 + q;
                    atomicAdd(cnt, 1u);
                    const long long t_spin = clock64();
                    unsigned seen;
                    do {
                        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(cnt) : "memory");
                        if (seen < static_cast<unsigned>(S)) {
                            __nanosleep(100);
                            if (clock64() - t_spin > 4000000000LL) {
                                printf("aria: split-K watchdog (block %d tile %d)\n", blockIdx.x, tile);
                                __trap();
                            }
                        }
                    } while (seen < static_cast<unsigned>(S));
                }
                __syncwarp();
                __threadfence();
                {
                    const int tmax = min(TT, p.M - t0);
                    const int j_beg = (sp * tmax) / S, j_end = ((sp + 1) * tmax) / S;
                    const int64_t sstride = static_cast<int64_t>(p.M) * p.N;
                    for (int j0 = j_beg; j0 < j_end; j0 += 8) {   // 8 tokens x 4 splits = 32 loads in flight
                        float y[8];
#pragma unroll
                        for (int j = 0; j < 8; ++j) y[j] = 0.0f;
                        for (int s = 0; s < S; s += 4) {          // fixed split order: deterministic sum
                            float a[4][8];
#pragma unroll
                            for (int ss = 0; ss < 4; ++ss)
#pragma unroll
                                for (int j = 0; j < 8; ++j) {
                                    const int64_t idx = static_cast<int64_t>(t0 + j0 + j) * p.N + n;
                                    const bool ok = n_ok && j0 + j < j_end && s + ss < S;
                                    a[ss][j] = ok ? __ldcg(p.partials + (s + ss) * sstride + idx) : 0.0f;
                                }
#pragma unroll
                            for (int ss = 0; ss < 4; ++ss)
#pragma unroll
                                for (int j = 0; j < 8; ++j) y[j] += a[ss][j];
                        }
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const int64_t idx = static_cast<int64_t>(t0 + j0 + j) * p.N + n;
                            if (n_ok && j0 + j < j_end) w4_store(p.Y, p.out_t, idx, GELU ? gelu_erf(y[j] + bv) : y[j] + bv);
                        }
                    }
                }
            }
            if (q == 0 && lane == 0) prof_stamp(p, 9 + 2 * min(3, (u - unit0) / unit_step), t_start);
            if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        }
    }

    if (warp >= W4_EPI_WARP0 && warp < W4_DEQ_WARP0 && lane == 0) tma_store_wait<0>();
    tc_fence_before();
    __syncthreads();
#ifdef ARIA_DEBUG
    if (threadIdx.x == 0 && p.prof) {
        unsigned long long gt;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));
        p.prof[blockIdx.x * 64 + 15] = static_cast<long long>(gt);
        p.prof[blockIdx.x * 64 + 13] = clock64() - t_start;
    }
#endif
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
    }
}

template <int TT, bool GELU, int WB>
static int launch_w4(const void* X, int M, int K, const uint8_t* Wq4, int N, const W4Params& p,
                     int grid, cudaStream_t st, bool pdl) {
    using Cfg = W4Cfg<TT, WB>;
    static std::atomic<uint64_t> attr_done{0};
    auto kern = w4a16_gemm_kernel<TT, GELU, WB>;
    if (!ensure_dyn_smem(kern, Cfg::SMEM_BYTES, attr_done)) return ARIA_ERR_CUDA;
    CUtensorMap tmP, tmX, tmY;
    int rc = make_tmap_2d(&tmP, Wq4, 1, N, K * WB / 8, W4_BN, Cfg::P_ROW, Cfg::P_ROW);
    if (rc != ARIA_OK) return rc;
    rc = make_tmap_2d(&tmX, X, 2, M, K, Cfg::X_ROWS, 64, 128);
    if (rc != ARIA_OK) return rc;
    // output: box = 32 tokens x 32 channels (64 B bf16 rows / 128 B fp32 rows)
    rc = make_tmap_2d(&tmY, p.Y, p.out_t == ARIA_F32 ? 4 : 2, M, N, 32, 32, p.out_t == ARIA_F32 ? 128 : 64);
    if (rc != ARIA_OK) return rc;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(Cfg::THREADS);
    cfg.dynamicSmemBytes = Cfg::SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    int na = 0;
    if (p.splits > 1) {
        // split-K units wait for one another (per-tile counters): a COOPERATIVE launch (grid <= #SMs, one CTA per SM)
        // either has every CTA resident or fails with ARIA_ERR_CUDA -- it cannot deadlock when another tenant's
        // kernel holds SMs.  Such a launch is not also a programmatic dependent.
        at[0].id = cudaLaunchAttributeCooperative;
        at[0].val.cooperative = 1;
        na = 1;
    } else if (pdl) {
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        na = 1;
    }
    cfg.attrs = at;
    cfg.numAttrs = na;
    return cudaLaunchKernelEx(&cfg, kern, tmP, tmX, tmY, p) == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
}

// Tile / split-K plan shared by the launcher and aria_workspace_bytes.  Cost model (cycles): a unit
// spends per k-block max(MMA, shared memory) = (256 TT + 40 KB) / 128 B/clk = 2 TT + 320 (the X tile
// is written by TMA and read by the MMA; packed weights, dequantised A tile and its MMA read are the
// constant), plus an epilogue ~ 40 TT, a fixed ~3000, and for split-K the fp32 partial round trip
// ~ 100 TT + 4000.  Pick the (TT, splits) with the fewest wave-quantised cycles.
void w4_plan(int M, int N, int K, int sms, int* tt_out, int* splits_out) {
    const int num_kb = (K + W4_BK - 1) / W4_BK;
    const int num_n = (N + W4_BN - 1) / W4_BN;
    const int tts[5] = {256, 192, 128, 64, 32};
    long best = -1;
    int best_tt = 32, best_s = 1;
    for (int i = 0; i < 5; ++i) {
        const int tt = tts[i];
        if (tt > 32 && tt >= 2 * M) continue;                 // mostly padding
        const int tiles = num_n * ((M + tt - 1) / tt);
        int smax = sms / tiles;
        if (smax > num_kb) smax = num_kb;
        if (smax > 16) smax = 16;
        if (smax < 1) smax = 1;
        for (int s = 1; s <= smax; ++s) {
            const long units = static_cast<long>(tiles) * s;
            const long waves = (units + sms - 1) / sms;
            const long kb = (num_kb + s - 1) / s;
            // measured steady-state cycles per 64-k block (role timestamps, C5 layers at M = 2048): tt = 256, A in
            // shared memory: ~800; tt = 192, A in tensor memory: ~560; smaller tiles: dequantiser bound, ~450
            const long kcost = tt == 256 ? 800 : tt == 192 ? 560 : 450;
            long unit = kb * kcost + 40L * tt + 3000;
            if (s > 1) unit += 100L * tt + 4000;
            const long cost = waves * unit;
            if (best < 0 || cost < best) { best = cost; best_tt = tt; best_s = s; }
        }
    }
    *tt_out = best_tt; *splits_out = best_s;
}

size_t w4_workspace_bytes(int M, int N, int K, int sms) {
    int tt, s;
    w4_plan(M, N, K, sms, &tt, &s);
    const size_t tiles = static_cast<size_t>((N + W4_BN - 1) / W4_BN) * ((M + tt - 1) / tt);
    size_t counters = (tiles * 4 * sizeof(unsigned) + 255) / 256 * 256;
    size_t partials = s > 1 ? static_cast<size_t>(s) * M * N * sizeof(float) : 0;
    return counters + (partials + 255) / 256 * 256;
}

int launch_gemm_w4a16(const void* X, int M, int K, const uint8_t* Wq4, const void* g_scale,
                      int N, const void* bias, int act, void* Y, int yt, void* ws, size_t ws_bytes,
                      cudaStream_t st, bool pdl, int wbits) {
    const int sms = num_sms();
    if (sms <= 0) return ARIA_ERR_CUDA;
    int tt, s;
    w4_plan(M, N, K, sms, &tt, &s);
    if (s > 1 && (ws == nullptr || ws_bytes < w4_workspace_bytes(M, N, K, sms))) s = 1;
    W4Params p;
    p.g_scale = g_scale; p.bias = bias; p.Y = Y;
    p.act = act; p.out_t = yt; p.M = M; p.N = N; p.K = K; p.splits = s;
#ifdef ARIA_DEBUG
    p.dbg = dbg_env("ARIA_W4_DBG") ? atoi(dbg_env("ARIA_W4_DBG")) : 0;
    p.prof = g_w4_prof ? g_w4_prof + static_cast<size_t>(g_w4_prof_launch++ % 256) * 148 * 64 : nullptr;
#endif
    const size_t tiles = static_cast<size_t>((N + W4_BN - 1) / W4_BN) * ((M + tt - 1) / tt);
    p.counters = static_cast<unsigned*>(ws);
    p.partials = s > 1 ? reinterpret_cast<float*>(static_cast<uint8_t*>(ws) +
                                                  (tiles * 4 * sizeof(unsigned) + 255) / 256 * 256)
                       : nullptr;
    const int units = static_cast<int>(tiles) * s;
    const int grid = units < sms ? units : sms;
    if (s > 1 && cudaMemsetAsync(p.counters, 0, tiles * 4 * sizeof(unsigned), st) != cudaSuccess)
        return ARIA_ERR_CUDA;
    const bool gelu = act == ARIA_ACT_GELU_ERF;
#define ARIA_W4_LAUNCH(TTV)                                                                           \
    if (wbits == 8)                                                                                   \
        return gelu ? launch_w4<TTV, true, 8>(X, M, K, Wq4, N, p, grid, st, pdl)                      \
                    : launch_w4<TTV, false, 8>(X, M, K, Wq4, N, p, grid, st, pdl);                    \
    return gelu ? launch_w4<TTV, true, 4>(X, M, K, Wq4, N, p, grid, st, pdl)                          \
                : launch_w4<TTV, false, 4>(X, M, K, Wq4, N, p, grid, st, pdl)
    if (tt == 32) { ARIA_W4_LAUNCH(32); }
    if (tt == 64) { ARIA_W4_LAUNCH(64); }
    if (tt == 128) { ARIA_W4_LAUNCH(128); }
    if (tt == 192) { ARIA_W4_LAUNCH(192); }
    ARIA_W4_LAUNCH(256);
#undef ARIA_W4_LAUNCH
}

}  // namespace aria
