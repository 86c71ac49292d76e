// w4a16_stream.cu -- S4 at small M (<= 32 tokens): ONE persistent weight-streaming kernel for a whole
// list of W4A16 linears (a denoising step's stack, or a batch of independent linears).
//
// At M <= 32 a linear moves ~4-5 MB of packed weights and does ~0.2 us of tensor work: it is bound by
// HBM, and a kernel per layer cannot even ramp the memory system up (0.7 us of data per launch).  Here
// the weight stream of ALL layers runs back to back through one deep TMA ring per SM; nothing in it
// depends on activations, so it keeps flowing while a layer waits for its input.
//
// Work unit = (layer, 128 output channels, ALL of K); a stage is 256 k-values of 128 weight rows:
// 16 KB of packed int4 (128-byte rows, SWIZZLE_128B) + 2 KB of fp16 group scales.  There is no
// split-K: a cross-CTA reduction costs a chain of ~6 global round trips per unit (partials, fence,
// counter, re-read) -- measured 4k-25k cycles per unit against ~2.7k cycles of dequantisation, the
// reason the per-layer kernel is latency bound at M = 32.  Instead the host deals the units of ALL
// layers to the CTAs at plan time (one global order, always to the CTA with the fewest stages so far),
// so every CTA streams the same number of stages and a layer with few tiles simply overlaps its
// neighbours; layers that read an earlier layer's output are moved behind the independent ones.
// Roles (768 threads, 1 CTA / SM; the single latency-critical warps have the HIGH warp ids because the
// SM's warp arbiter prefers them):
//   warps 0-15  four dequantiser groups (thread = weight row; group g = 64-k sub-block g of every
//               stage): LDS -> registers -> tcgen05.st into a ring of TMEM A slots.  The dequantised
//               tile never touches shared memory: per weight shared memory sees 0.5 B (TMA write)
//               + 0.5 B (LDS) instead of 4.5 B with an smem A tile, which would cap the stream at
//               ~28 weights/clk/SM -- below the ~41 weights/clk/SM that HBM delivers.
//   warps 16-19 epilogue: tcgen05.ld -> + bias, GELU, cast -> coalesced stores; a layer that feeds a
//               later layer also writes that layer's fp16 operand copy and bumps its completion
//               counter (release).
//   warp 20     X producer: [32 tokens x 64 k] fp16 tiles by TMA (L2 resident), after the unit's
//               dependency (a chained layer waits for its producer layer's completion counter).
//   warp 21     MMA issuer: tcgen05.mma kind::f16, A = dequantised weights IN TENSOR MEMORY
//               (128 rows x 16 k per instruction), B = X tile in shared memory, D = fp32 in TMEM;
//               17 instructions per stage: 16 of weights + 1 of zero points (below).
//   warp 22     weight producer: packed + scale tiles by TMA, evict-first (the HBM stream).
// Dequantisation (AF16), 9 instructions per 8 weights (the loop is issue bound, so this count IS the
// kernel's speed): the offset-binary nibble u = q + 8 is masked into the mantissa of an fp16 constant
// (1024 + u or 64 + u, one LOP3 per pair of weights) and one HFMA2 (B + u) sg - B sg returns
// fp16_rn(u sg), the correctly rounded UNSIGNED dequantised weight.  The zero point -8 sg x is linear
// and exact, so the tensor core applies it: per stage 16 extra k-values with A = -8 sg of the stage's
// 8 groups and B = the (hi, lo) fp16 split of the groups' activation sums.  The dequantised weight is
// therefore w^ = fp16_rn((q + 8) sg) - 8 sg (reading R12c, oracle variant 3).  kind::f16
// takes fp16 x fp16 or bf16 x bf16 but not a mix (illegal instruction on sm_100a), so the bf16
// activations are converted to fp16 too: external inputs once per launch by the dequantiser and
// epilogue warps, chained outputs by the producing epilogue (exact for 2^-14 <= |x| <= 65504), both
// in the k order the dequantiser produces ([0,4,1,5,2,6,3,7] inside each 8-k word) and with the
// group sums appended to every 256-k stage.  AF16 = false keeps w^ = bf16_rne(q sg) and bf16
// activations (18 instructions per 8 weights; used when a chained layer's geometry rules the fp16
// copy out).
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "internal.cuh"

namespace aria {

constexpr int WS_TT = 32;        // tokens per tile = MMA N
constexpr int WS_ROWS = 128;     // output channels per tile = MMA M
constexpr int WS_SBK = 256;      // k-values per stage
constexpr int WS_PS = 6;         // weight ring depth (stages of 18 KB); the dequantiser loop is unrolled by WS_PS
constexpr int WS_XS = 4;         // X ring depth (stages of 20 KB): X must be requested BEFORE the weights of its stage
constexpr int WS_NA = 3;         // TMEM A slots, one STAGE each (128 columns = 128 rows x 256 k)
constexpr int WS_G = 4;          // dequantiser groups
constexpr int WS_NTACC = 3;      // accumulator buffers: a slow (GELU + fp16 copy) epilogue must not stall the MMA
// Warp roles.  The SM's warp arbiter prefers HIGH warp ids (B300_MICROARCH "hi-wid-first"), so the
// latency-critical single warps (MMA issue, the two TMA producers) and the epilogue sit above the 16
// dequantiser warps, which would otherwise win every issue slot they are eligible for.
constexpr int WS_DEQ_WARP0 = 0;                              // warps 0-15 (warp % 4 == TMEM lane quarter)
constexpr int WS_EPI_WARP0 = 4 * WS_G;                       // warps 16-19 (same)
constexpr int WS_XPROD_WARP = WS_EPI_WARP0 + 4;              // 20
constexpr int WS_MMA_WARP = WS_EPI_WARP0 + 5;                // 21
constexpr int WS_WPROD_WARP = WS_EPI_WARP0 + 6;              // 22 (warp 23 idles)
constexpr int WS_THREADS = 32 * (WS_EPI_WARP0 + 8);          // 768
constexpr int WS_P_BYTES = WS_ROWS * 128;                    // 16 KB
constexpr int WS_S_BYTES = WS_ROWS * 16;                     // 2 KB
constexpr int WS_XSUB = 5;                                   // X sub-tiles [32 x 64] per stage: 4 of activations + 1 of group sums (AF16)
constexpr int WS_X_BYTES = WS_XSUB * WS_TT * 128;            // 20 KB
constexpr int WS_XLD = 320;                                  // fp16 elements per 256-k stage of the X16 copy: 256 x + 16 sums + pad
constexpr int WS_A_SLOT = 136;                               // TMEM columns per A slot: 128 (256 k) + 8 (16 zero-point k)
constexpr int WS_P_OFF = 0;
constexpr int WS_X_OFF = WS_P_OFF + WS_PS * WS_P_BYTES;
constexpr int WS_S_OFF = WS_X_OFF + WS_XS * WS_X_BYTES;
constexpr int WS_BAR_OFF = WS_S_OFF + WS_PS * WS_S_BYTES;
constexpr int WS_NBAR = 2 * WS_PS + 2 * WS_XS + 2 * WS_NA + 2 * WS_NTACC;
constexpr int WS_SMEM_BYTES = WS_BAR_OFF + WS_NBAR * 8 + 16 + 1024;
// Accumulators (WS_NACC > 1 would spread the k-steps over independent accumulators that the epilogue
// adds; measured: no gain -- back-to-back N = 32 MMAs into one accumulator do not serialise).
constexpr int WS_NACC = 1;
constexpr int WS_ACC_COL0 = 0;                               // 2 buffers x 4 fp32 accumulators x 32 columns
constexpr int WS_A_COL0 = WS_NTACC * WS_NACC * WS_TT;
constexpr int WS_TMEM_COLS = 512;
static_assert(WS_SMEM_BYTES <= 227 * 1024, "shared memory");
static_assert(WS_PS % WS_NA == 0 && (WS_PS / WS_NA) % 2 == 0, "the unrolled dequantiser loop needs static A-slot parities");
static_assert(WS_A_COL0 + WS_NA * WS_A_SLOT <= WS_TMEM_COLS, "tensor memory");

// One linear of the list, as the kernel sees it (device memory; tensor maps need 64-byte alignment).
struct alignas(128) WsLayer {
    CUtensorMap tmP;          // packed int4 [N, K/2] u8, box 128 rows x 128 B, SWIZZLE_128B
    CUtensorMap tmS;          // group scales [N, K/32] fp16, box 128 rows x 8, no swizzle
    CUtensorMap tmX;          // activations [M, K] bf16, box 32 rows x 64, SWIZZLE_128B
    const void* bias;         // bf16 [N] or nullptr
    void* Y;                  // [M, N] bf16 / fp32
    void* Y16;                // fp16 copy of the bf16 output for the layers that read it (AF16), or nullptr
    int N, K;
    int num_n, num_sb;        // 128-row tiles, 256-k stages
    int act, out_t;
    int dep;                  // layer whose completion this layer's input needs, or -1
    int notify;               // 1 if a later layer depends on this one (epilogue bumps done[l])
    unsigned done_target;     // num_n * 4 quarter-tiles complete the layer
    int in_ext;               // index of the external input this layer reads (AF16 range tracking), or -1 if chained
};

// AF16: external bf16 inputs are converted once per launch to fp16 (the MMA needs both operands in
// the same 16-bit format); segment i covers 16-byte chunks [chunk0, chunk0 + chunks).
struct WsConv {
    const uint4* src;         // bf16 [M, K], 8 per chunk
    uint16_t* dst;            // fp16 [M, ld16] in the stream layout (see x16_pos)
    int chunk0, chunks;
    int kc8, ld16;            // K / 8 chunks per row; K / 256 * WS_XLD
};

struct WsParams {
    const WsLayer* layers;    // [n_layers]
    const WsConv* conv;       // [n_conv] (AF16)
    int n_conv, conv_chunks;
    // Dense schedule: CTA b owns units sched[b * max_units .. + sched_cnt[b].x), each {layer << 16 | tile,
    // stages of the unit}; sched_cnt[b] = {units, total stages}.  One load per unit, and the first
    // unit's address depends on nothing: it is fetched at kernel entry, before the prologue's barrier.
    const int2* sched;
    const int2* sched_cnt;
    int max_units;
    unsigned* done;           // [n_layers] completion counters + [n_layers] = CTAs done converting (zeroed before each launch)
    // Domain of the fp16 operand path (AF16), tracked per launch in words zeroed with `done`:
    //   flag   != 0: some activation (external or chained) or a 32-k group sum exceeds the fp16 range, or
    //               a whole input tensor is so small (0 < absmax < WS_MIN_ABSMAX) that fp16 subnormals
    //               would cost relative precision -> the bf16 fallback launch recomputes the list.
    //   inmax  [n_ext]    bit pattern of max |x| of every external input (conversion pre-pass)
    //   outmax [n_layers] bit pattern of max |y| of every chained output (producing epilogue)
    unsigned* flag;
    unsigned* inmax;
    unsigned* outmax;
    const unsigned* run_if;   // fallback launch: run only if *run_if != 0 (after the previous grid completed)
    int n_layers, M;
    long long* prof;          // debug builds: per-CTA role timestamps (16 per CTA), or nullptr
    int dbg;                  // debug builds (ARIA_WS_DBG): 1 = skip dequant math, 2 = skip MMAs
};

constexpr float WS_F16_MAX = 65504.0f;
constexpr float WS_MIN_ABSMAX = 0.0078125f;   // 2^-7: see DESIGN.md (fp16 subnormal error vs output magnitude)

#ifdef ARIA_DEBUG
static long long* g_ws_prof = nullptr;
void ws_set_profile_buffer(long long* p) { g_ws_prof = p; }
#endif
#define WS_TIMED(accum, stmt) do { if (PROF) { const long long t_ = clock64(); stmt; accum += clock64() - t_; } else { stmt; } } while (0)
#define WS_STAMP(slot) do { if (PROF && p.prof) p.prof[blockIdx.x * 16 + (slot)] = clock64() - t_start; } while (0)

__device__ __forceinline__ unsigned ld_acquire(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// Spin until a completion counter reaches its target.  Producers are earlier units of CTAs that are
// resident (grid <= #SMs, 1 CTA/SM); a watchdog turns a scheduling bug into a trap, not a hang.
__device__ __forceinline__ void wait_counter(const unsigned* p, unsigned target) {
    if (ld_acquire(p) >= target) return;
    const long long t0 = clock64();
    while (ld_acquire(p) < target) {
        __nanosleep(64);
        if (clock64() - t0 > 4000000000LL) {
            printf("aria: stream-kernel dependency watchdog (block %d)\n", blockIdx.x);
            __trap();
        }
    }
}
__device__ __forceinline__ uint32_t bf16x2_to_f16x2(uint32_t v) {
    const float lo = __uint_as_float(v << 16), hi = __uint_as_float(v & 0xFFFF0000u);
    uint32_t r;
    asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}
__device__ __forceinline__ void fence_proxy_async_all() {
    asm volatile("fence.proxy.async;" ::: "memory");
}
// ---- dequantisation, 8 codes of one 32-bit word (nibble i = code of k = 8w + i) -> 4 packed pairs
__device__ __forceinline__ uint32_t ws_lop_and_xor(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0x6A;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
__device__ __forceinline__ uint32_t hfma2_u32(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r;
    asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
// fp16 path, 9 instructions per 8 weights (1 SHF, 4 LOP3, 4 HFMA2).  The offset-binary nibble
// u = q + 8 (two's-complement nibble XOR 8) is dropped into the mantissa of an fp16 constant whose ulp
// is 1 at that bit position: bits 0-3 of 0x6400 (= 1024) give 1024 + u, bits 4-7 of 0x5400 (= 64) give
// 64 + u.  One HFMA2 (B + u) sg - B sg has an exact product and an exactly representable addend
// (B sg, B a power of two), so it returns fp16_rn(u sg): the correctly rounded UNSIGNED dequantised
// weight.  The zero point -8 sg x is exact and linear, so the tensor core applies it: 16 extra k per
// stage with A = -8 sg (per group) and B = the group sums of x (hi + lo fp16 split), see the MMA warp.
// Output register i holds the pair (k_i, k_{i+4}) of the word: the k order inside each 8-k word is
// [0,4,1,5,2,6,3,7], and the fp16 activation copy is written in the same order (x16_pos).
// S2 = (sg, sg), C0 = -(1024 sg), C1 = -(64 sg): exact unless 1024 sg overflows (sg > 63.9, i.e.
// |w| > 447: such a group takes the value inf/nan -- documented limit of the fp16 path).
__device__ __forceinline__ void dequant_word_f16(uint32_t w, uint32_t S2, uint32_t C0, uint32_t C1, uint32_t* o) {
    const uint32_t t = w >> 8;
    o[0] = hfma2_u32(ws_lop_and_xor(w, 0x000F000Fu, 0x64086408u), S2, C0);   // k0, k4
    o[1] = hfma2_u32(ws_lop_and_xor(w, 0x00F000F0u, 0x54805480u), S2, C1);   // k1, k5
    o[2] = hfma2_u32(ws_lop_and_xor(t, 0x000F000Fu, 0x64086408u), S2, C0);   // k2, k6
    o[3] = hfma2_u32(ws_lop_and_xor(t, 0x00F000F0u, 0x54805480u), S2, C1);   // k3, k7
}
// position of k inside one 256-k stage row of the fp16 activation copy (word order [0,4,1,5,2,6,3,7])
__device__ __forceinline__ int x16_pos(int k) {
    const int i = k & 7;
    return (k & ~7) | ((i & 3) << 1) | (i >> 2);
}
// exact bf16 path (same arithmetic as gemm_w4a16.cu): nibble at mantissa bit pos of 1.0f, one FMA
// with exactly representable addends, one cvt.rn.bf16x2.
__device__ __forceinline__ uint32_t ws_fma2_bf16x2(uint32_t e0, uint32_t e1, uint64_t s, uint64_t c) {
    uint64_t x, d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(x) : "r"(e0), "r"(e1));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(x), "l"(s), "l"(c));
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(d));
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}
__device__ __forceinline__ void dequant_word_bf16(uint32_t w, float sg, uint32_t* o) {
    const float s8 = sg * 32768.0f, c8 = -(sg * 32776.0f);
    const float s12 = sg * 2048.0f, c12 = -(sg * 2056.0f);
    const float s16 = sg * 128.0f, c16 = -(sg * 136.0f);
    const uint32_t wa = w << 8, wb = w >> 12;
    const uint32_t M8 = 0x00000F00u, M12 = 0x0000F000u, M16 = 0x000F0000u;
    const uint32_t X8 = 0x3F800800u, X12 = 0x3F808000u, X16 = 0x3F880000u;
    o[0] = ws_fma2_bf16x2(ws_lop_and_xor(wa, M8, X8), ws_lop_and_xor(wa, M12, X12), pack_f2(s8, s12), pack_f2(c8, c12));
    o[1] = ws_fma2_bf16x2(ws_lop_and_xor(wa, M16, X16), ws_lop_and_xor(w, M12, X12), pack_f2(s16, s12), pack_f2(c16, c12));
    o[2] = ws_fma2_bf16x2(ws_lop_and_xor(w, M16, X16), ws_lop_and_xor(wb, M8, X8), pack_f2(s16, s8), pack_f2(c16, c8));
    o[3] = ws_fma2_bf16x2(ws_lop_and_xor(wb, M12, X12), ws_lop_and_xor(wb, M16, X16), pack_f2(s12, s16), pack_f2(c12, c16));
}

__device__ __forceinline__ uint4 ws_lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "r"(addr));
    return v;
}
__device__ __forceinline__ uint32_t ws_lds32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

// Lean mbarrier wait for the dequantiser loop (no watchdog code in the hot loop; try_wait suspends in
// hardware; a pipeline bug is caught by the watchdogs of the other roles).
__device__ __forceinline__ void mbar_wait_lean(uint32_t bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {}
}

// Walks this CTA's unit list; every role runs an identical copy.
struct UnitIter {
    const int2* sched;
    int i, end;
    int l, tile, sb0, sb1;
    int2 pre;                 // the CTA's first unit, loaded at kernel entry
    bool first;
    __device__ __forceinline__ UnitIter(const WsParams& p, int2 cnt, int2 u0)
        : sched(p.sched + static_cast<size_t>(blockIdx.x) * p.max_units), i(0), end(cnt.x), pre(u0), first(true) {}
    __device__ __forceinline__ bool valid() const { return i < end; }
    __device__ __forceinline__ void locate(const WsParams&) {   // call when valid()
        const int2 e = i == 0 ? pre : __ldg(sched + i);
        l = e.x >> 16;
        tile = e.x & 0xFFFF;
        sb0 = 0;
        sb1 = e.y;
    }
    __device__ __forceinline__ void next() { ++i; first = false; }
};

template <bool AF16, bool PROF>
__global__ void __launch_bounds__(WS_THREADS, 1) w4a16_stream_kernel(const WsParams p) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    uint8_t* gbase = smem_raw + (base - raw);
    const uint32_t sP = base + WS_P_OFF, sX = base + WS_X_OFF, sS = base + WS_S_OFF;
    const uint32_t bars = base + WS_BAR_OFF;
    const uint32_t pfull0 = bars, pempty0 = pfull0 + 8 * WS_PS;
    const uint32_t xfull0 = pempty0 + 8 * WS_PS, xempty0 = xfull0 + 8 * WS_XS;
    const uint32_t afull0 = xempty0 + 8 * WS_XS, aempty0 = afull0 + 8 * WS_NA;
    const uint32_t tfull0 = aempty0 + 8 * WS_NA, tempty0 = tfull0 + 8 * WS_NTACC;
    const uint32_t tmem_slot = tempty0 + 8 * WS_NTACC;
    volatile uint32_t* tmem_slot_g =
        reinterpret_cast<volatile uint32_t*>(gbase + WS_BAR_OFF + WS_NBAR * 8);

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    // Fallback launch (exact bf16 operands): runs only if the fp16 launch before it left its domain.
    if (p.run_if) {
        pdl_wait_prior_grid();
        if (ld_acquire(p.run_if) == 0) return;
    }
    pdl_launch_dependents();

    // Start-up chain: the CTA's unit count / stage total and its first unit come from two independent
    // loads issued here, and the producers prefetch the first layer's tensor maps, all while the
    // barriers are initialised and tensor memory is allocated.
    const int2 sched_cnt = __ldg(p.sched_cnt + blockIdx.x);
    const int2 unit0 = __ldg(p.sched + static_cast<size_t>(blockIdx.x) * p.max_units);
    if (lane == 0 && sched_cnt.x > 0) {
        const WsLayer& L0 = p.layers[unit0.x >> 16];
        if (warp == WS_WPROD_WARP) { tma_prefetch_desc(&L0.tmP); tma_prefetch_desc(&L0.tmS); }
        if (warp == WS_XPROD_WARP) tma_prefetch_desc(&L0.tmX);
    }

    if (warp == WS_XPROD_WARP && lane == 0) {
        for (int s = 0; s < WS_PS; ++s) {
            mbar_init(pfull0 + 8 * s, 1);
            mbar_init(pempty0 + 8 * s, 4 * WS_G);     // every dequantiser warp reads every stage
        }
        for (int s = 0; s < WS_XS; ++s) {
            mbar_init(xfull0 + 8 * s, 1);
            mbar_init(xempty0 + 8 * s, 1);            // MMA commit
        }
        for (int a = 0; a < WS_NA; ++a) {
            mbar_init(afull0 + 8 * a, 4 * WS_G);      // every dequantiser warp fills its part of the slot
            mbar_init(aempty0 + 8 * a, 1);            // MMA commit
        }
        for (int a = 0; a < WS_NTACC; ++a) {
            mbar_init(tfull0 + 8 * a, 1);
            mbar_init(tempty0 + 8 * a, 4);
        }

        fence_mbar_init();
    }
    if (warp == WS_MMA_WARP) {
        tmem_alloc(tmem_slot, WS_TMEM_COLS);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_g;
    const long long t_start = clock64();
    unsigned long long gt_start = 0;
    if (PROF) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt_start));

    if (AF16 && p.n_conv > 0 && warp < WS_XPROD_WARP) {
        // bf16 -> fp16 of the external inputs (exact for 2^-14 <= |x| <= 65504, saturating above,
        // absolute error <= 2^-25 below); the producers and the MMA warp start streaming meanwhile.
        // Written in the stream layout: per 256-k stage WS_XLD fp16 = 256 x (k order of
        // dequant_word_f16) + 8 x (hi, lo) sums of the stage's 32-k groups (the zero-point operand).
        constexpr int CT = 32 * WS_XPROD_WARP;            // dequantiser + epilogue warps
        const int ctid = threadIdx.x;
        for (int cb = blockIdx.x * CT + (ctid & ~31); cb < p.conv_chunks; cb += gridDim.x * CT) {   // warp-uniform
            const int c = cb + lane;
            const bool ok = c < p.conv_chunks;       // chunk counts are multiples of 32: a warp never straddles two inputs
            float sum = 0.0f, amax = 0.0f;
            uint16_t* drow = nullptr;
            int kc = 0, seg = 0;
            if (ok) {
                int lo = 0, hi = p.n_conv - 1;         // segment of chunk c
                while (lo < hi) {
                    const int mid = (lo + hi + 1) >> 1;
                    if (__ldg(&p.conv[mid].chunk0) <= c) lo = mid; else hi = mid - 1;
                }
                seg = lo;
                const WsConv cv = p.conv[lo];
                const int ci = c - cv.chunk0;
                const int m = ci / cv.kc8;
                kc = ci - m * cv.kc8;
                const uint4 v = __ldg(cv.src + ci);
                {   // max |x| of the 8 bf16 values (non-negative floats order like their bit patterns)
                    const uint32_t w4[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                    for (int i = 0; i < 4; ++i)
                        amax = fmaxf(amax, fmaxf(fabsf(__uint_as_float(w4[i] << 16)), fabsf(__uint_as_float(w4[i] & 0xFFFF0000u))));
                }
                const uint32_t h01 = bf16x2_to_f16x2(v.x), h23 = bf16x2_to_f16x2(v.y);
                const uint32_t h45 = bf16x2_to_f16x2(v.z), h67 = bf16x2_to_f16x2(v.w);
                uint4 o;                               // pairs (k_i, k_{i+4})
                o.x = __byte_perm(h01, h45, 0x5410); o.y = __byte_perm(h01, h45, 0x7632);
                o.z = __byte_perm(h23, h67, 0x5410); o.w = __byte_perm(h23, h67, 0x7632);
                drow = cv.dst + static_cast<size_t>(m) * cv.ld16 + (kc >> 5) * WS_XLD;
                *reinterpret_cast<uint4*>(drow + (kc & 31) * 8) = o;
                const float2 f01 = __half22float2(*reinterpret_cast<const __half2*>(&h01));
                const float2 f23 = __half22float2(*reinterpret_cast<const __half2*>(&h23));
                const float2 f45 = __half22float2(*reinterpret_cast<const __half2*>(&h45));
                const float2 f67 = __half22float2(*reinterpret_cast<const __half2*>(&h67));
                sum = ((f01.x + f01.y) + (f23.x + f23.y)) + ((f45.x + f45.y) + (f67.x + f67.y));
            }
            sum += __shfl_xor_sync(0xffffffffu, sum, 1);     // 4 chunks = one 32-k group
            sum += __shfl_xor_sync(0xffffffffu, sum, 2);
            if (ok && (kc & 3) == 0) {
                const __half sh = __float2half_rn(fminf(fmaxf(sum, -WS_F16_MAX), WS_F16_MAX));
                const __half sl = __float2half_rn(sum - __half2float(sh));
                *reinterpret_cast<__half2*>(drow + 256 + 2 * ((kc >> 2) & 7)) = __halves2half2(sh, sl);
            }
            // domain of the fp16 operand: every |x| and every group sum within the fp16 range
            const unsigned mb = __reduce_max_sync(0xffffffffu, __float_as_uint(amax));
            const bool over = __any_sync(0xffffffffu, amax > WS_F16_MAX || fabsf(sum) > WS_F16_MAX);
            if (lane == 0 && ok) {
                atomicMax(p.inmax + seg, mb);
                if (over) atomicOr(p.flag, 1u);
            }
        }
        __threadfence();
        named_bar_sync(1, CT);
        if (ctid == 0) atomicAdd(p.done + p.n_layers, 1u);
    }

    if (warp == WS_XPROD_WARP) {
        // ------------------------------------------------------------ X producer
        if (AF16 && p.n_conv > 0) {
            if (lane == 0) {
                wait_counter(p.done + p.n_layers, gridDim.x);
                fence_proxy_async_all();
            }
            __syncwarp();
        }
        int stage = 0;
        uint32_t phase = 0;
        for (UnitIter it(p, sched_cnt, unit0); it.valid(); it.next()) {
            it.locate(p);
            const WsLayer& L = p.layers[it.l];
            if (L.dep >= 0 && !(PROF && (p.dbg & 128))) {       // chained layer: the producer layer must be complete
                if (lane == 0) {
                    wait_counter(p.done + L.dep, p.layers[L.dep].done_target);
                    fence_proxy_async_all();   // generic-proxy stores of other SMs -> this TMA read
                }
                __syncwarp();
            }
            if (AF16 && lane == 0) {
                // a whole input tensor far below the fp16 normal range: the subnormal grid (2^-24) would cost
                // relative precision -> flag the launch (an all-zero input is exact)
                const unsigned mb = ld_acquire(L.dep >= 0 ? p.outmax + L.dep : p.inmax + L.in_ext);
                if (mb != 0 && mb < __float_as_uint(WS_MIN_ABSMAX)) atomicOr(p.flag, 2u);
            }
            for (int sb = it.sb0; sb < it.sb1; ++sb) {
                mbar_wait(xempty0 + 8 * stage, phase ^ 1);
                if (elect_one()) {
                    constexpr int NSUB = AF16 ? WS_XSUB : 4;
                    mbar_arrive_expect_tx(xfull0 + 8 * stage, NSUB * WS_TT * 128);
#pragma unroll
                    for (int j = 0; j < NSUB; ++j)
                        tma_load_2d(sX + stage * WS_X_BYTES + j * (WS_TT * 128), &L.tmX,
                                    sb * (AF16 ? WS_XLD : WS_SBK) + j * 64, 0, xfull0 + 8 * stage);
                }
                __syncwarp();
                if (++stage == WS_XS) { stage = 0; phase ^= 1; }
            }
        }
        if (lane == 0) WS_STAMP(0);
    } else if (warp == WS_WPROD_WARP) {
        // ------------------------------------------------------------ weight producer (the HBM stream)
        const uint64_t pol_w = policy_evict_first();
        int stage = 0;
        uint32_t phase = 0;
        for (UnitIter it(p, sched_cnt, unit0); it.valid(); it.next()) {
            it.locate(p);
            const WsLayer& L = p.layers[it.l];
            const int n0 = it.tile * WS_ROWS;
            for (int sb = it.sb0; sb < it.sb1; ++sb) {
                mbar_wait(pempty0 + 8 * stage, phase ^ 1);
                if (elect_one()) {
                    mbar_arrive_expect_tx(pfull0 + 8 * stage, WS_P_BYTES + ((PROF && (p.dbg & 4)) ? 0 : WS_S_BYTES));
                    if (PROF && (p.dbg & 32)) tma_load_2d_hint(sP + stage * WS_P_BYTES, &L.tmP, 0, n0 * (L.K / 2) / 128 + sb * 128, pfull0 + 8 * stage, pol_w);
                    else
                    tma_load_2d_hint(sP + stage * WS_P_BYTES, &L.tmP, sb * 128, n0, pfull0 + 8 * stage, pol_w);
                    if (PROF && (p.dbg & 64)) tma_load_2d_hint(sS + stage * WS_S_BYTES, &L.tmS, 0, n0 * (L.K / 16) / 16 + sb * 128, pfull0 + 8 * stage, pol_w);
                    else
                    if (!(PROF && (p.dbg & 4))) tma_load_2d_hint(sS + stage * WS_S_BYTES, &L.tmS, sb * 8, n0, pfull0 + 8 * stage, pol_w);
                }
                __syncwarp();
                if (++stage == WS_PS) { stage = 0; phase ^= 1; }
            }
        }
        if (lane == 0) WS_STAMP(1);
    } else if (warp == WS_MMA_WARP) {
        // ------------------------------------------------------------ MMA issuer
        constexpr uint32_t idesc = make_idesc(1, AF16 ? 0u : 1u, AF16 ? 0u : 1u, WS_ROWS, WS_TT);
        const uint64_t desc_hi = make_smem_desc_sw128(0);
        int xs = 0, slot = 0, acc = 0;
        uint32_t xphase = 0, aphase = 0, acc_phase = 0;
        long long w_t = 0, w_x = 0, w_a = 0;
        for (UnitIter it(p, sched_cnt, unit0); it.valid(); it.next()) {
            it.locate(p);
            WS_TIMED(w_t, mbar_wait(tempty0 + 8 * acc, acc_phase ^ 1));
            tc_fence_after();
            const uint32_t d_tmem = tmem_base + WS_ACC_COL0 + acc * (WS_NACC * WS_TT);
            for (int sb = it.sb0; sb < it.sb1; ++sb) {
                WS_TIMED(w_x, mbar_wait(xfull0 + 8 * xs, xphase));
                WS_TIMED(w_a, mbar_wait(afull0 + 8 * slot, aphase));       // all 4 sub-blocks of the stage dequantised
                tc_fence_after();
                if (lane == 0 && it.first && sb == it.sb0) WS_STAMP(2);
                const uint32_t a_tmem = tmem_base + WS_A_COL0 + slot * WS_A_SLOT;
                const uint64_t b_desc = desc_hi | (((sX + xs * WS_X_BYTES) & 0x3FFFF) >> 4);
                if (elect_one()) {
#pragma unroll
                    for (int j = 0; j < 4; ++j)             // 64-k sub-tile of X: 4 KB apart
#pragma unroll
                        for (int k = 0; k < 4; ++k)
                            if (!(PROF && (p.dbg & 2)))
                                mma_f16_ts(d_tmem + (k % WS_NACC) * WS_TT, a_tmem + j * 32 + k * 8,
                                           b_desc + j * (WS_TT * 128 / 16) + 2 * k, idesc,
                                           (sb != it.sb0 || j * 4 + k >= WS_NACC) ? 1u : 0u);
                    // zero point: 16 more k with A = -8 sg of the stage's 8 groups (each twice) and
                    // B = (hi, lo) of the groups' activation sums
                    if (AF16 && !(PROF && (p.dbg & 2)))
                        mma_f16_ts(d_tmem, a_tmem + 128, b_desc + 4 * (WS_TT * 128 / 16), idesc, 1u);
                    tc_commit(aempty0 + 8 * slot);
                    tc_commit(xempty0 + 8 * xs);
                    if (sb == it.sb1 - 1) tc_commit(tfull0 + 8 * acc);
                }
                __syncwarp();
                if (++slot == WS_NA) { slot = 0; aphase ^= 1; }
                if (++xs == WS_XS) { xs = 0; xphase ^= 1; }
            }
            if (++acc == WS_NTACC) { acc = 0; acc_phase ^= 1; }
        }
        if (lane == 0) { WS_STAMP(3); if (PROF && p.prof) { p.prof[blockIdx.x * 16 + 9] = w_t; p.prof[blockIdx.x * 16 + 10] = w_x; p.prof[blockIdx.x * 16 + 11] = w_a; } }
    } else if (warp < WS_EPI_WARP0) {
        // ------------------------------------------------------------ dequantiser groups
        // The dequantisers do not care about unit boundaries: they see one sequence of `total` stages.
        // Software pipelined per warp: the packed bytes of stage s+1 are loaded before the arithmetic
        // of stage s, each half (32 k) goes to TMEM as soon as its 16 registers are ready, and the
        // "A slot full" signal of stage s is sent in the middle of stage s+1 (its stores have long
        // landed by then).  The loop is ISSUE bound (ncu: the 16 dequantiser warps own ~90% of the
        // SM's issued instructions), so it is unrolled by the weight-ring depth: every ring index,
        // barrier address and A-slot parity is a compile-time constant and the register rotation of
        // the software pipeline costs no moves.
        const int dw = warp - WS_DEQ_WARP0;
        const int g = dw >> 2;                    // group = 64-k sub-block of the stage
        const int q = dw & 3;                     // TMEM lane quarter (== warp % 4)
        const int r = q * 32 + lane;              // weight row inside the tile
        const uint32_t xr = r & 7;
        const uint32_t pa0 = sP + r * 128 + (((2 * g) ^ xr) << 4);        // 128-byte swizzle
        const uint32_t pa1 = sP + r * 128 + (((2 * g + 1) ^ xr) << 4);
        const uint32_t sa = sS + r * 16 + g * 4;
        const uint32_t a_base = tmem_base + WS_A_COL0 + g * 32 + (static_cast<uint32_t>(q * 32) << 16);
        const uint32_t z_base = tmem_base + WS_A_COL0 + 128 + g * 2 + (static_cast<uint32_t>(q * 32) << 16);
        const int total = sched_cnt.y;            // stages of this CTA
        uint4 pk0 = make_uint4(0, 0, 0, 0), pk1 = pk0;
        uint32_t sc2 = 0;
        if (total > 0) {
            mbar_wait(pfull0, 0);
            if (PROF && dw == 0 && lane == 0) WS_STAMP(4);
            sc2 = ws_lds32(sa);
            pk0 = ws_lds128(pa0);
            pk1 = ws_lds128(pa1);
        }
        uint32_t pphase = 0;                      // parity of the weight-ring pass of this round
        for (int s0 = 0; s0 < total; s0 += WS_PS) {
#pragma unroll
            for (int j = 0; j < WS_PS; ++j) {
                const int s = s0 + j;
                if (s < total) {                  // warp-uniform
                    const int slot = j % WS_NA;                              // compile-time after unrolling
                    const uint32_t a_par = static_cast<uint32_t>((j / WS_NA) & 1);
                    const int nj = (j + 1) % WS_PS;
                    // ---- start the loads of the next stage
                    uint4 nk0 = pk0, nk1 = pk1;
                    uint32_t nsc = sc2;
                    if (s + 1 < total) {
                        mbar_wait_lean(pfull0 + 8 * nj, nj == 0 ? pphase ^ 1u : pphase);
                        nsc = ws_lds32(sa + nj * WS_S_BYTES);
                        nk0 = ws_lds128(pa0 + nj * WS_P_BYTES);
                        nk1 = ws_lds128(pa1 + nj * WS_P_BYTES);
                    }
                    uint32_t o[16];
                    uint32_t z0 = 0, z1 = 0;      // (-8 sg, -8 sg) of the sub-block's two groups (AF16)
                    // ---- first half: k 0..31 of the sub-block
                    if (PROF && (p.dbg & 1)) {
#pragma unroll
                        for (int i = 0; i < 16; ++i) o[i] = pk0.x + i;
                    } else if (AF16) {
                        const __half2 sh = __half2half2(__ushort_as_half(static_cast<uint16_t>(sc2 & 0xFFFFu)));
                        const __half2 A = __hmul2(sh, __floats2half2_rn(-1024.0f, -1024.0f)), B = __hmul2(sh, __floats2half2_rn(-64.0f, -64.0f));
                        const __half2 Z = __hmul2(sh, __floats2half2_rn(-8.0f, -8.0f));
                        const uint32_t S2 = *reinterpret_cast<const uint32_t*>(&sh);
                        const uint32_t C0 = *reinterpret_cast<const uint32_t*>(&A), C1 = *reinterpret_cast<const uint32_t*>(&B);
                        z0 = *reinterpret_cast<const uint32_t*>(&Z);
                        dequant_word_f16(pk0.x, S2, C0, C1, o + 0);  dequant_word_f16(pk0.y, S2, C0, C1, o + 4);
                        dequant_word_f16(pk0.z, S2, C0, C1, o + 8);  dequant_word_f16(pk0.w, S2, C0, C1, o + 12);
                    } else {
                        const float sf = __half2float(__ushort_as_half(static_cast<uint16_t>(sc2 & 0xFFFFu)));
                        dequant_word_bf16(pk0.x, sf, o + 0);  dequant_word_bf16(pk0.y, sf, o + 4);
                        dequant_word_bf16(pk0.z, sf, o + 8);  dequant_word_bf16(pk0.w, sf, o + 12);
                    }
                    if (s > 0) {                  // publish the previous stage's sub-block
                        tmem_wait_st();
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(afull0 + 8 * ((slot + WS_NA - 1) % WS_NA));
                    }
                    mbar_wait_lean(aempty0 + 8 * slot, a_par ^ 1u);   // MMAs reading this slot retired
                    tc_fence_after();
                    tmem_st_32x32b_x16(a_base + slot * WS_A_SLOT, o);
                    // ---- second half: k 32..63
                    if (PROF && (p.dbg & 1)) {
#pragma unroll
                        for (int i = 0; i < 16; ++i) o[i] = pk1.x + i;
                    } else if (AF16) {
                        const __half2 sh = __half2half2(__ushort_as_half(static_cast<uint16_t>(sc2 >> 16)));
                        const __half2 A = __hmul2(sh, __floats2half2_rn(-1024.0f, -1024.0f)), B = __hmul2(sh, __floats2half2_rn(-64.0f, -64.0f));
                        const __half2 Z = __hmul2(sh, __floats2half2_rn(-8.0f, -8.0f));
                        const uint32_t S2 = *reinterpret_cast<const uint32_t*>(&sh);
                        const uint32_t C0 = *reinterpret_cast<const uint32_t*>(&A), C1 = *reinterpret_cast<const uint32_t*>(&B);
                        z1 = *reinterpret_cast<const uint32_t*>(&Z);
                        dequant_word_f16(pk1.x, S2, C0, C1, o + 0);  dequant_word_f16(pk1.y, S2, C0, C1, o + 4);
                        dequant_word_f16(pk1.z, S2, C0, C1, o + 8);  dequant_word_f16(pk1.w, S2, C0, C1, o + 12);
                    } else {
                        const float sf = __half2float(__ushort_as_half(static_cast<uint16_t>(sc2 >> 16)));
                        dequant_word_bf16(pk1.x, sf, o + 0);  dequant_word_bf16(pk1.y, sf, o + 4);
                        dequant_word_bf16(pk1.z, sf, o + 8);  dequant_word_bf16(pk1.w, sf, o + 12);
                    }
                    tmem_st_32x32b_x16(a_base + slot * WS_A_SLOT + 16, o);
                    if (AF16) tmem_st_32x32b_x2(z_base + slot * WS_A_SLOT, z0, z1);
                    __syncwarp();
                    if (lane == 0) mbar_arrive(pempty0 + 8 * j);   // this stage's packed bytes are consumed
                    pk0 = nk0; pk1 = nk1; sc2 = nsc;
                }
            }
            pphase ^= 1u;
        }
        if (total > 0) {
            tmem_wait_st();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(afull0 + 8 * ((total - 1) % WS_NA));
        }
        if (PROF && dw == 0 && lane == 0) WS_STAMP(5);
    } else if (warp < WS_XPROD_WARP) {
        // ------------------------------------------------------------ epilogue (warps 4..7)
        const int q = warp & 3;
        int acc = 0;
        uint32_t acc_phase = 0;
        for (UnitIter it(p, sched_cnt, unit0); it.valid(); it.next()) {
            it.locate(p);
            // layer fields into registers FIRST: the compiler must assume the output stores below may
            // alias the layer table and would otherwise re-load them from L2 after every store
            // (measured: 10k cycles per epilogue instead of a few hundred)
            const WsLayer* Lp = p.layers + it.l;
            const int N = __ldg(&Lp->N), M = p.M;
            const int act = __ldg(&Lp->act), out_t = __ldg(&Lp->out_t), notify = __ldg(&Lp->notify);
            const __nv_bfloat16* bias = static_cast<const __nv_bfloat16*>(
                reinterpret_cast<const void*>(__ldg(reinterpret_cast<const unsigned long long*>(&Lp->bias))));
            void* const Yp = reinterpret_cast<void*>(__ldg(reinterpret_cast<const unsigned long long*>(&Lp->Y)));
            void* const Y16p = (PROF && (p.dbg & 256)) ? nullptr : reinterpret_cast<void*>(__ldg(reinterpret_cast<const unsigned long long*>(&Lp->Y16)));
            const int n = it.tile * WS_ROWS + q * 32 + lane;
            const bool n_ok = n < N;
            const float bv = bias && n_ok ? __bfloat162float(bias[n]) : 0.0f;
            mbar_wait(tfull0 + 8 * acc, acc_phase);
            tc_fence_after();
            if (q == 0 && lane == 0 && it.first) WS_STAMP(6);
            uint32_t v[32];
            {
                const uint32_t t_addr = tmem_base + WS_ACC_COL0 + acc * (WS_NACC * WS_TT) + (static_cast<uint32_t>(q * 32) << 16);
                tmem_ld_32x32b_x32(t_addr, v);
                tmem_wait_ld();
#pragma unroll
                for (int a = 1; a < WS_NACC; ++a) {          // fixed order: deterministic
                    uint32_t w[32];
                    tmem_ld_32x32b_x32(t_addr + a * WS_TT, w);
                    tmem_wait_ld();
#pragma unroll
                    for (int t = 0; t < WS_TT; ++t) v[t] = __float_as_uint(__uint_as_float(v[t]) + __uint_as_float(w[t]));
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty0 + 8 * acc);             // accumulator is in registers
            if (++acc == WS_NTACC) { acc = 0; acc_phase ^= 1; }

            const bool gelu = act == ARIA_ACT_GELU_ERF;
            if (out_t == ARIA_F32) {
                if (n_ok) {
                    float* Y = static_cast<float*>(Yp) + n;
#pragma unroll
                    for (int t = 0; t < WS_TT; ++t) {
                        if (t < M) {
                            float y = __uint_as_float(v[t]) + bv;
                            if (gelu) y = gelu_erf(y);
                            Y[static_cast<size_t>(t) * N] = y;           // a warp writes 32 consecutive n
                        }
                    }
                }
            } else if (AF16 && Y16p) {
                // A later layer reads this output (its K = this N, a multiple of 256): besides the bf16
                // result write what that layer's MMA reads -- the bf16 value as fp16, in the stream
                // layout, and the (hi, lo) sum of this warp's 32 channels = one 32-k group of that layer.
                __nv_bfloat16* Y = static_cast<__nv_bfloat16*>(Yp) + n;
                const int n0 = it.tile * WS_ROWS + q * 32;                // warp-uniform; N % 256 == 0 here
                const int ld16 = (N >> 8) * WS_XLD;
                __half* Yrow = static_cast<__half*>(Y16p) + (n0 >> 8) * WS_XLD;
                const int xpos = x16_pos(n & 255), spos = 256 + 2 * ((n0 >> 5) & 7);
                float hs[WS_TT];                                          // the bf16 outputs, as fp32
                float amax = 0.0f;
#pragma unroll
                for (int t = 0; t < WS_TT; t += 2) {
                    float y0 = __uint_as_float(v[t]) + bv, y1 = __uint_as_float(v[t + 1]) + bv;
                    if (gelu) gelu_erf2(y0, y1);
                    uint32_t yb2, yh2;
                    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(yb2) : "f"(y1), "f"(y0));
                    hs[t] = __uint_as_float(yb2 << 16);
                    hs[t + 1] = __uint_as_float(yb2 & 0xFFFF0000u);
                    // what the next layer's MMA reads: the bf16 value as fp16 (exact for 2^-14 <= |y| <= 65504)
                    asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(yh2) : "f"(hs[t + 1]), "f"(hs[t]));
                    if (t < M) {                                          // M is warp-uniform
                        reinterpret_cast<uint16_t*>(Y)[static_cast<size_t>(t) * N] = static_cast<uint16_t>(yb2);
                        reinterpret_cast<uint16_t*>(Yrow)[static_cast<size_t>(t) * ld16 + xpos] = static_cast<uint16_t>(yh2);
                        amax = fmaxf(amax, fabsf(hs[t]));
                    }
                    if (t + 1 < M) {
                        amax = fmaxf(amax, fabsf(hs[t + 1]));
                        reinterpret_cast<uint16_t*>(Y)[static_cast<size_t>(t + 1) * N] = static_cast<uint16_t>(yb2 >> 16);
                        reinterpret_cast<uint16_t*>(Yrow)[static_cast<size_t>(t + 1) * ld16 + xpos] = static_cast<uint16_t>(yh2 >> 16);
                    }
                }
                // sums over the warp's 32 channels for all 32 tokens by recursive halving: 31 independent
                // shuffles instead of 32 dependent 5-step butterflies; lane L ends with token L's sum
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) {
                    const bool up = (lane & d) != 0;
#pragma unroll
                    for (int i = 0; i < d; ++i) {
                        const float keep = up ? hs[i + d] : hs[i];
                        const float give = up ? hs[i] : hs[i + d];
                        hs[i] = keep + __shfl_xor_sync(0xffffffffu, give, d);
                    }
                }
                if (lane < M) {
                    const __half sh = __float2half_rn(fminf(fmaxf(hs[0], -WS_F16_MAX), WS_F16_MAX));
                    const __half sl = __float2half_rn(hs[0] - __half2float(sh));
                    *reinterpret_cast<__half2*>(Yrow + static_cast<size_t>(lane) * ld16 + spos) = __halves2half2(sh, sl);
                }
                {   // domain of the consumer's fp16 operand (see the conversion pre-pass)
                    const unsigned mb = __reduce_max_sync(0xffffffffu, __float_as_uint(amax));
                    const bool over = __any_sync(0xffffffffu, amax > WS_F16_MAX || (lane < M && fabsf(hs[0]) > WS_F16_MAX));
                    if (lane == 0) {
                        atomicMax(p.outmax + it.l, mb);
                        if (over) atomicOr(p.flag, 1u);
                    }
                }
            } else if (n_ok) {
                uint16_t* Y = static_cast<uint16_t*>(Yp) + n;
#pragma unroll
                for (int t = 0; t < WS_TT; t += 2) {
                    if (t < M) {
                        float y0 = __uint_as_float(v[t]) + bv, y1 = __uint_as_float(v[t + 1]) + bv;
                        if (gelu) gelu_erf2(y0, y1);
                        uint32_t yb2;
                        asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(yb2) : "f"(y1), "f"(y0));
                        Y[static_cast<size_t>(t) * N] = static_cast<uint16_t>(yb2);
                        if (t + 1 < M) Y[static_cast<size_t>(t + 1) * N] = static_cast<uint16_t>(yb2 >> 16);
                    }
                }
            }
            if (notify) {                   // a later layer reads this output: publish the quarter-tile
                __threadfence();
                __syncwarp();
                if (lane == 0) atomicAdd(p.done + it.l, 1u);
            }
            if (q == 0 && lane == 0 && it.first) WS_STAMP(7);
        }
        if (q == 0 && lane == 0) {
            WS_STAMP(8);
            if (PROF && p.prof) {      // slot 15: the same interval in ns (globaltimer) -> SM clock of this run
                unsigned long long gt;
                asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));
                p.prof[blockIdx.x * 16 + 15] = static_cast<long long>(gt - gt_start);
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == WS_MMA_WARP) {
        tc_fence_after();
        tmem_dealloc(tmem_base, WS_TMEM_COLS);
    }
}

}  // namespace aria

// ------------------------------------------------------------------------------------------------
// Host side: pre-encoded tensor maps, the unit schedule and the scratch of one layer list.
namespace aria {

struct WsPlan {
    bool a_f16 = true;
    WsPlan* fallback = nullptr;     // a_f16 plans: the same list with exact bf16 operands, run if the flag is set
    bool owns_done = true;
    WsLayer* d_layers = nullptr;
    int2* d_sched = nullptr;        // dense unit lists + per-CTA counts
    unsigned* d_done = nullptr;
    size_t done_bytes = 0;
    WsConv* d_conv = nullptr;
    void* d_x16 = nullptr;          // fp16 copies of external inputs and of chained outputs
    WsParams params{};
    int grid = 0;
};

void ws_plan_destroy(WsPlan* p) {
    if (!p) return;
    ws_plan_destroy(p->fallback);
    cudaFree(p->d_layers);
    cudaFree(p->d_sched);
    if (p->owns_done) cudaFree(p->d_done);
    cudaFree(p->d_conv);
    cudaFree(p->d_x16);
    delete p;
}

static bool overlaps(const void* a, size_t an, const void* b, size_t bn) {
    const uintptr_t a0 = reinterpret_cast<uintptr_t>(a), b0 = reinterpret_cast<uintptr_t>(b);
    return a0 < b0 + bn && b0 < a0 + an;
}

// The stream kernel runs layers concurrently where the list allows it, so it is used only when
// running them in array order cannot be told apart: bf16 I/O, M <= 32, K % 256 == 0 (16-byte pitch of
// the scale tensor map), no output buffer that overlaps another layer's output or an EARLIER layer's
// input, and a later layer's input that touches an earlier layer's output must BE that output (same
// address, K == that layer's N): the chained case, tracked by one completion counter per layer.  An
// input that only partly overlaps an earlier output, or spans two of them, takes the per-layer path.
bool ws_eligible(const aria_layer* layers, int n_layers, int M, int mode, int io) {
    if (mode != ARIA_W4A16 || io != ARIA_BF16 || M > WS_TT) return false;
    if (dbg_env("ARIA_NO_STREAM")) return false;
    for (int i = 0; i < n_layers; ++i) {
        if (layers[i].K % WS_SBK != 0) return false;
        const size_t ob = static_cast<size_t>(M) * layers[i].N * 2;
        const void* in = layers[i].in ? layers[i].in : (i > 0 ? layers[i - 1].out : nullptr);
        for (int j = 0; j < n_layers; ++j) {
            if (j == i) continue;
            if (overlaps(layers[i].out, ob, layers[j].out, static_cast<size_t>(M) * layers[j].N * 2)) return false;
            if (j < i && layers[j].in &&
                overlaps(layers[i].out, ob, layers[j].in, static_cast<size_t>(M) * layers[j].K * 2))
                return false;
            if (j < i && in &&
                overlaps(in, static_cast<size_t>(M) * layers[i].K * 2, layers[j].out, static_cast<size_t>(M) * layers[j].N * 2) &&
                !(in == layers[j].out && layers[j].N == layers[i].K))
                return false;
        }
    }
    return true;
}

// max over the fp16 magnitudes of a scale tensor (bit patterns order like the values; NaN / inf sort last)
__global__ void ws_scale_max_kernel(const uint16_t* __restrict__ sg, size_t n, unsigned* out) {
    unsigned m = 0;
    for (size_t i = static_cast<size_t>(blockIdx.x) * blockDim.x + threadIdx.x; i < n; i += static_cast<size_t>(gridDim.x) * blockDim.x)
        m = max(m, static_cast<unsigned>(sg[i] & 0x7FFFu));
    m = __reduce_max_sync(0xffffffffu, m);
    if ((threadIdx.x & 31) == 0) atomicMax(out, m);
}

// force_bf16 / ext_done: used by the recursive creation of a plan's bf16 fallback (its counters live in
// the primary plan's buffer so that one memset arms both launches).
static int ws_plan_create_impl(const aria_layer* layers, int n_layers, int M, int io, bool force_bf16,
                               unsigned* ext_done, WsPlan** out) {
    *out = nullptr;
    WsPlan* plan = new (std::nothrow) WsPlan;
    if (!plan) return ARIA_ERR_CUDA;
    const int sms = num_sms();
    if (sms <= 0) { ws_plan_destroy(plan); return ARIA_ERR_CUDA; }
    // Operand format.  fp16 (see the header comment) needs 1024 sg <= 65504 for every group scale, which is
    // a property of the weights: scan them once (plan creation may synchronise).  Activations are checked on
    // the device in every launch (flag + bf16 fallback launch).
    plan->a_f16 = !force_bf16;
    if (const char* e = dbg_env("ARIA_W4_F16A")) plan->a_f16 = plan->a_f16 && e[0] != '0';   // debug builds only
    if (plan->a_f16) {
        unsigned* d_max = nullptr;
        unsigned h_max = 0;
        bool ok = cudaMalloc(&d_max, sizeof(unsigned)) == cudaSuccess && cudaMemset(d_max, 0, sizeof(unsigned)) == cudaSuccess;
        for (int i = 0; ok && i < n_layers; ++i) {
            const size_t n = static_cast<size_t>(layers[i].N) * (layers[i].K / 32);
            ws_scale_max_kernel<<<2 * sms, 256>>>(static_cast<const uint16_t*>(layers[i].w_scale), n, d_max);
            ok = cudaGetLastError() == cudaSuccess;
        }
        ok = ok && cudaMemcpy(&h_max, d_max, sizeof(unsigned), cudaMemcpyDeviceToHost) == cudaSuccess;
        cudaFree(d_max);
        if (!ok) { ws_plan_destroy(plan); return ARIA_ERR_CUDA; }
        if (h_max > 0x53FFu) plan->a_f16 = false;      // sg > 63.96875 (or inf / NaN): 1024 sg overflows fp16
    }
    std::vector<WsLayer> h(n_layers);
    int total_units = 0;
    // pass 1: shapes, dependencies; fp16 scratch layout (AF16)
    std::vector<const void*> ext_src;          // distinct external inputs
    std::vector<size_t> ext_elems, ext_off;
    std::vector<size_t> y16_off(n_layers, 0);
    std::vector<int> in_ext(n_layers, -1);
    size_t x16_elems = 0;
    for (int i = 0; i < n_layers; ++i) {
        const aria_layer& L = layers[i];
        WsLayer& w = h[i];
        memset(&w, 0, sizeof(w));
        const void* in = L.in ? L.in : layers[i - 1].out;
        w.bias = L.bias; w.Y = L.out; w.N = L.N; w.K = L.K;
        w.num_n = (L.N + WS_ROWS - 1) / WS_ROWS;
        w.num_sb = L.K / WS_SBK;
        w.act = L.act; w.out_t = io;
        // dependency: an input that overlaps an earlier layer's output waits for that layer
        w.dep = -1;
        for (int j = i - 1; j >= 0; --j)
            if (overlaps(in, static_cast<size_t>(M) * L.K * 2, layers[j].out, static_cast<size_t>(M) * layers[j].N * 2)) {
                w.dep = j;
                break;
            }
        w.in_ext = -1;
        if (w.dep >= 0) {
            // ws_eligible: the input IS the producer's output, so the fp16 copy has the right geometry
            h[w.dep].notify = 1;
        } else {
            size_t e = 0;
            while (e < ext_src.size() && !(ext_src[e] == in && ext_elems[e] == static_cast<size_t>(M) * L.K)) ++e;
            if (e == ext_src.size()) { ext_src.push_back(in); ext_elems.push_back(static_cast<size_t>(M) * L.K); }
            in_ext[i] = static_cast<int>(e);
            w.in_ext = static_cast<int>(e);
        }
        w.done_target = static_cast<unsigned>(w.num_n * 4);
        total_units += w.num_n;
        if (w.num_n > 0xFFFF || n_layers > 0x7FFF || (static_cast<size_t>(M) * L.K) % 8 != 0) { ws_plan_destroy(plan); return ARIA_ERR_SHAPE; }
    }
    std::vector<WsConv> conv;
    if (plan->a_f16) {
        // fp16 copies in the stream layout: [M, K / 256 * WS_XLD] per distinct external input and per
        // chained output (the pad columns are never read by an MMA; zeroed once for tidiness)
        auto x16_size = [&](size_t K) { return (static_cast<size_t>(M) * (K / WS_SBK) * WS_XLD + 127) / 128 * 128; };
        for (size_t e = 0; e < ext_src.size(); ++e) { ext_off.push_back(x16_elems); x16_elems += x16_size(ext_elems[e] / M); }
        for (int i = 0; i < n_layers; ++i)
            if (h[i].notify) { y16_off[i] = x16_elems; x16_elems += x16_size(layers[i].N); }
        if (cudaMalloc(&plan->d_x16, x16_elems * 2 + 256) != cudaSuccess ||
            cudaMemset(plan->d_x16, 0, x16_elems * 2 + 256) != cudaSuccess) { ws_plan_destroy(plan); return ARIA_ERR_CUDA; }
        int chunk0 = 0;
        for (size_t e = 0; e < ext_src.size(); ++e) {
            WsConv c;
            const size_t K = ext_elems[e] / M;
            c.src = static_cast<const uint4*>(ext_src[e]);
            c.dst = static_cast<uint16_t*>(plan->d_x16) + ext_off[e];
            c.chunk0 = chunk0; c.chunks = static_cast<int>(ext_elems[e] / 8);
            c.kc8 = static_cast<int>(K / 8); c.ld16 = static_cast<int>(K / WS_SBK * WS_XLD);
            chunk0 += c.chunks;
            conv.push_back(c);
        }
        plan->params.conv_chunks = chunk0;
    }
    // pass 2: tensor maps
    for (int i = 0; i < n_layers; ++i) {
        const aria_layer& L = layers[i];
        WsLayer& w = h[i];
        const void* in = L.in ? L.in : layers[i - 1].out;
        if (plan->a_f16) {
            uint16_t* x16 = static_cast<uint16_t*>(plan->d_x16);
            in = w.dep >= 0 ? x16 + y16_off[w.dep] : x16 + ext_off[in_ext[i]];
            if (w.notify) w.Y16 = x16 + y16_off[i];
        }
        const int dbg_ = dbg_env("ARIA_WS_DBG") ? atoi(dbg_env("ARIA_WS_DBG")) : 0;
        if (((dbg_ & 32) ? make_tmap_2d(&w.tmP, L.wq, 1, static_cast<uint64_t>(L.N) * (L.K / 2) / 128, 128, WS_ROWS, 128, 128)
                         : make_tmap_2d(&w.tmP, L.wq, 1, L.N, L.K / 2, WS_ROWS, 128, 128)) != ARIA_OK ||
            ((dbg_ & 64) ? make_tmap_2d(&w.tmS, L.w_scale, 2, static_cast<uint64_t>(L.N) * (L.K / 32) / 8, 8, WS_ROWS, 8, 0)
                         : make_tmap_2d(&w.tmS, L.w_scale, 2, L.N, L.K / 32, WS_ROWS, 8, 0)) != ARIA_OK ||
            make_tmap_2d(&w.tmX, in, 2, M, plan->a_f16 ? L.K / WS_SBK * WS_XLD : L.K, WS_TT, 64, 128) != ARIA_OK) {
            ws_plan_destroy(plan);
            return ARIA_ERR_CUDA;
        }
    }
    // Schedule.  Units are dealt in ONE global order, each to the CTA with the least work so far, so
    // all CTAs stream the same number of stages.  The order is the array order, except that a layer
    // whose input is an earlier layer's output is held back until every CTA has been given ~GAP
    // producer-unit durations of other work since its producer: by then the producer's last tile has
    // been stored and the consumer's units do not stall the weight ring (measured on config C5's
    // wiring: dependents right behind their producer cost +30% -- CTAs drift apart by ~15% -- while
    // "dependents last" runs at the rate of a list without dependencies).  It stays a topological
    // order and every CTA walks its units in that order, so a dependency always points to a unit
    // that is earlier in some CTA's list: no deadlock.  Layers that may run concurrently write
    // disjoint buffers (ws_eligible), so results equal array order.
    const int grid = total_units < sms ? total_units : sms;
    std::vector<int> order;
    {
        const char* eg = dbg_env("ARIA_WS_GAP");
        const double gap_units = eg ? atof(eg) : 32.0;      // in producer-unit durations
        std::vector<char> placed(n_layers, 0);
        std::vector<double> placed_at(n_layers, 0.0);
        double cum = 0.0;                                   // work per CTA dealt so far
        int n_placed = 0;
        while (n_placed < n_layers) {
            int pick = -1, fallback = -1;
            for (int i = 0; i < n_layers && pick < 0; ++i) {
                if (placed[i]) continue;
                const int d = h[i].dep;
                if (d < 0) { pick = i; break; }
                if (!placed[d]) continue;
                if (fallback < 0) fallback = i;
                if (cum - placed_at[d] >= gap_units * (2 * h[d].num_sb + 1)) pick = i;
            }
            if (pick < 0) pick = fallback;                  // nothing independent left: take the stall
            placed[pick] = 1;
            cum += static_cast<double>(h[pick].num_n) * (2 * h[pick].num_sb + 1) / grid;
            placed_at[pick] = cum;
            order.push_back(pick);
            ++n_placed;
        }
    }
    // cost of a unit in quarter stages: its stages, ~1/4 stage of accumulator hand-off, and the issue
    // slots a GELU / fp16-copy epilogue takes from the dequantisers of its SM
    const char* ec = dbg_env("ARIA_WS_EPI_COST");
    const int epi_cost = ec ? atoi(ec) : 1;
    auto unit_cost = [&](const WsLayer& w) {
        return 4 * w.num_sb + 1 + ((w.act == ARIA_ACT_GELU_ERF ? 1 : 0) + (w.notify ? 1 : 0)) * epi_cost;
    };
    std::vector<std::vector<int>> lists(grid);
    std::vector<long> load(grid, 0);
    std::vector<int> totals(grid, 0);
    for (int i : order)
        for (int t = 0; t < h[i].num_n; ++t) {
            int best = 0;
            for (int c = 1; c < grid; ++c)
                if (load[c] < load[best]) best = c;
            lists[best].push_back((i << 16) | t);
            load[best] += unit_cost(h[i]);
            totals[best] += h[i].num_sb;
        }
    size_t max_units = 1;
    for (int c = 0; c < grid; ++c) max_units = lists[c].size() > max_units ? lists[c].size() : max_units;
    std::vector<int2> sched(static_cast<size_t>(grid) * max_units, make_int2(0, 0));
    std::vector<int2> cnt(grid);
    for (int c = 0; c < grid; ++c) {
        for (size_t i = 0; i < lists[c].size(); ++i)
            sched[c * max_units + i] = make_int2(lists[c][i], h[lists[c][i] >> 16].num_sb);
        cnt[c] = make_int2(static_cast<int>(lists[c].size()), totals[c]);
    }
    const size_t sched_n = sched.size();
    sched.insert(sched.end(), cnt.begin(), cnt.end());
    // armed words, zeroed by ONE memset per step: [n_layers done][1 conversions done][1 flag][n_ext inmax]
    // [n_layers outmax], then the same for the bf16 fallback plan
    const size_t words = 2 * static_cast<size_t>(n_layers) + 2 + ext_src.size();
    const size_t words_fb = words;
    if (ext_done) {
        plan->d_done = ext_done;
        plan->owns_done = false;
        plan->done_bytes = 0;
    } else {
        plan->done_bytes = (words + (plan->a_f16 ? words_fb : 0)) * sizeof(unsigned);
        if (cudaMalloc(&plan->d_done, plan->done_bytes) != cudaSuccess) { ws_plan_destroy(plan); return ARIA_ERR_CUDA; }
    }
    if (cudaMalloc(&plan->d_layers, h.size() * sizeof(WsLayer)) != cudaSuccess ||
        cudaMalloc(&plan->d_sched, sched.size() * sizeof(int2)) != cudaSuccess ||
        cudaMemcpy(plan->d_layers, h.data(), h.size() * sizeof(WsLayer), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(plan->d_sched, sched.data(), sched.size() * sizeof(int2), cudaMemcpyHostToDevice) != cudaSuccess ||
        (!conv.empty() && (cudaMalloc(&plan->d_conv, conv.size() * sizeof(WsConv)) != cudaSuccess ||
                           cudaMemcpy(plan->d_conv, conv.data(), conv.size() * sizeof(WsConv), cudaMemcpyHostToDevice) != cudaSuccess))) {
        ws_plan_destroy(plan);
        return ARIA_ERR_CUDA;
    }
    plan->params.layers = plan->d_layers;
    plan->params.sched = plan->d_sched;
    plan->params.sched_cnt = plan->d_sched + sched_n;
    plan->params.max_units = static_cast<int>(max_units);
    plan->params.done = plan->d_done;
    plan->params.flag = plan->d_done + n_layers + 1;
    plan->params.inmax = plan->d_done + n_layers + 2;
    plan->params.outmax = plan->d_done + n_layers + 2 + ext_src.size();
    plan->params.run_if = nullptr;
    plan->params.conv = plan->d_conv;
    plan->params.n_conv = static_cast<int>(conv.size());
    plan->params.n_layers = n_layers;
    plan->params.M = M;
#ifdef ARIA_DEBUG
    plan->params.prof = g_ws_prof;
#else
    plan->params.prof = nullptr;
#endif
    plan->params.dbg = dbg_env("ARIA_WS_DBG") ? atoi(dbg_env("ARIA_WS_DBG")) : 0;
    plan->grid = grid;
    if (plan->a_f16) {   // the exact bf16 plan of the same list, run when a launch leaves the fp16 domain
        const int rc = ws_plan_create_impl(layers, n_layers, M, io, true, plan->d_done + words, &plan->fallback);
        if (rc != ARIA_OK) { ws_plan_destroy(plan); return rc; }
        plan->fallback->params.run_if = plan->params.flag;
    }
    *out = plan;
    return ARIA_OK;
}

int ws_plan_create(const aria_layer* layers, int n_layers, int M, int io, WsPlan** out) {
    return ws_plan_create_impl(layers, n_layers, M, io, false, nullptr, out);
}

int ws_plan_kind(const WsPlan* plan) { return plan->a_f16 ? 1 : 2; }

int ws_plan_fallback_fired(const WsPlan* plan, int* fired) {
    *fired = 0;
    if (!plan->a_f16) return ARIA_OK;
    unsigned f = 0;
    if (cudaMemcpy(&f, plan->params.flag, sizeof(unsigned), cudaMemcpyDeviceToHost) != cudaSuccess) return ARIA_ERR_CUDA;
    *fired = static_cast<int>(f);
    return ARIA_OK;
}

// The kernel's CTAs wait on one another (completion counters), so the whole grid must be co-resident:
// a COOPERATIVE launch, which is either fully resident or not started (and fails cleanly when the grid
// can never fit), instead of deadlocking on a CTA that has no SM, e.g. because another tenant's kernel
// holds SMs.  This holds for BOTH launches of a plan: the bf16 fallback runs the same cross-CTA waits when
// the fp16 launch left its domain, so it is cooperative too and follows the fp16 launch in plain stream
// order (it is not a programmatic dependent: its griddepcontrol.wait is then a no-op, and the flag it
// reads is complete when it starts).
template <bool AF16, bool PROF>
static int ws_launch(const WsPlan* plan, cudaStream_t st) {
    static std::atomic<uint64_t> attr_done{0};
    auto kern = w4a16_stream_kernel<AF16, PROF>;
    if (!ensure_dyn_smem(kern, WS_SMEM_BYTES, attr_done)) return ARIA_ERR_CUDA;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(plan->grid);
    cfg.blockDim = dim3(WS_THREADS);
    cfg.dynamicSmemBytes = WS_SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeCooperative;
    at[0].val.cooperative = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, plan->params) == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
}

static int ws_run_one(const WsPlan* plan, cudaStream_t st) {
#ifdef ARIA_DEBUG
    const bool prof = plan->params.prof != nullptr || (plan->params.dbg & 127) != 0;   // instrumented kernel
    if (prof) return plan->a_f16 ? ws_launch<true, true>(plan, st) : ws_launch<false, true>(plan, st);
#endif
    return plan->a_f16 ? ws_launch<true, false>(plan, st) : ws_launch<false, false>(plan, st);
}

// One step = a memset of the counters and flags, the stream kernel and, for fp16-operand plans, the
// bf16 fallback kernel (which exits at once unless the first launch raised its domain flag).
int ws_plan_run(const WsPlan* plan, cudaStream_t st) {
    if (cudaMemsetAsync(plan->d_done, 0, plan->done_bytes, st) != cudaSuccess) return ARIA_ERR_CUDA;
    int rc = ws_run_one(plan, st);
    if (rc == ARIA_OK && plan->fallback) rc = ws_run_one(plan->fallback, st);
    return rc;
}

}  // namespace aria
