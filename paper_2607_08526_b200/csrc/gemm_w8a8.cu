// gemm_w8a8.cu -- S2 + S3: int8 x int8 GEMM on tcgen05 (kind::i8, int32 accumulators in TMEM) with
// the per-token x per-channel rescale + bias (+ GELU) epilogue fused in.
//
// Persistent, warp-specialised, one CTA per SM:
//   warp 0      TMA producer: Xq tile [128 x 128 B] and Wq tile [BN x 128 B] per k-block into a
//               STAGES-deep shared-memory ring (128-byte swizzle), completion on `full` mbarriers.
//   warp 1      MMA issuer (one thread): 4 x tcgen05.mma (K = 32 each) per k-block into one of two
//               TMEM accumulators [128 lanes x BN columns]; tcgen05.commit frees the ring slot and,
//               after the last k-block, signals `tmem_full`.
//   warps 2..9  epilogue (two warps per TMEM lane quarter): tcgen05.ld 32 lanes x 32 columns ->
//               registers -> x sx[m] x sw[n] + b[n] (scales/bias staged in smem per tile) -> GELU ->
//               cast -> 64-byte-swizzled smem block -> TMA store.  Runs on accumulator `a` while the
//               MMA warp fills accumulator `a^1`.
// Tails: TMA zero-fills rows >= M / >= N and bytes >= K on load (zero codes add nothing) and clips
// them on store.
#include "internal.cuh"

namespace aria {

constexpr int W8_BM = 128;        // MMA M (TMEM lanes)
constexpr int W8_BK = 128;        // bytes (= int8 elements) per k-block: one 128-byte swizzle row
constexpr int W8_UMMA_K = 32;     // K per tcgen05.mma for 8-bit operands
constexpr int W8_EPI_WARPS = 8;   // two warps per TMEM lane quarter, interleaved over column chunks
constexpr int W8_THREADS = 64 + 32 * W8_EPI_WARPS;
constexpr int W8_STG_BYTES = 2048;  // per-warp output staging: 32 rows x 64 bytes (64-byte swizzle)

// CTAS = 1: one CTA computes a 128 x BN tile.  CTAS = 2: a CTA PAIR (cluster of 2, tcgen05 cta_group::2)
// computes a 256 x BN tile; each CTA stages its own 128 rows of A and only HALF of the B tile, which
// halves the shared-memory traffic per MAC (TMA writes + MMA operand reads share 128 B/clk per SM).
template <int BN, int CTAS>
struct W8Cfg {
    static constexpr int A_BYTES = W8_BM * W8_BK;
    static constexpr int B_ROWS = BN / CTAS;                   // B rows staged by one CTA
    static constexpr int B_BYTES = B_ROWS * W8_BK;
    static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
    static constexpr int RING_BUDGET = 227 * 1024 - 1024 - 256 - W8_EPI_WARPS * W8_STG_BYTES - 2 * BN * 4;
    static constexpr int STAGES = RING_BUDGET / STAGE_BYTES > 8 ? 8 : RING_BUDGET / STAGE_BYTES;
    static constexpr int ACC_STRIDE = BN <= 32 ? 32 : BN <= 64 ? 64 : BN <= 128 ? 128 : 256;
    static constexpr int TMEM_COLS = 2 * ACC_STRIDE < 32 ? 32 : 2 * ACC_STRIDE;
    static constexpr int RING_BYTES = STAGES * STAGE_BYTES;
    static constexpr int STG_OFF = RING_BYTES;                               // [8][2 KB] staging
    static constexpr int SWB_OFF = STG_OFF + W8_EPI_WARPS * W8_STG_BYTES;    // float sw[BN], bias[BN]
    static constexpr int BAR_OFF = SWB_OFF + 2 * BN * 4;
    static constexpr int BAR_BYTES = (2 * STAGES + 4) * 8 + 16;
    static constexpr int SMEM_BYTES = BAR_OFF + BAR_BYTES + 1024;            // + alignment slack
    static_assert(BN % 32 == 0 && BN >= 32 && BN <= 256, "BN");
    static_assert(B_BYTES % 1024 == 0, "B tile must keep 1024-byte alignment");
    static_assert(SMEM_BYTES <= 227 * 1024, "shared memory");
};

struct W8Params {
    const float* sx;
    const float* sw;
    const void* bias;
    int bias_t, act;
    int M, N, K;
    long long* prof;   // debug: per-CTA role timestamps (clock64), or nullptr
};

static long long* g_w8_prof = nullptr;
void w8_set_profile_buffer(long long* p) { g_w8_prof = p; }
__device__ __forceinline__ void w8_stamp(const W8Params& p, int slot, long long t0) {
    if (p.prof) p.prof[blockIdx.x * 16 + slot] = clock64() - t0;
}

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
    __nv_bfloat162 t = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&t);
}
__device__ __forceinline__ void sts128(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d)
                 : "memory");
}

// Epilogue for 16 accumulator columns of this thread's row: x sx[m] x sw[n] + b[n] -> GELU -> cast ->
// 32 B (bf16) or 64 B (fp32 / int32) into the warp's 64-byte-swizzled [32 rows x 64 B] staging block;
// each completed 64-byte block goes out as one TMA store (clipped at M / N by the tensor map).
template <int BN, int OUT_T, bool GELU>
__device__ __forceinline__ void w8_epilogue_16(const uint32_t (&v)[16], const float* swb, int cb, float sxv,
                                               uint32_t stg, int lane, const CUtensorMap* tmY, int n0,
                                               int row0) {
    const uint32_t rowb = stg + lane * 64;
    const uint32_t xr = (lane >> 1) & 3;
    const bool first = OUT_T != 1 || (cb & 16) == 0;   // first group of a 64-byte block
    const bool last = OUT_T != 1 || (cb & 16) != 0;    // block complete after this group
    uint32_t w[16];
    if (OUT_T == 2) {
#pragma unroll
        for (int j = 0; j < 16; ++j) w[j] = v[j];
    } else {
        float f[16];
#pragma unroll
        for (int j = 0; j < 16; j += 4) {
            const float4 s4 = *reinterpret_cast<const float4*>(swb + cb + j);
            const float4 b4 = *reinterpret_cast<const float4*>(swb + BN + cb + j);
            f[j] = fmaf(static_cast<float>(static_cast<int32_t>(v[j])) * sxv, s4.x, b4.x);
            f[j + 1] = fmaf(static_cast<float>(static_cast<int32_t>(v[j + 1])) * sxv, s4.y, b4.y);
            f[j + 2] = fmaf(static_cast<float>(static_cast<int32_t>(v[j + 2])) * sxv, s4.z, b4.z);
            f[j + 3] = fmaf(static_cast<float>(static_cast<int32_t>(v[j + 3])) * sxv, s4.w, b4.w);
        }
        if (GELU) {
#pragma unroll
            for (int j = 0; j < 16; ++j) f[j] = gelu_erf(f[j]);
        }
        if (OUT_T == 1) {
#pragma unroll
            for (int j = 0; j < 8; ++j) w[j] = pack_bf16x2(f[2 * j], f[2 * j + 1]);
        } else {
#pragma unroll
            for (int j = 0; j < 16; ++j) w[j] = __float_as_uint(f[j]);
        }
    }
    if (first) {   // the previous TMA store must have finished reading the staging block
        if (lane == 0) tma_store_wait_read<0>();
        __syncwarp();
    }
    if (OUT_T == 1) {
        const uint32_t c0 = (cb & 16) ? 2u : 0u;
        sts128(rowb + (((c0) ^ xr) << 4), w[0], w[1], w[2], w[3]);
        sts128(rowb + (((c0 + 1) ^ xr) << 4), w[4], w[5], w[6], w[7]);
    } else {
#pragma unroll
        for (int c = 0; c < 4; ++c)
            sts128(rowb + ((static_cast<uint32_t>(c) ^ xr) << 4), w[4 * c], w[4 * c + 1], w[4 * c + 2], w[4 * c + 3]);
    }
    if (last) {
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
            tma_store_2d(tmY, stg, n0 + (OUT_T == 1 ? (cb & ~31) : cb), row0);
            tma_store_commit();
        }
    }
}

// OUT_T: 0 = fp32, 1 = bf16, 2 = raw int32 accumulators.  GELU: apply exact-erf GELU (compiled in only
// where used: 32 inlined erff bodies would thrash the instruction cache of every role).
template <int BN, int OUT_T, bool GELU, int CTAS>
__global__ void __launch_bounds__(W8_THREADS, 1)
w8a8_gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                 const __grid_constant__ CUtensorMap tmY, const W8Params p) {
    using Cfg = W8Cfg<BN, CTAS>;
    constexpr int STAGES = Cfg::STAGES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;  // 128-byte swizzle atoms need 1024-byte alignment
    uint8_t* gbase = smem_raw + (base - raw);
    const uint32_t sA = base;
    const uint32_t sB = base + STAGES * Cfg::A_BYTES;
    const uint32_t bars = base + Cfg::BAR_OFF;
    const uint32_t full0 = bars, empty0 = bars + 8 * STAGES;
    const uint32_t tfull0 = bars + 16 * STAGES, tempty0 = tfull0 + 16;
    const uint32_t tmem_slot = tempty0 + 16;
    volatile uint32_t* tmem_slot_g =
        reinterpret_cast<volatile uint32_t*>(gbase + Cfg::BAR_OFF + 16 * STAGES + 32);
    float* swb = reinterpret_cast<float*>(gbase + Cfg::SWB_OFF);

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const uint32_t rank = CTAS == 2 ? cluster_ctarank() : 0u;   // position in the CTA pair
    const int unit0 = blockIdx.x / CTAS, unit_step = gridDim.x / CTAS;
    constexpr int UM = W8_BM * CTAS;                            // rows per work unit
    const int num_m = (p.M + UM - 1) / UM;
    const int num_n = (p.N + BN - 1) / BN;
    const int num_tiles = num_m * num_n;
    const int num_kb = (p.K + W8_BK - 1) / W8_BK;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmA);
        tma_prefetch_desc(&tmB);
        tma_prefetch_desc(&tmY);
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, 1);
        }
        for (int a = 0; a < 2; ++a) {
            mbar_init(tfull0 + 8 * a, 1);
            mbar_init(tempty0 + 8 * a, W8_EPI_WARPS * CTAS);   // the pair's epilogue warps all report to the leader
        }
        fence_mbar_init();
    }
    if (warp == 1) {
        if (CTAS == 2) {
            tmem_alloc_2sm(tmem_slot, Cfg::TMEM_COLS);
            tmem_relinquish_2sm();
        } else {
            tmem_alloc(tmem_slot, Cfg::TMEM_COLS);
            tmem_relinquish();
        }
    }
    tc_fence_before();
    if (CTAS == 2) cluster_sync(); else __syncthreads();       // barriers visible to the peer CTA too
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_g;

    // Everything above overlaps the previous kernel's tail under programmatic dependent launch;
    // global memory written by it (Xq, sx) is only touched after this point.
    pdl_wait_prior_grid();
    pdl_launch_dependents();   // the next kernel may become resident now; it blocks in its own wait
    const long long t_start = clock64();

    if (warp == 0) {
        // ------------------------------------------------------------ TMA producer (every CTA)
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int t = unit0; t < num_tiles; t += unit_step) {
                const int m0 = (t % num_m) * UM + rank * W8_BM;
                const int n0 = (t / num_m) * BN + rank * Cfg::B_ROWS;
                for (int kb = 0; kb < num_kb; ++kb) {
                    mbar_wait(empty0 + 8 * stage, phase ^ 1);
                    if (CTAS == 2) {
                        // both CTAs' bytes are counted on the LEADER's barrier, where the MMA thread waits
                        const uint32_t lbar = (full0 + 8 * stage) & PEER_BIT_MASK;
                        if (rank == 0) mbar_arrive_expect_tx(full0 + 8 * stage, Cfg::STAGE_BYTES * 2);
                        tma_load_2d_2sm(sA + stage * Cfg::A_BYTES, &tmA, kb * W8_BK, m0, lbar);
                        tma_load_2d_2sm(sB + stage * Cfg::B_BYTES, &tmB, kb * W8_BK, n0, lbar);
                    } else {
                        mbar_arrive_expect_tx(full0 + 8 * stage, Cfg::STAGE_BYTES);
                        tma_load_2d(sA + stage * Cfg::A_BYTES, &tmA, kb * W8_BK, m0, full0 + 8 * stage);
                        tma_load_2d(sB + stage * Cfg::B_BYTES, &tmB, kb * W8_BK, n0, full0 + 8 * stage);
                    }
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
            }
            w8_stamp(p, 0, t_start);
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------ MMA issuer (leader CTA only)
        if (lane == 0 && rank == 0) {
            constexpr uint32_t idesc = idesc_i8(UM, BN);
            int stage = 0;
            uint32_t phase = 0;
            int acc = 0;
            uint32_t acc_phase = 0;
            for (int t = unit0; t < num_tiles; t += unit_step) {
                mbar_wait(tempty0 + 8 * acc, acc_phase ^ 1);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + acc * Cfg::ACC_STRIDE;
                for (int kb = 0; kb < num_kb; ++kb) {
                    mbar_wait(full0 + 8 * stage, phase);
                    tc_fence_after();
                    const uint64_t a_desc = make_smem_desc_sw128(sA + stage * Cfg::A_BYTES);
                    const uint64_t b_desc = make_smem_desc_sw128(sB + stage * Cfg::B_BYTES);
#pragma unroll
                    for (int k = 0; k < W8_BK / W8_UMMA_K; ++k) {
                        if (CTAS == 2)
                            mma_i8_ss_2sm(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb | k) != 0 ? 1u : 0u);
                        else
                            mma_i8_ss(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb | k) != 0 ? 1u : 0u);
                    }
                    // ring slot reusable (in both CTAs) once these MMAs retire
                    if (CTAS == 2) tc_commit_2sm(empty0 + 8 * stage, 3); else tc_commit(empty0 + 8 * stage);
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
                // accumulator complete: wake the epilogue warps of both CTAs
                if (CTAS == 2) tc_commit_2sm(tfull0 + 8 * acc, 3); else tc_commit(tfull0 + 8 * acc);
                if (++acc == 2) { acc = 0; acc_phase ^= 1; }
                w8_stamp(p, 2 + min(5, (t - unit0) / unit_step), t_start);
            }
            w8_stamp(p, 1, t_start);
        }
    } else {
        // ------------------------------------------------------------ epilogue (warps 2..9)
        const int ew = warp - 2;
        const int q = warp & 3;          // TMEM lane quarter this warp may read
        constexpr int PQ = W8_EPI_WARPS / 4;   // warps per TMEM lane quarter
        const int part = ew >> 2;        // this warp takes the 32-column chunks c = part, part + PQ, ...
        const int et = threadIdx.x - 64; // 0..255
        const uint32_t stg = base + Cfg::STG_OFF + ew * W8_STG_BYTES;
        int acc = 0;
        uint32_t acc_phase = 0;
        const uint32_t tempty_leader = CTAS == 2 ? mapa_shared(tempty0, 0) : 0u;
        for (int t = unit0; t < num_tiles; t += unit_step) {
            const int m0 = (t % num_m) * UM + rank * W8_BM, n0 = (t / num_m) * BN;
            const int row0 = m0 + q * 32;
            float sxv = 0.0f;
            if (OUT_T != 2) {
                if (row0 + lane < p.M) sxv = __ldg(p.sx + row0 + lane);
                // per-tile column scales and bias -> shared memory (broadcast reads later)
                named_bar_sync(1, 32 * W8_EPI_WARPS);  // previous tile's readers are done
                for (int i = et; i < BN; i += 32 * W8_EPI_WARPS) {
                    const int c = n0 + i;
                    float s = 0.0f, b = 0.0f;
                    if (c < p.N) {
                        s = __ldg(p.sw + c);
                        if (p.bias)
                            b = p.bias_t == ARIA_F32
                                    ? __ldg(static_cast<const float*>(p.bias) + c)
                                    : __bfloat162float(static_cast<const __nv_bfloat16*>(p.bias)[c]);
                    }
                    swb[i] = s;
                    swb[BN + i] = b;
                }
                named_bar_sync(1, 32 * W8_EPI_WARPS);
            }
            mbar_wait(tfull0 + 8 * acc, acc_phase);
            tc_fence_after();
            if (ew == 0 && lane == 0) w8_stamp(p, 8 + 2 * min(3, (t - unit0) / unit_step), t_start);
            const uint32_t t_addr = tmem_base + acc * Cfg::ACC_STRIDE + (static_cast<uint32_t>(q * 32) << 16);
            // A chunk is two groups of 16 columns held in two register sets; the refill of the first set
            // for the next chunk is in flight while the second set is processed.
            constexpr int NC = BN / 32;
            uint32_t va[16], vb[16];
            int c = part;
            if (c < NC) {
                tmem_ld_32x32b_x16(t_addr + c * 32, va);
                tmem_ld_32x32b_x16(t_addr + c * 32 + 16, vb);
                tmem_wait_ld_x16(va);
                tmem_wait_ld_x16(vb);
            }
#pragma unroll 1
            for (; c < NC; c += PQ) {
                const int cn = c + PQ;
                w8_epilogue_16<BN, OUT_T, GELU>(va, swb, c * 32, sxv, stg, lane, &tmY, n0, row0);
                if (cn < NC) tmem_ld_32x32b_x16(t_addr + cn * 32, va);
                w8_epilogue_16<BN, OUT_T, GELU>(vb, swb, c * 32 + 16, sxv, stg, lane, &tmY, n0, row0);
                if (cn < NC) {
                    tmem_ld_32x32b_x16(t_addr + cn * 32 + 16, vb);
                    tmem_wait_ld_x16(va);
                    tmem_wait_ld_x16(vb);
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
                if (CTAS == 2) mbar_arrive_cluster(tempty_leader + 8 * acc);   // leader's barrier
                else mbar_arrive(tempty0 + 8 * acc);
            }
            if (ew == 0 && lane == 0) w8_stamp(p, 9 + 2 * min(3, (t - unit0) / unit_step), t_start);
            if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        }
        if (lane == 0) tma_store_wait<0>();  // all of this warp's output has been written
    }

    tc_fence_before();
    if (CTAS == 2) cluster_sync(); else __syncthreads();       // the peer may still read our smem / TMEM
    if (warp == 1) {
        tc_fence_after();
        if (CTAS == 2) tmem_dealloc_2sm(tmem_base, Cfg::TMEM_COLS);
        else tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
    }
}

template <int BN, int OUT_T, bool GELU, int CTAS>
static int launch_one(const CUtensorMap& tmA, const CUtensorMap& tmB, const CUtensorMap& tmY,
                      const W8Params& p, int grid, cudaStream_t st, bool pdl) {
    using Cfg = W8Cfg<BN, CTAS>;
    static bool attr_set = false;
    auto kern = w8a8_gemm_kernel<BN, OUT_T, GELU, CTAS>;
    if (!attr_set) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES) !=
            cudaSuccess)
            return ARIA_ERR_CUDA;
        attr_set = true;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(W8_THREADS);
    cfg.dynamicSmemBytes = Cfg::SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute at[2];
    int na = 0;
    if (pdl) {
        at[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    if (CTAS == 2) {
        at[na].id = cudaLaunchAttributeClusterDimension;
        at[na].val.clusterDim.x = 2;
        at[na].val.clusterDim.y = 1;
        at[na].val.clusterDim.z = 1;
        ++na;
    }
    cfg.attrs = at;
    cfg.numAttrs = na;
    return cudaLaunchKernelEx(&cfg, kern, tmA, tmB, tmY, p) == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
}

template <int BN, int CTAS>
static int launch_bn(const CUtensorMap& tmA, const CUtensorMap& tmB, const CUtensorMap& tmY,
                     const W8Params& p, int out_t, int grid, cudaStream_t st, bool pdl) {
    const bool gelu = p.act == ARIA_ACT_GELU_ERF;
    switch (out_t) {
        case 0: return gelu ? launch_one<BN, 0, true, CTAS>(tmA, tmB, tmY, p, grid, st, pdl)
                            : launch_one<BN, 0, false, CTAS>(tmA, tmB, tmY, p, grid, st, pdl);
        case 1: return gelu ? launch_one<BN, 1, true, CTAS>(tmA, tmB, tmY, p, grid, st, pdl)
                            : launch_one<BN, 1, false, CTAS>(tmA, tmB, tmY, p, grid, st, pdl);
        default: return launch_one<BN, 2, false, CTAS>(tmA, tmB, tmY, p, grid, st, pdl);
    }
}

// Tile plan: CTAS in {1, 2} x BN in {64, 128, 192, 256} with the fewest wave-quantised cycles.  Per
// 32-byte k-step a work unit costs max(MMA, shared memory) cycles: the MMA takes BN/2 cycles in either
// mode (128 x BN per CTA at 8192 MAC/clk); each CTA's shared memory moves its operands twice (TMA write
// + MMA read) at 128 B/clk: 2 (4096 + 32 BN / CTAS) / 128 = 2 (32 + BN / (4 CTAS)).  Ties go to the
// wider tile and to the pair.
struct W8Plan { int bn, ctas; };
static W8Plan pick_plan(int M, int N, int sms) {
    const int cands[4] = {256, 192, 128, 64};
    W8Plan best = {256, 1};
    long best_cost = -1;
    for (int ctas = 2; ctas >= 1; --ctas) {
        if (ctas == 2 && (M <= W8_BM || sms < 2)) continue;
        const int num_m = (M + W8_BM * ctas - 1) / (W8_BM * ctas);
        const int slots = sms / ctas;
        for (int i = 0; i < 4; ++i) {
            const int bn = cands[i];
            if (ctas == 2 && bn < 128) continue;
            const long tiles = static_cast<long>(num_m) * ((N + bn - 1) / bn);
            const long waves = (tiles + slots - 1) / slots;
            const long mma = bn / 2, smem = 2 * (32 + bn / (4 * ctas));
            const long cost = waves * (mma > smem ? mma : smem);
            if (best_cost < 0 || cost < best_cost) { best_cost = cost; best.bn = bn; best.ctas = ctas; }
        }
    }
    return best;
}

int launch_gemm_w8a8(const int8_t* Xq, const int8_t* Wq, int M, int N, int K, const W8Epilogue& ep,
                     cudaStream_t st, bool pdl) {
    const int sms = num_sms();
    if (sms <= 0) return ARIA_ERR_CUDA;
    const W8Plan plan = pick_plan(M, N, sms);
    const int bn = plan.bn, ctas = plan.ctas;
    CUtensorMap tmA, tmB;
    int rc = make_tmap_2d(&tmA, Xq, 1, M, K, W8_BM, W8_BK, 128);
    if (rc != ARIA_OK) return rc;
    rc = make_tmap_2d(&tmB, Wq, 1, N, K, bn / ctas, W8_BK, 128);
    if (rc != ARIA_OK) return rc;
    // output tensor map: [M, N] of 2- or 4-byte elements, box = 32 rows x 64 bytes, 64-byte swizzle
    CUtensorMap tmY;
    const int esz = ep.out_t == 1 ? 2 : 4;
    rc = make_tmap_2d(&tmY, ep.Y, esz, M, N, 32, 64 / esz, 64);
    if (rc != ARIA_OK) return rc;
    W8Params p;
    p.sx = ep.sx; p.sw = ep.sw; p.bias = ep.bias;
    p.bias_t = ep.bias_t; p.act = ep.act;
    p.M = M; p.N = N; p.K = K;
    p.prof = g_w8_prof;
    const int um = W8_BM * ctas;
    const int tiles = ((M + um - 1) / um) * ((N + bn - 1) / bn);
    const int slots = sms / ctas;
    const int grid = (tiles < slots ? tiles : slots) * ctas;
    if (ctas == 2) {
        switch (bn) {
            case 128: return launch_bn<128, 2>(tmA, tmB, tmY, p, ep.out_t, grid, st, pdl);
            case 192: return launch_bn<192, 2>(tmA, tmB, tmY, p, ep.out_t, grid, st, pdl);
            default: return launch_bn<256, 2>(tmA, tmB, tmY, p, ep.out_t, grid, st, pdl);
        }
    }
    switch (bn) {
        case 64: return launch_bn<64, 1>(tmA, tmB, tmY, p, ep.out_t, grid, st, pdl);
        case 128: return launch_bn<128, 1>(tmA, tmB, tmY, p, ep.out_t, grid, st, pdl);
        case 192: return launch_bn<192, 1>(tmA, tmB, tmY, p, ep.out_t, grid, st, pdl);
        default: return launch_bn<256, 1>(tmA, tmB, tmY, p, ep.out_t, grid, st, pdl);
    }
}

}  // namespace aria
