// peak.cu -- measurement helper: the tensor pipe's own peak on this device (SURVEY.md S7 hard part 2,
// S8(d): "measure an int8 peak on the box first (a plain back-to-back tcgen05.mma kind::i8 issue loop
// with no memory traffic)").  Not on the hot path; bench.py calls it to get the denominator of the W8A8
// roofline instead of deriving it from the bf16 figure.
//
// One CTA per SM (or one CTA pair per two SMs).  Every CTA fills one A tile [128 x 128 B] and one B tile
// [256 / CTAS x 128 B] in shared memory with a pseudo-random bit pattern (finite values; random data draws
// realistic power, all-zero operands hold higher clocks), allocates all 512 tensor-memory columns and has
// ONE thread issue `iters` groups of 4 back-to-back tcgen05.mma (the 4 k-steps of a 128-byte k-block, the
// same descriptors as the GEMM kernels) alternating between two 256-column accumulators.  Nothing is
// loaded or stored while the MMAs run.  Operations per group: 2 x (128 CTAS) x 256 x (4 K) with K = 32
// (kind::i8) or 16 (kind::f16, bf16 operands).
#include "internal.cuh"

namespace aria {

constexpr int PK_A_BYTES = 128 * 128;
constexpr int PK_THREADS = 128;

template <int KIND, int CTAS>   // KIND 0: kind::i8 (s8 x s8 -> s32), 1: kind::f16 (bf16 x bf16 -> f32)
__global__ void __launch_bounds__(PK_THREADS, 1) tensor_peak_kernel(int iters, long long* stamps, int ncols, int commit_every) {
    constexpr int B_ROWS = 256 / CTAS;
    constexpr int B_BYTES = B_ROWS * 128;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    uint8_t* gbase = smem_raw + (base - raw);
    const uint32_t sA = base, sB = base + PK_A_BYTES;
    const uint32_t bar = base + PK_A_BYTES + B_BYTES;
    const uint32_t tmem_slot = bar + 8;   // bar + 16: spare barrier
    volatile uint32_t* tmem_slot_g = reinterpret_cast<volatile uint32_t*>(gbase + PK_A_BYTES + B_BYTES + 8);
    const int warp = threadIdx.x >> 5;
    const uint32_t rank = CTAS == 2 ? cluster_ctarank() : 0u;

    // operands: a hash of the byte offset; bf16 words get a fixed exponent (values in +-[0.5, 1)), int8 any byte
    uint32_t* w = reinterpret_cast<uint32_t*>(gbase);
    for (int i = threadIdx.x; i < (PK_A_BYTES + B_BYTES) / 4; i += PK_THREADS) {
        uint32_t h = (i + 1 + blockIdx.x * 7919u) * 2654435761u;
        h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
        w[i] = KIND == 1 ? ((h & 0x807F807Fu) | 0x3F003F00u) : h;
    }
    fence_proxy_async_smem();
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        mbar_init(bar + 16, 1 << 20);      // debug experiments: a barrier that absorbs extra commits
        fence_mbar_init();
    }
    if (warp == 1) {
        if (CTAS == 2) { tmem_alloc_2sm(tmem_slot, 512); tmem_relinquish_2sm(); }
        else { tmem_alloc(tmem_slot, 512); tmem_relinquish(); }
    }
    tc_fence_before();
    if (CTAS == 2) cluster_sync(); else __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_g;

    if (warp == 0 && rank == 0) {
        // ncols = 256 in the product; debug builds may time narrower instructions (ARIA_PEAK_N)
        const uint32_t idesc = KIND == 0 ? idesc_i8(128 * CTAS, ncols) : idesc_bf16(128 * CTAS, ncols);
        const uint64_t desc_hi = make_smem_desc_sw128(0);
        const uint64_t a_desc = desc_hi | ((sA & 0x3FFFF) >> 4);
        const uint64_t b_desc = desc_hi | ((sB & 0x3FFFF) >> 4);
        unsigned long long g0 = 0, g1 = 0;
        long long c0 = 0, c1 = 0;
        if (elect_one()) {
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
            c0 = clock64();
            for (int it = 0; it < iters; ++it) {
                const uint32_t d = tmem_base + (it & 1) * 256;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const uint32_t accum = ((it & 31) >> 1) != 0 || k != 0 ? 1u : 0u;   // restart the sums every 16 groups
                    if (KIND == 0) {
                        if (CTAS == 2) mma_i8_ss_2sm(d, a_desc + 2 * k, b_desc + 2 * k, idesc, accum);
                        else mma_i8_ss(d, a_desc + 2 * k, b_desc + 2 * k, idesc, accum);
                    } else {
                        if (CTAS == 2) mma_f16_ss_2sm(d, a_desc + 2 * k, b_desc + 2 * k, idesc, accum);
                        else mma_f16_ss(d, a_desc + 2 * k, b_desc + 2 * k, idesc, accum);
                    }
                }
#ifdef ARIA_DEBUG
                if (commit_every > 0 && (it % commit_every) == commit_every - 1) {     // timing experiment: commits in the stream
                    if (CTAS == 2) tc_commit_2sm(bar + 16, 1); else tc_commit(bar + 16);
                }
#endif
            }
            if (CTAS == 2) tc_commit_2sm(bar, 1); else tc_commit(bar);
        }
        __syncwarp();
        mbar_wait(bar, 0);            // every MMA has retired
        if (elect_one()) {
            c1 = clock64();
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
            stamps[2 * (blockIdx.x / CTAS)] = c1 - c0;
            stamps[2 * (blockIdx.x / CTAS) + 1] = static_cast<long long>(g1 - g0);
        }
        __syncwarp();
    }
    tc_fence_before();
    if (CTAS == 2) cluster_sync(); else __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        if (CTAS == 2) tmem_dealloc_2sm(tmem_base, 512); else tmem_dealloc(tmem_base, 512);
    }
}

template <int KIND, int CTAS>
static int run_peak(int iters, int sms, long long* d_stamps, cudaStream_t st) {
    constexpr int SMEM = PK_A_BYTES + (256 / CTAS) * 128 + 64 + 1024;
    static std::atomic<uint64_t> attr_done{0};
    auto kern = tensor_peak_kernel<KIND, CTAS>;
    if (!ensure_dyn_smem(kern, SMEM, attr_done)) return ARIA_ERR_CUDA;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((sms / CTAS) * CTAS);
    cfg.blockDim = dim3(PK_THREADS);
    cfg.dynamicSmemBytes = SMEM;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = CTAS;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    static const char* n_env = dbg_env("ARIA_PEAK_N");
    const int ncols = n_env ? atoi(n_env) : 256;
    static const char* c_env = dbg_env("ARIA_PEAK_COMMIT");
    const int commit_every = c_env ? atoi(c_env) : 0;
    return cudaLaunchKernelEx(&cfg, kern, iters, d_stamps, ncols, commit_every) == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
}

int tensor_peak(int kind, int ctas, int iters, double seconds, double* out, cudaStream_t st) {
    const int sms = num_sms();
    if (sms <= 0) return ARIA_ERR_CUDA;
    const int units = sms / ctas;
    long long* d_stamps = nullptr;
    if (cudaMalloc(&d_stamps, sizeof(long long) * 2 * units) != cudaSuccess) return ARIA_ERR_CUDA;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = cudaEventCreate(&e0) == cudaSuccess && cudaEventCreate(&e1) == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
    auto launch = [&]() {
        if (kind == 0) return ctas == 2 ? run_peak<0, 2>(iters, sms, d_stamps, st) : run_peak<0, 1>(iters, sms, d_stamps, st);
        return ctas == 2 ? run_peak<1, 2>(iters, sms, d_stamps, st) : run_peak<1, 1>(iters, sms, d_stamps, st);
    };
    if (rc == ARIA_OK) rc = launch();                                   // warm-up
    if (rc == ARIA_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = ARIA_ERR_CUDA;
    // Launches are repeated back to back until `seconds` of device time have passed; the LAST launch is
    // the one reported (after seconds of load it runs at the clocks the power cap allows).
    double elapsed = 0.0, last_ms = 0.0;
    int launches = 0;
    while (rc == ARIA_OK && (launches == 0 || elapsed < seconds)) {
        float ms = 0.0f;
        if (cudaEventRecord(e0, st) != cudaSuccess) { rc = ARIA_ERR_CUDA; break; }
        rc = launch();
        if (rc != ARIA_OK) break;
        if (cudaEventRecord(e1, st) != cudaSuccess || cudaEventSynchronize(e1) != cudaSuccess ||
            cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) { rc = ARIA_ERR_CUDA; break; }
        last_ms = ms;
        elapsed += ms * 1e-3;
        ++launches;
    }
    if (rc == ARIA_OK) {
        long long h[2] = {0, 0};
        if (cudaMemcpy(h, d_stamps, sizeof(h), cudaMemcpyDeviceToHost) != cudaSuccess) rc = ARIA_ERR_CUDA;
        const double k_per_mma = kind == 0 ? 32.0 : 16.0;
        const double ops = 2.0 * 128.0 * ctas * 256.0 * 4.0 * k_per_mma * iters * units;
        out[0] = ops / (last_ms * 1e-3);                                // op/s over the whole launch (CUDA events)
        out[1] = h[1] > 0 ? 1e3 * static_cast<double>(h[0]) / static_cast<double>(h[1]) : 0.0;   // SM MHz in the loop
        out[2] = static_cast<double>(h[0]) / (4.0 * iters);            // SM cycles per tcgen05.mma (unit 0)
        out[3] = static_cast<double>(launches);
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(d_stamps);
    return rc;
}

}  // namespace aria
