// internal.cuh -- declarations shared by the translation units of libaria_b200.
#pragma once
#include <cstdio>

#include <atomic>
#include <cstdlib>

#include "../../include/aria.h"
#include "ptx.cuh"

namespace aria {

// Debug switches (environment variables, role-timestamp buffers, the aria_debug_* exports) exist only
// in builds with -DARIA_DEBUG (python -m paper_2607_08526_b200.build --debug).  The product library
// reads no environment variable: dbg_env() folds to nullptr and every switch to its default.
#ifdef ARIA_DEBUG
inline const char* dbg_env(const char* name) { return getenv(name); }
#else
inline const char* dbg_env(const char*) { return nullptr; }
#endif

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-DEVICE attribute of a kernel: set it once per
// (kernel instantiation, device).  `mask` is that instantiation's bit set of devices already done.
template <typename Kern>
inline bool ensure_dyn_smem(Kern kern, int bytes, std::atomic<uint64_t>& mask) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return false;
    const uint64_t bit = 1ull << dev;
    if (mask.load(std::memory_order_acquire) & bit) return true;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) != cudaSuccess) return false;
    mask.fetch_or(bit, std::memory_order_release);
    return true;
}

// ---- quant.cu
// known_absmax: per-row max |x| already computed by the producing epilogue (fused S1): the pass
// skips its reduction.  zero_absmax: a [R] buffer this pass zeroes (the buffer the GEMM that consumes
// this pass's codes will atomicMax into).  check_known: known_absmax comes from outside the library and may be
// too small -- rows where it is are rounded by the clamping path (the other kernels check for free, always).
int launch_quant_rows_i8(const void* X, int xt, int R, int C, int8_t* q, float* s, cudaStream_t st,
                         bool pdl, const float* known_absmax = nullptr, float* zero_absmax = nullptr,
                         bool check_known = false);
int launch_quant_groups_i4(const void* W, int wt, int N, int K, uint8_t* q4, uint16_t* sg,
                           cudaStream_t st);

// ---- tensormap.cu
// 2-D row-major tensor [rows, cols] of `elem_bytes`-wide elements; box = [box_rows, box_cols];
// swizzle_bytes in {0, 32, 64, 128}.  Returns ARIA_OK or ARIA_ERR_CUDA.
int make_tmap_2d(CUtensorMap* out, const void* base, int elem_bytes, uint64_t rows, uint64_t cols,
                 uint32_t box_rows, uint32_t box_cols, int swizzle_bytes);
// 3-D tensor, dims (d0 innermost, d1, d2) with byte strides of d1 and d2; box = (box0, box1, box2).
int make_tmap_3d(CUtensorMap* out, const void* base, int elem_bytes, uint64_t d0, uint64_t d1, uint64_t d2,
                 uint64_t stride1_bytes, uint64_t stride2_bytes, uint32_t box0, uint32_t box1, uint32_t box2,
                 int swizzle_bytes);
int num_sms();
int check_arch();  // ARIA_OK on compute capability 10.x, else ARIA_ERR_ARCH / ARIA_ERR_CUDA

// ---- gemm_w8a8.cu
// out_t: 0 = fp32, 1 = bf16, 2 = raw int32 accumulators (sx/sw/bias ignored).
struct W8Epilogue {
    const float* sx;
    const float* sw;
    const void* bias;  // may be nullptr
    int bias_t;        // aria_dtype of bias
    int act;           // aria_act
    void* Y;
    int out_t;
    float* row_absmax = nullptr;   // fused S1 (first half): per-row max |y| as stored, atomicMax; or nullptr
};
// S1 of the NEXT layer, run by the GEMM kernel's epilogue warps while they wait for their first accumulator
// (gemm_w8a8.cu: w8_side_quant).  Only for an input that the GEMM does not write.
struct W8Side {
    const void* X = nullptr;             // [M, K2] activations of the next layer, a row <= 8 KB; nullptr: no side job
    int xt = 0, K2 = 0;
    int8_t* q = nullptr;                 // [M, K2] codes
    float* s = nullptr;                  // [M] scales
    float* zero_absmax = nullptr;        // the [M] absmax buffer the NEXT GEMM's epilogue will reduce into: zeroed here
};
int launch_gemm_w8a8(const int8_t* Xq, const int8_t* Wq, int M, int N, int K, const W8Epilogue& ep,
                     cudaStream_t st, bool pdl, const W8Side* side = nullptr);

void w8_tile_plan(int M, int N, int sms, int* bn, int* ctas);   // the (BN, CTAS) launch_gemm_w8a8 picks
#ifdef ARIA_DEBUG
void w8_set_profile_buffer(long long* p);  // per-CTA role timestamps
#endif

// ---- gemm_w4a16.cu
// ws: split-K partials + tile counters (w4_workspace_bytes); too small / null -> no split-K.
// wbits = 4: Wq = packed int4 [N, K/2], scale = fp16 bits [N, K/32];  wbits = 8 (W8A16): Wq = int8 [N, K],
// scale = fp32 [N].
int launch_gemm_w4a16(const void* X, int M, int K, const uint8_t* Wq, const void* scale,
                      int N, const void* bias, int act, void* Y, int yt, void* ws, size_t ws_bytes,
                      cudaStream_t st, bool pdl, int wbits = 4);
size_t w4_workspace_bytes(int M, int N, int K, int sms);
void w4_plan(int M, int N, int K, int sms, int* tt, int* splits);   // the (token tile, split-K) launch_gemm_w4a16 picks
#ifdef ARIA_DEBUG
void w4_set_profile_buffer(long long* p);  // per-CTA role timestamps
#endif

// ---- steer.cu: in-graph activation steering (eq. 2 / projection), strength read from device memory
int launch_steer(void* H, int ht, int M, int D, const float* d, const float* strength, float hbar_norm, int op,
                 cudaStream_t st);

// ---- norm.cu: LayerNorm / RMSNorm fused with the S1 quantiser (NEXT-2).  Xn (normalised tensor, dtype xt) may be nullptr.
int launch_norm_quant(const void* X, int xt, int M, int K, const float* gamma, const float* beta, int kind, float eps,
                      void* Xn, int8_t* q, float* s, cudaStream_t st, bool pdl);

// ---- attention.cu: fused full self-attention on the [B*S, 3*H*64] bf16 output of the QKV projection (NEXT-2)
int launch_attention(const void* QKV, int B, int S, int H, float scale, void* O, float* row_absmax, cudaStream_t st,
                     bool pdl);
#ifdef ARIA_DEBUG
void att_set_profile_buffer(long long* p);  // per-CTA role timings
#endif

// ---- peak.cu: measurement helper (tensor-pipe issue loop)
int tensor_peak(int kind, int ctas, int iters, double seconds, double* out, cudaStream_t st);

// ---- w4a16_stream.cu: persistent weight-streaming kernel for a list of W4A16 linears at M <= 32
struct WsPlan;
bool ws_eligible(const aria_layer* layers, int n_layers, int M, int mode, int io);
int ws_plan_create(const aria_layer* layers, int n_layers, int M, int io, WsPlan** out);
int ws_plan_run(const WsPlan* plan, cudaStream_t st);
void ws_plan_destroy(WsPlan* plan);
int ws_plan_kind(const WsPlan* plan);                       // 1: fp16 operands + armed bf16 fallback, 2: bf16 operands
int ws_plan_fallback_fired(const WsPlan* plan, int* fired); // synchronous read of the last launch's domain flag
#ifdef ARIA_DEBUG
void ws_set_profile_buffer(long long* p);  // per-CTA role timestamps (read at plan creation)
#endif

}  // namespace aria
