// internal.cuh -- declarations shared by the translation units of libaria_b200.
#pragma once
#include <cstdio>

#include "../../include/aria.h"
#include "ptx.cuh"

namespace aria {

// ---- quant.cu
// early (needs pdl): the pass does not wait for the previous grid before it starts -- the caller
// guarantees that grid neither writes X nor touches q / s -- but still waits for it before it ends.
int launch_quant_rows_i8(const void* X, int xt, int R, int C, int8_t* q, float* s, cudaStream_t st,
                         bool pdl, bool early = false);
int launch_quant_groups_i4(const void* W, int wt, int N, int K, uint8_t* q4, uint16_t* sg,
                           cudaStream_t st);

// ---- tensormap.cu
// 2-D row-major tensor [rows, cols] of `elem_bytes`-wide elements; box = [box_rows, box_cols];
// swizzle_bytes in {0, 32, 64, 128}.  Returns ARIA_OK or ARIA_ERR_CUDA.
int make_tmap_2d(CUtensorMap* out, const void* base, int elem_bytes, uint64_t rows, uint64_t cols,
                 uint32_t box_rows, uint32_t box_cols, int swizzle_bytes);
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
};
int launch_gemm_w8a8(const int8_t* Xq, const int8_t* Wq, int M, int N, int K, const W8Epilogue& ep,
                     cudaStream_t st, bool pdl);

void w8_set_profile_buffer(long long* p);  // debug hook: per-CTA role timestamps

// ---- gemm_w4a16.cu
// ws: split-K partials + tile counters (w4_workspace_bytes); too small / null -> no split-K.
int launch_gemm_w4a16(const void* X, int M, int K, const uint8_t* Wq4, const uint16_t* g_scale,
                      int N, const void* bias, int act, void* Y, int yt, void* ws, size_t ws_bytes,
                      cudaStream_t st, bool pdl);
size_t w4_workspace_bytes(int M, int N, int K, int sms);
void w4_set_profile_buffer(long long* p);  // debug hook: per-CTA role timestamps

// ---- w4a16_stream.cu: persistent weight-streaming kernel for a list of W4A16 linears at M <= 32
struct WsPlan;
bool ws_eligible(const aria_layer* layers, int n_layers, int M, int mode, int io);
int ws_plan_create(const aria_layer* layers, int n_layers, int M, int io, WsPlan** out);
int ws_plan_run(const WsPlan* plan, cudaStream_t st);
void ws_plan_destroy(WsPlan* plan);
void ws_set_profile_buffer(long long* p);  // debug hook: per-CTA role timestamps (read at plan creation)

}  // namespace aria
