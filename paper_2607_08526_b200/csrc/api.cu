// api.cu -- the extern "C" boundary declared in include/aria.h: argument validation and the
// sequencing of kernels.  Device entry points only enqueue on the caller's stream.
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "internal.cuh"

using namespace aria;

namespace {

inline bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }
inline bool bad_dtype(int t) { return t != ARIA_F32 && t != ARIA_BF16; }
inline bool bad_act(int a) { return a != ARIA_ACT_NONE && a != ARIA_ACT_GELU_ERF; }
inline size_t up256(size_t x) { return (x + 255) / 256 * 256; }
inline size_t dsize(int t) { return t == ARIA_F32 ? 4 : 2; }

int check_rows_args(const void* in, int t, int R, int C, const void* q, const void* s) {
    if (!in || !q || !s) return ARIA_ERR_NULL;
    if (R <= 0 || C <= 0 || C % 32 != 0) return ARIA_ERR_SHAPE;
    if (bad_dtype(t)) return ARIA_ERR_DTYPE;
    if (misaligned(in) || misaligned(q) || misaligned(s)) return ARIA_ERR_ALIGN;
    return check_arch();
}

// per-token absmax [M] of one fused-S1 producer
size_t w8_fuse_bytes(int M) { return up256(static_cast<size_t>(M) * 4); }

size_t w8_ws_bytes(int M, int K) { return up256(static_cast<size_t>(M) * K) + up256(static_cast<size_t>(M) * 4); }

// One W8A8 linear as two launches: the S1 kernel, then the GEMM as its programmatic dependent (the GEMM's
// prologue -- barrier init, tensor-memory allocation, tensor-map prefetch -- overlaps the quantiser).
// pdl_first: whether the S1 kernel itself is a programmatic dependent of what precedes it on the stream.  The
// rule is the one include/aria.h states under "Programmatic dependent launch": the stand-alone entry points
// pass true (safe after every predecessor except a foreign programmatic dependent that never waits); layer 0
// of aria_denoiser_linears passes false, so a captured step starts with a fully serialised launch.
int linear_w8a8_impl(const void* X, int xt, int M, int K, const int8_t* Wq, const float* w_scale,
                     int N, const void* bias, int bt, int act, void* Y, int yt, void* ws,
                     cudaStream_t st, bool pdl_first, bool pdl) {
    int8_t* Xq = static_cast<int8_t*>(ws);
    float* sx = reinterpret_cast<float*>(static_cast<uint8_t*>(ws) + up256(static_cast<size_t>(M) * K));
    int rc = launch_quant_rows_i8(X, xt, M, K, Xq, sx, st, pdl_first);
    if (rc != ARIA_OK) return rc;
    W8Epilogue ep;
    ep.sx = sx; ep.sw = w_scale; ep.bias = bias; ep.bias_t = bt; ep.act = act; ep.Y = Y;
    ep.out_t = yt == ARIA_F32 ? 0 : 1;
    return launch_gemm_w8a8(Xq, Wq, M, N, K, ep, st, pdl);
}

int check_layers(const aria_layer* layers, int n_layers, int M, int mode, int io, int* maxK,
                 int* maxN, bool host_io) {
    if (!layers) return ARIA_ERR_NULL;
    if (n_layers <= 0 || M <= 0) return ARIA_ERR_SHAPE;
    if (mode != ARIA_W8A8 && mode != ARIA_W4A16 && mode != ARIA_W8A16) return ARIA_ERR_DTYPE;
    if (bad_dtype(io) || (mode != ARIA_W8A8 && io != ARIA_BF16)) return ARIA_ERR_DTYPE;
    *maxK = 0; *maxN = 0;
    for (int i = 0; i < n_layers; ++i) {
        const aria_layer& L = layers[i];
        if (!L.wq || !L.w_scale || !L.out) return ARIA_ERR_NULL;
        if (!L.in && (i == 0 || layers[i - 1].N != L.K)) return i == 0 ? ARIA_ERR_NULL : ARIA_ERR_SHAPE;
        if (L.K <= 0 || L.N <= 0 || L.K % 32 != 0 || L.N % 8 != 0) return ARIA_ERR_SHAPE;
        if (bad_act(L.act)) return ARIA_ERR_DTYPE;
        if (misaligned(L.wq) || misaligned(L.w_scale) || misaligned(L.bias)) return ARIA_ERR_ALIGN;
        if (!host_io && (misaligned(L.in) || misaligned(L.out))) return ARIA_ERR_ALIGN;
        if (L.K > *maxK) *maxK = L.K;
        if (L.N > *maxN) *maxN = L.N;
    }
    return check_arch();
}

// first: this is the first kernel sequence of a chain (no programmatic dependency on what precedes it).
int run_layer(const aria_layer& L, const void* in, void* out, int M, int mode, int io, void* ws,
              size_t ws_bytes, cudaStream_t st, bool first) {
    static const bool pdl = dbg_env("ARIA_NO_PDL") == nullptr;            // debug builds only
    if (mode == ARIA_W8A8)
        return linear_w8a8_impl(in, io, M, L.K, static_cast<const int8_t*>(L.wq),
                                static_cast<const float*>(L.w_scale), L.N, L.bias, io, L.act, out, io,
                                ws, st, pdl && !first, pdl);
    return launch_gemm_w4a16(in, M, L.K, static_cast<const uint8_t*>(L.wq), L.w_scale, L.N, L.bias, L.act,
                             out, io, ws, ws_bytes, st, pdl && !first, mode == ARIA_W8A16 ? 8 : 4);
}

}  // namespace

// Copy streams and events of aria_denoiser_linears_host, created once per device.
struct HostPipe {
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t ev_start = nullptr, ev_in[2] = {nullptr, nullptr}, ev_comp[2] = {nullptr, nullptr},
                ev_out[2] = {nullptr, nullptr};
    bool ok = false;
};
static HostPipe* host_pipe() {
    static HostPipe pipes[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
    HostPipe& h = pipes[dev];
    if (!h.ok) {
        bool good = cudaStreamCreateWithFlags(&h.s_in, cudaStreamNonBlocking) == cudaSuccess &&
                    cudaStreamCreateWithFlags(&h.s_out, cudaStreamNonBlocking) == cudaSuccess &&
                    cudaEventCreateWithFlags(&h.ev_start, cudaEventDisableTiming) == cudaSuccess;
        for (int i = 0; good && i < 2; ++i)
            good = cudaEventCreateWithFlags(&h.ev_in[i], cudaEventDisableTiming) == cudaSuccess &&
                   cudaEventCreateWithFlags(&h.ev_comp[i], cudaEventDisableTiming) == cudaSuccess &&
                   cudaEventCreateWithFlags(&h.ev_out[i], cudaEventDisableTiming) == cudaSuccess;
        if (!good) return nullptr;
        h.ok = true;
    }
    return &h;
}

struct aria_stack_plan {
    std::vector<aria_layer> layers;
    int M = 0, mode = 0, io = 0;
    WsPlan* ws_plan = nullptr;      // small-M W4A16: the persistent stream kernel (w4a16_stream.cu)
    void* d_ws = nullptr;           // otherwise: scratch of the per-layer path
    size_t ws_bytes = 0;
};

extern "C" {

const char* aria_version(void) { return "aria-b200 0.1 sm_100a"; }

const char* aria_status_string(int status) {
    switch (status) {
        case ARIA_OK: return "ok";
        case ARIA_ERR_NULL: return "null pointer";
        case ARIA_ERR_SHAPE: return "bad shape";
        case ARIA_ERR_ALIGN: return "pointer not 16-byte aligned";
        case ARIA_ERR_DTYPE: return "bad dtype / activation / mode";
        case ARIA_ERR_ARCH: return "device is not sm_100 (no fallback)";
        case ARIA_ERR_WORKSPACE: return "workspace missing or too small";
        case ARIA_ERR_CUDA: return "CUDA error";
        default: return "unknown status";
    }
}

size_t aria_workspace_bytes(int M, int maxK, int maxN, int mode) {
    if (M <= 0 || maxK <= 0 || maxN <= 0) return 0;
    // two (Xq, sx) buffers and two per-token absmax buffers (fused S1): see aria_denoiser_linears
    if (mode == ARIA_W8A8) return 2 * w8_ws_bytes(M, maxK) + 2 * w8_fuse_bytes(M);
    if (mode == ARIA_W4A16 || mode == ARIA_W8A16) {
        // Split-K bound: splits * tiles <= #SMs and a tile holds <= 128 x TT outputs, so the fp32
        // partials never exceed #SMs * 128 * TT * 4 bytes; one counter quad per tile.
        int sms = num_sms();
        if (sms <= 0) sms = 148;
        size_t tiles = static_cast<size_t>((maxN + 127) / 128) * ((M + 31) / 32);
        return up256(tiles * 16) + up256(static_cast<size_t>(sms) * 128 * 256 * 4);
    }
    return 0;
}

size_t aria_workspace_bytes_host(int M, int maxK, int maxN, int mode, int io) {
    const size_t dev = aria_workspace_bytes(M, maxK, maxN, mode);
    if (dev == 0 || bad_dtype(io)) return 0;
    // device scratch + two input staging buffers + two output staging buffers
    return up256(dev) + 2 * up256(static_cast<size_t>(M) * maxK * dsize(io)) +
           2 * up256(static_cast<size_t>(M) * maxN * dsize(io));
}

int aria_quantize_weights_int8(const void* W, int wt, int N, int K, int8_t* Wq, float* w_scale,
                               void* stream) {
    int rc = check_rows_args(W, wt, N, K, Wq, w_scale);
    if (rc != ARIA_OK) return rc;
    return launch_quant_rows_i8(W, wt, N, K, Wq, w_scale, static_cast<cudaStream_t>(stream), false);
}

int aria_quantize_act_int8(const void* X, int xt, int M, int K, int8_t* Xq, float* x_scale,
                           void* stream) {
    int rc = check_rows_args(X, xt, M, K, Xq, x_scale);
    if (rc != ARIA_OK) return rc;
    return launch_quant_rows_i8(X, xt, M, K, Xq, x_scale, static_cast<cudaStream_t>(stream), true);
}

int aria_quantize_weights_int4(const void* W, int wt, int N, int K, int group, uint8_t* Wq4,
                               uint16_t* g_scale, void* stream) {
    if (!W || !Wq4 || !g_scale) return ARIA_ERR_NULL;
    if (N <= 0 || K <= 0 || K % 32 != 0 || group != 32) return ARIA_ERR_SHAPE;
    if (bad_dtype(wt)) return ARIA_ERR_DTYPE;
    if (misaligned(W) || misaligned(Wq4) || misaligned(g_scale)) return ARIA_ERR_ALIGN;
    int rc = check_arch();
    if (rc != ARIA_OK) return rc;
    return launch_quant_groups_i4(W, wt, N, K, Wq4, g_scale, static_cast<cudaStream_t>(stream));
}

int aria_linear_w8a8(const void* X, int xt, int M, int K, const int8_t* Wq, const float* w_scale,
                     int N, const void* bias, int bt, int act, void* Y, int yt, void* ws,
                     size_t ws_bytes, void* stream) {
    if (!X || !Wq || !w_scale || !Y) return ARIA_ERR_NULL;
    if (M <= 0 || N <= 0 || K <= 0 || K % 32 != 0 || N % 8 != 0) return ARIA_ERR_SHAPE;
    if (bad_dtype(xt) || bad_dtype(yt) || (bias && bad_dtype(bt)) || bad_act(act)) return ARIA_ERR_DTYPE;
    if (misaligned(X) || misaligned(Wq) || misaligned(w_scale) || misaligned(bias) || misaligned(Y) ||
        misaligned(ws))
        return ARIA_ERR_ALIGN;
    if (!ws || ws_bytes < w8_ws_bytes(M, K)) return ARIA_ERR_WORKSPACE;
    int rc = check_arch();
    if (rc != ARIA_OK) return rc;
    // both kernels are programmatic dependents of what precedes them (each waits before it touches global
    // memory): the S1 pass overlaps the previous kernel's tail, the GEMM's prologue -- barrier init,
    // tensor-memory allocation, tensor-map prefetch -- overlaps the quantiser
    return linear_w8a8_impl(X, xt, M, K, Wq, w_scale, N, bias, bt, act, Y, yt, ws,
                            static_cast<cudaStream_t>(stream), true, true);
}

int aria_linear_w8a8_q(const int8_t* Xq, const float* x_scale, int M, int K, const int8_t* Wq,
                       const float* w_scale, int N, const void* bias, int bt, int act, void* Y,
                       int yt, void* stream) {
    if (!Xq || !x_scale || !Wq || !w_scale || !Y) return ARIA_ERR_NULL;
    if (M <= 0 || N <= 0 || K <= 0 || K % 32 != 0 || N % 8 != 0) return ARIA_ERR_SHAPE;
    if (bad_dtype(yt) || (bias && bad_dtype(bt)) || bad_act(act)) return ARIA_ERR_DTYPE;
    if (misaligned(Xq) || misaligned(x_scale) || misaligned(Wq) || misaligned(w_scale) ||
        misaligned(bias) || misaligned(Y))
        return ARIA_ERR_ALIGN;
    int rc = check_arch();
    if (rc != ARIA_OK) return rc;
    W8Epilogue ep;
    ep.sx = x_scale; ep.sw = w_scale; ep.bias = bias; ep.bias_t = bt; ep.act = act; ep.Y = Y;
    ep.out_t = yt == ARIA_F32 ? 0 : 1;
    // every kernel of this library touches global memory only after griddepcontrol.wait, so it may be launched as
    // a programmatic dependent of WHATEVER precedes it on the stream: its prologue overlaps that kernel's tail
    return launch_gemm_w8a8(Xq, Wq, M, N, K, ep, static_cast<cudaStream_t>(stream), true);
}

int aria_linear_w4a16(const void* X, int M, int K, const uint8_t* Wq4, const uint16_t* g_scale,
                      int group, int N, const void* bias, int act, void* Y, int yt, void* ws,
                      size_t ws_bytes, void* stream) {
    if (!X || !Wq4 || !g_scale || !Y) return ARIA_ERR_NULL;
    if (M <= 0 || N <= 0 || K <= 0 || K % 32 != 0 || N % 8 != 0 || group != 32) return ARIA_ERR_SHAPE;
    if (bad_dtype(yt) || bad_act(act)) return ARIA_ERR_DTYPE;
    if (misaligned(X) || misaligned(Wq4) || misaligned(g_scale) || misaligned(bias) || misaligned(Y) ||
        misaligned(ws))
        return ARIA_ERR_ALIGN;
    int rc = check_arch();
    if (rc != ARIA_OK) return rc;
    return launch_gemm_w4a16(X, M, K, Wq4, g_scale, N, bias, act, Y, yt, ws, ws ? ws_bytes : 0,
                             static_cast<cudaStream_t>(stream), false);
}

int aria_linear_w8a16(const void* X, int M, int K, const int8_t* Wq, const float* w_scale, int N,
                      const void* bias, int act, void* Y, int yt, void* ws, size_t ws_bytes, void* stream) {
    if (!X || !Wq || !w_scale || !Y) return ARIA_ERR_NULL;
    if (M <= 0 || N <= 0 || K <= 0 || K % 32 != 0 || N % 8 != 0) return ARIA_ERR_SHAPE;
    if (bad_dtype(yt) || bad_act(act)) return ARIA_ERR_DTYPE;
    if (misaligned(X) || misaligned(Wq) || misaligned(w_scale) || misaligned(bias) || misaligned(Y) ||
        misaligned(ws))
        return ARIA_ERR_ALIGN;
    int rc = check_arch();
    if (rc != ARIA_OK) return rc;
    return launch_gemm_w4a16(X, M, K, reinterpret_cast<const uint8_t*>(Wq), w_scale, N, bias, act, Y, yt, ws,
                             ws ? ws_bytes : 0, static_cast<cudaStream_t>(stream), false, 8);
}

int aria_gemm_i8_i32(const int8_t* Xq, const int8_t* Wq, int M, int N, int K, int32_t* acc,
                     void* stream) {
    if (!Xq || !Wq || !acc) return ARIA_ERR_NULL;
    if (M <= 0 || N <= 0 || K <= 0 || K % 32 != 0 || N % 8 != 0) return ARIA_ERR_SHAPE;
    if (misaligned(Xq) || misaligned(Wq) || misaligned(acc)) return ARIA_ERR_ALIGN;
    int rc = check_arch();
    if (rc != ARIA_OK) return rc;
    W8Epilogue ep;
    ep.sx = nullptr; ep.sw = nullptr; ep.bias = nullptr; ep.bias_t = ARIA_F32; ep.act = ARIA_ACT_NONE;
    ep.Y = acc; ep.out_t = 2;
    return launch_gemm_w8a8(Xq, Wq, M, N, K, ep, static_cast<cudaStream_t>(stream), false);
}

#ifdef ARIA_DEBUG
/* Debug builds only (-DARIA_DEBUG, not in aria.h): per-CTA role timestamps of the three GEMM kernels. */
__attribute__((visibility("default"))) void aria_debug_w4_profile(long long* buf) { w4_set_profile_buffer(buf); }
__attribute__((visibility("default"))) void aria_debug_ws_profile(long long* buf) { ws_set_profile_buffer(buf); }
__attribute__((visibility("default"))) void aria_debug_w8_profile(long long* buf) { w8_set_profile_buffer(buf); }
__attribute__((visibility("default"))) void aria_debug_att_profile(long long* buf) { att_set_profile_buffer(buf); }
#endif

int aria_steer(void* H, int ht, int M, int D, const float* d, const float* strength, float hbar_norm, int op,
               void* stream) {
    if (!H || !d || !strength) return ARIA_ERR_NULL;
    if (M <= 0 || D <= 0 || D % 8 != 0) return ARIA_ERR_SHAPE;
    if (bad_dtype(ht) || (op != ARIA_STEER_ADD && op != ARIA_STEER_PROJECT)) return ARIA_ERR_DTYPE;
    if (misaligned(H) || misaligned(d) || (reinterpret_cast<uintptr_t>(strength) & 3u)) return ARIA_ERR_ALIGN;
    int rc = check_arch();
    if (rc != ARIA_OK) return rc;
    return launch_steer(H, ht, M, D, d, strength, hbar_norm, op, static_cast<cudaStream_t>(stream));
}

int aria_norm_quantize_act_int8(const void* X, int xt, int M, int K, const float* gamma, const float* beta, int norm,
                                float eps, void* Xn, int8_t* Xq, float* x_scale, void* stream) {
    // argument validation first (it needs no device), the architecture check last
    if (!gamma) return ARIA_ERR_NULL;
    if (norm != ARIA_NORM_LAYER && norm != ARIA_NORM_RMS) return ARIA_ERR_DTYPE;
    if (!(eps >= 0.0f) || K > 24576) return ARIA_ERR_SHAPE;
    if (misaligned(gamma) || misaligned(beta) || misaligned(Xn)) return ARIA_ERR_ALIGN;
    int rc = check_rows_args(X, xt, M, K, Xq, x_scale);
    if (rc != ARIA_OK) return rc;
    return launch_norm_quant(X, xt, M, K, gamma, beta, norm, eps, Xn, Xq, x_scale, static_cast<cudaStream_t>(stream), true);
}

int aria_attention(const void* QKV, int B, int S, int H, int Dh, float scale, void* O, float* row_absmax, void* stream) {
    if (!QKV || !O) return ARIA_ERR_NULL;
    if (B <= 0 || S <= 0 || H <= 0 || Dh != 64 || !(scale > 0.0f) || B > 65535 || H > 65535) return ARIA_ERR_SHAPE;
    if (misaligned(QKV) || misaligned(O) || (reinterpret_cast<uintptr_t>(row_absmax) & 3u)) return ARIA_ERR_ALIGN;
    int rc = check_arch();
    if (rc != ARIA_OK) return rc;
    return launch_attention(QKV, B, S, H, scale, O, row_absmax, static_cast<cudaStream_t>(stream), true);
}

int aria_round_act_int8(const void* X, int xt, int M, int K, float* absmax, int clear, int8_t* Xq, float* x_scale,
                        void* stream) {
    if (!absmax) return ARIA_ERR_NULL;
    if (reinterpret_cast<uintptr_t>(absmax) & 3u) return ARIA_ERR_ALIGN;
    int rc = check_rows_args(X, xt, M, K, Xq, x_scale);
    if (rc != ARIA_OK) return rc;
    return launch_quant_rows_i8(X, xt, M, K, Xq, x_scale, static_cast<cudaStream_t>(stream), true, absmax, clear ? absmax : nullptr,
                                true);
}

int aria_tensor_peak(int kind, int ctas, int iters, double seconds, double* out, void* stream) {
    if (!out) return ARIA_ERR_NULL;
    if ((kind != 0 && kind != 1) || (ctas != 1 && ctas != 2) || iters <= 0 || iters > (1 << 24) || seconds < 0.0 ||
        seconds > 30.0)
        return ARIA_ERR_SHAPE;
    int rc = check_arch();
    if (rc != ARIA_OK) return rc;
    return tensor_peak(kind, ctas, iters, seconds, out, static_cast<cudaStream_t>(stream));
}

int aria_w8a8_tile_plan(int M, int N, int sms, int* bn, int* ctas) {
    if (!bn || !ctas) return ARIA_ERR_NULL;
    if (M <= 0 || N <= 0 || sms <= 0) return ARIA_ERR_SHAPE;
    w8_tile_plan(M, N, sms, bn, ctas);
    return ARIA_OK;
}

int aria_w4a16_tile_plan(int M, int N, int K, int sms, int* tt, int* splits) {
    if (!tt || !splits) return ARIA_ERR_NULL;
    if (M <= 0 || N <= 0 || K <= 0 || sms <= 0) return ARIA_ERR_SHAPE;
    w4_plan(M, N, K, sms, tt, splits);
    return ARIA_OK;
}

int aria_denoiser_linears(const aria_layer* layers, int n_layers, int M, int mode, int io, void* ws,
                          size_t ws_bytes, void* stream) {
    int maxK, maxN;
    int rc = check_layers(layers, n_layers, M, mode, io, &maxK, &maxN, false);
    if (rc != ARIA_OK) return rc;
    if (misaligned(ws)) return ARIA_ERR_ALIGN;
    if (!ws || ws_bytes < aria_workspace_bytes(M, maxK, maxN, mode)) return ARIA_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (mode != ARIA_W8A8) {
        for (int i = 0; i < n_layers; ++i) {
            const aria_layer& L = layers[i];
            rc = run_layer(L, L.in ? L.in : layers[i - 1].out, L.out, M, mode, io, ws, ws_bytes, st, i == 0);
            if (rc != ARIA_OK) return rc;
        }
        return ARIA_OK;
    }
    // W8A8.  The (Xq, sx) scratch alternates between two buffers.
    //  - A layer whose input is NOT written by the previous layer gets its S1 pass from the previous layer's
    //    GEMM kernel: the epilogue warps quantise it while they wait for their first accumulator
    //    (gemm_w8a8.cu: w8_side_quant).  The GEMM of layer i+1 is then the direct programmatic dependent
    //    of the GEMM of layer i: one completion -> launch hop between GEMMs instead of two.
    //  - A layer whose input IS the previous layer's output (in == NULL, or in == that out) takes the fused
    //    S1 (north_star "activation-quantization pass fused into the previous epilogue"): the producing
    //    epilogue reduces the per-token absmax of what it stores (atomicMax into one of two [M] buffers) and
    //    a stand-alone S1 kernel only rounds.  The buffer a GEMM reduces into is zeroed by the S1 pass of
    //    that same layer (side job of the previous GEMM, or the stand-alone kernel).
    //  - Layer 0, and a layer whose input only partly overlaps the previous output or whose rows exceed the
    //    side job's 8 KB staging buffer, get a plain stand-alone S1 kernel.
    // Every kernel waits for its predecessor (griddepcontrol.wait) before it touches global memory, so
    // "kernel k complete" implies "kernels < k complete"; the side job of GEMM i writes the Xq buffer last
    // read by GEMM i-1, and results equal array order bit for bit.
    static const bool no_fuse = dbg_env("ARIA_NO_FUSED_ABSMAX") != nullptr;   // debug builds only
    static const bool no_side = dbg_env("ARIA_NO_SIDE_QUANT") != nullptr;
    static const bool pdl = dbg_env("ARIA_NO_PDL") == nullptr;
    const size_t half = w8_ws_bytes(M, maxK);
    uint8_t* wsb = static_cast<uint8_t*>(ws);
    float* amax[2] = {reinterpret_cast<float*>(wsb + 2 * half), reinterpret_cast<float*>(wsb + 2 * half + w8_fuse_bytes(M))};
    auto xq_of = [&](int i) { return reinterpret_cast<int8_t*>(wsb + (i & 1) * half); };
    auto sx_of = [&](int i) { return reinterpret_cast<float*>(wsb + (i & 1) * half + up256(static_cast<size_t>(M) * maxK)); };
    auto in_of = [&](int i) { return layers[i].in ? layers[i].in : layers[i - 1].out; };
    auto feeds_next = [&](int i) {   // layer i+1 reads exactly layer i's [M, N] output
        if (no_fuse || i + 1 >= n_layers) return false;
        return in_of(i + 1) == layers[i].out && layers[i + 1].K == layers[i].N;
    };
    auto independent_of_prev = [&](int i) {   // layer i's input is not written by layer i-1
        const uintptr_t a0 = reinterpret_cast<uintptr_t>(in_of(i)), a1 = a0 + static_cast<size_t>(M) * layers[i].K * dsize(io);
        const uintptr_t b0 = reinterpret_cast<uintptr_t>(layers[i - 1].out),
                        b1 = b0 + static_cast<size_t>(M) * layers[i - 1].N * dsize(io);
        return !(a0 < b1 && b0 < a1);
    };
    std::vector<int> prod(n_layers, -1);       // producer index (selects the absmax buffer), or -1
    for (int i = 0, k = 0; i < n_layers; ++i)
        if (feeds_next(i)) prod[i] = k++;
    bool s1_done = false;                      // layer i's S1 was done by the side job of GEMM i-1
    for (int i = 0; i < n_layers; ++i) {
        const aria_layer& L = layers[i];
        if (!s1_done) {
            rc = launch_quant_rows_i8(in_of(i), io, M, L.K, xq_of(i), sx_of(i), st, pdl && i > 0,
                                      i > 0 && prod[i - 1] >= 0 ? amax[prod[i - 1] & 1] : nullptr,
                                      prod[i] >= 0 ? amax[prod[i] & 1] : nullptr);
            if (rc != ARIA_OK) return rc;
        }
        W8Side side;
        s1_done = false;
        if (!no_side && i + 1 < n_layers && prod[i] < 0 && independent_of_prev(i + 1) &&
            static_cast<size_t>(layers[i + 1].K) * dsize(io) <= 8192) {
            side.X = in_of(i + 1);
            side.xt = io;
            side.K2 = layers[i + 1].K;
            side.q = xq_of(i + 1);
            side.s = sx_of(i + 1);
            if (prod[i + 1] >= 0) side.zero_absmax = amax[prod[i + 1] & 1];
            s1_done = true;
        }
        W8Epilogue ep;
        ep.sx = sx_of(i); ep.sw = static_cast<const float*>(L.w_scale); ep.bias = L.bias; ep.bias_t = io;
        ep.act = L.act; ep.Y = L.out; ep.out_t = io == ARIA_F32 ? 0 : 1;
        ep.row_absmax = prod[i] >= 0 ? amax[prod[i] & 1] : nullptr;
        rc = launch_gemm_w8a8(xq_of(i), static_cast<const int8_t*>(L.wq), M, L.N, L.K, ep, st, pdl, &side);
        if (rc != ARIA_OK) return rc;
    }
    return ARIA_OK;
}

int aria_stack_plan_create(const aria_layer* layers, int n_layers, int M, int mode, int io,
                           aria_stack_plan** plan_out) {
    if (!plan_out) return ARIA_ERR_NULL;
    *plan_out = nullptr;
    int maxK, maxN;
    int rc = check_layers(layers, n_layers, M, mode, io, &maxK, &maxN, false);
    if (rc != ARIA_OK) return rc;
    aria_stack_plan* plan = new (std::nothrow) aria_stack_plan;
    if (!plan) return ARIA_ERR_CUDA;
    plan->layers.assign(layers, layers + n_layers);
    plan->M = M; plan->mode = mode; plan->io = io;
    if (ws_eligible(layers, n_layers, M, mode, io)) {
        rc = ws_plan_create(layers, n_layers, M, io, &plan->ws_plan);
    } else {
        plan->ws_bytes = aria_workspace_bytes(M, maxK, maxN, mode);
        rc = cudaMalloc(&plan->d_ws, plan->ws_bytes) == cudaSuccess ? ARIA_OK : ARIA_ERR_CUDA;
    }
    if (rc != ARIA_OK) {
        aria_stack_plan_destroy(plan);
        return rc;
    }
    *plan_out = plan;
    return ARIA_OK;
}

int aria_stack_plan_run(const aria_stack_plan* plan, void* stream) {
    if (!plan) return ARIA_ERR_NULL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (plan->ws_plan) return ws_plan_run(plan->ws_plan, st);
    return aria_denoiser_linears(plan->layers.data(), static_cast<int>(plan->layers.size()), plan->M,
                                 plan->mode, plan->io, plan->d_ws, plan->ws_bytes, stream);
}

int aria_stack_plan_is_streaming(const aria_stack_plan* plan) {
    return plan && plan->ws_plan ? ws_plan_kind(plan->ws_plan) : 0;
}

int aria_stack_plan_fallback_fired(const aria_stack_plan* plan, int* fired) {
    if (!plan || !fired) return ARIA_ERR_NULL;
    *fired = 0;
    return plan->ws_plan ? ws_plan_fallback_fired(plan->ws_plan, fired) : ARIA_OK;
}

void aria_stack_plan_destroy(aria_stack_plan* plan) {
    if (!plan) return;
    ws_plan_destroy(plan->ws_plan);
    cudaFree(plan->d_ws);
    delete plan;
}

int aria_denoiser_linears_host(const aria_layer* layers, int n_layers, int M, int mode, int io,
                               void* ws, size_t ws_bytes, void* stream) {
    int maxK, maxN;
    int rc = check_layers(layers, n_layers, M, mode, io, &maxK, &maxN, true);
    if (rc != ARIA_OK) return rc;
    if (misaligned(ws)) return ARIA_ERR_ALIGN;
    if (!ws || ws_bytes < aria_workspace_bytes_host(M, maxK, maxN, mode, io)) return ARIA_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t dev = up256(aria_workspace_bytes(M, maxK, maxN, mode));
    const size_t in_b = up256(static_cast<size_t>(M) * maxK * dsize(io));
    const size_t out_b = up256(static_cast<size_t>(M) * maxN * dsize(io));
    uint8_t* base = static_cast<uint8_t*>(ws);
    uint8_t* in_stage[2] = {base + dev, base + dev + in_b};
    uint8_t* out_stage[2] = {base + dev + 2 * in_b, base + dev + 2 * in_b + out_b};
    // Three streams: H2D(in_i) on a copy-in stream, layer_i on the caller's stream, D2H(out_i) on a
    // copy-out stream, chained by events, so the (full-duplex) PCIe copies of neighbouring layers overlap
    // each other and the compute.  Two staging buffers per direction: in_stage[b] is rewritten by
    // H2D(i+2) only after layer i has run, out_stage[b] by layer i+2 only after D2H(i) has read it; a
    // chained layer (in == NULL) reads the previous layer's device output on the compute stream.
    HostPipe* hp = host_pipe();
    if (!hp) return ARIA_ERR_CUDA;
    bool ok = cudaEventRecord(hp->ev_start, st) == cudaSuccess &&
              cudaStreamWaitEvent(hp->s_in, hp->ev_start, 0) == cudaSuccess &&
              cudaStreamWaitEvent(hp->s_out, hp->ev_start, 0) == cudaSuccess;
    for (int i = 0; ok && i < n_layers; ++i) {
        const aria_layer& L = layers[i];
        const int b = i & 1;
        const void* din;
        if (L.in) {
            if (i >= 2) ok = ok && cudaStreamWaitEvent(hp->s_in, hp->ev_comp[b], 0) == cudaSuccess;
            ok = ok && cudaMemcpyAsync(in_stage[b], L.in, static_cast<size_t>(M) * L.K * dsize(io),
                                       cudaMemcpyHostToDevice, hp->s_in) == cudaSuccess &&
                 cudaEventRecord(hp->ev_in[b], hp->s_in) == cudaSuccess &&
                 cudaStreamWaitEvent(st, hp->ev_in[b], 0) == cudaSuccess;
            din = in_stage[b];
        } else {
            din = out_stage[(i - 1) & 1];
        }
        if (i >= 2) ok = ok && cudaStreamWaitEvent(st, hp->ev_out[b], 0) == cudaSuccess;
        if (!ok) break;
        rc = run_layer(L, din, out_stage[b], M, mode, io, ws, dev, st, true);
        if (rc != ARIA_OK) break;
        ok = cudaEventRecord(hp->ev_comp[b], st) == cudaSuccess &&
             cudaStreamWaitEvent(hp->s_out, hp->ev_comp[b], 0) == cudaSuccess &&
             cudaMemcpyAsync(L.out, out_stage[b], static_cast<size_t>(M) * L.N * dsize(io),
                             cudaMemcpyDeviceToHost, hp->s_out) == cudaSuccess &&
             cudaEventRecord(hp->ev_out[b], hp->s_out) == cudaSuccess;
    }
    // always drain all three streams, also on an error path: the staging buffers are the caller's
    const bool s1 = cudaStreamSynchronize(hp->s_in) == cudaSuccess;
    const bool s2 = cudaStreamSynchronize(st) == cudaSuccess;
    const bool s3 = cudaStreamSynchronize(hp->s_out) == cudaSuccess;
    if (rc != ARIA_OK) return rc;
    return ok && s1 && s2 && s3 ? ARIA_OK : ARIA_ERR_CUDA;
}

}  // extern "C"
