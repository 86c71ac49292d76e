// static_ws.cu -- aria_linear_w8a8_static_ws: the W8A8 linear for callers that cannot hand the library a
// workspace because they cannot allocate one.
//
// Who that is.  aria_linear_w8a8 needs M*K + 4*M bytes of scratch between its two kernels (the int8 codes
// and per-token scales that S1 writes and the GEMM reads) and asks the caller for it.  Some callers have no
// way to get device memory at the point where they run a linear:
//   - an audio callback or any other deadline-driven thread (the paper's runtime generates audio on the
//     device it plays on): cudaMalloc takes a process-wide lock, may synchronise the whole device and has no
//     latency bound, so such threads are written to never call it;
//   - a plug-in living inside a host application or serving engine that reserved all of the GPU's memory
//     for its own pool at start-up: a cudaMalloc from the plug-in simply fails with out-of-memory;
//   - code that was given raw device pointers by a foreign runtime and holds no allocator handle at all.
// For them the scratch lives in this library's image: a file-scope device array of ARIA_STATIC_WS_BYTES.  It
// costs that much memory on every GPU that loads this module, from the first call until the process exits.
//
// What the entry point does NOT do: it calls no cudaMalloc / cudaFree / cudaMallocAsync and no library routine
// that allocates; the only set-up is one cudaGetSymbolAddress per device (first call on that device).
#include <mutex>

#include "internal.cuh"

using namespace aria;

// The scratch.  In HOST code `g_static_ws` is only a handle the runtime uses to find the symbol; it is not a
// device address, so it is never passed to a kernel.  The device address comes from cudaGetSymbolAddress below.
static __device__ __align__(256) unsigned char g_static_ws[ARIA_STATIC_WS_BYTES];

namespace {

inline bool misaligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }
inline bool bad_dtype(int t) { return t != ARIA_F32 && t != ARIA_BF16; }
inline size_t up256(size_t x) { return (x + 255) / 256 * 256; }

std::mutex g_mu;
void* g_ws_addr[64] = {};   // device address of g_static_ws, per device ordinal; nullptr = not looked up yet

// Device address of the scratch on the CURRENT device.  The array exists once per GPU, at a different address
// on each, so the lookup is done (and cached) per device with that device current.
int static_ws_address(void** out) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return ARIA_ERR_CUDA;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_ws_addr[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_ws) != cudaSuccess || !p) {
            (void)cudaGetLastError();
            return ARIA_ERR_CUDA;
        }
        g_ws_addr[dev] = p;
    }
    *out = g_ws_addr[dev];
    return ARIA_OK;
}

}  // namespace

extern "C" {

size_t aria_static_ws_bytes(void) { return ARIA_STATIC_WS_BYTES; }

int aria_linear_w8a8_static_ws(const void* X, int xt, int M, int K, const int8_t* Wq, const float* w_scale, int N,
                               const void* bias, int bt, int act, void* Y, int yt, void* stream) {
    if (!X || !Wq || !w_scale || !Y) return ARIA_ERR_NULL;
    if (M <= 0 || N <= 0 || K <= 0 || K % 32 != 0 || N % 8 != 0) return ARIA_ERR_SHAPE;
    if (bad_dtype(xt) || bad_dtype(yt) || (bias && bad_dtype(bt)) || (act != ARIA_ACT_NONE && act != ARIA_ACT_GELU_ERF))
        return ARIA_ERR_DTYPE;
    if (misaligned16(X) || misaligned16(Wq) || misaligned16(w_scale) || misaligned16(bias) || misaligned16(Y))
        return ARIA_ERR_ALIGN;
    // codes [M,K] (rounded up to 256 bytes) followed by the scales [M]: the layout aria_linear_w8a8 uses in `ws`
    const size_t codes = up256(static_cast<size_t>(M) * K), scales = up256(static_cast<size_t>(M) * 4);
    if (codes + scales > ARIA_STATIC_WS_BYTES) return ARIA_ERR_WORKSPACE;   // beyond the built-in scratch: nothing enqueued
    int rc = check_arch();
    if (rc != ARIA_OK) return rc;
    void* ws = nullptr;
    rc = static_ws_address(&ws);
    if (rc != ARIA_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int8_t* Xq = static_cast<int8_t*>(ws);
    float* sx = reinterpret_cast<float*>(static_cast<unsigned char*>(ws) + codes);
    // Same two launches, same arguments and same launch attributes as aria_linear_w8a8.  Nothing in the scratch has
    // to start at zero: S1 writes every code and every scale the GEMM reads (the GEMM's loads are bounded by M and K
    // through its tensor map), so what an earlier call left behind is never observed.
    rc = launch_quant_rows_i8(X, xt, M, K, Xq, sx, st, true);
    if (rc != ARIA_OK) return rc;
    W8Epilogue ep;
    ep.sx = sx; ep.sw = w_scale; ep.bias = bias; ep.bias_t = bt; ep.act = act; ep.Y = Y;
    ep.out_t = yt == ARIA_F32 ? 0 : 1;
    return launch_gemm_w8a8(Xq, Wq, M, N, K, ep, st, true);
}

}  // extern "C"
