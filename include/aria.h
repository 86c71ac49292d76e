/*
 * aria.h -- C ABI of libaria_b200: the quantized linear layers of the DiT denoiser of
 * arxiv/paper_2607_08526 ("aria"), written for NVIDIA B200 (sm_100a).
 *
 * Source of the operations.  PAPER.md L78 (SIII-A(b), "Quantization and its evaluation"):
 * the transformer's weights are "compressed to 8-bit or 4-bit integers (q8, q4)"; "an
 * optional mode also runs the arithmetic in 8-bit, quantizing activations alongside weights
 * (W8A8), on the GPU's integer tensor cores"; "the compressed copy owns its memory, the
 * runtime frees the full-precision source once packed".  PAPER.md L73: the "per-step
 * denoising loop is captured once and replayed as a single GPU graph".  The paper fixes no
 * quantization scheme; the schemes are those of BASELINE.json `configs` C1-C5, as read in
 * DESIGN.md "Readings" (R1-R17) and SURVEY.md S8(c).
 *
 * Conventions (all entry points):
 *  - X[M,K] activations, row = token; W[N,K] weights, row = output channel; y = x W^T + b;
 *    Y[M,N].  All matrices are dense row-major with no padding.
 *  - Unless a name ends in `_host`, every data pointer is a DEVICE pointer owned by the
 *    caller.  The library allocates and frees nothing on these calls and keeps no pointer
 *    after return.  The fp source of a weight may be freed by the caller as soon as
 *    aria_quantize_weights_* has completed on the stream (the paper's "releases the original").
 *  - `stream` is a cudaStream_t passed as void*.  Device entry points only ENQUEUE work on it:
 *    no host synchronisation, no allocation -- every one of them may be captured in a CUDA
 *    graph.  `_host` entry points copy and synchronise (see there);
 *    aria_linear_w8a8_static_ws has a one-time set-up on its first call per device and states
 *    its own rules (this sentence says nothing about it).
 *  - Programmatic dependent launch.  aria_quantize_act_int8, aria_linear_w8a8, aria_linear_w8a8_static_ws,
 *    aria_linear_w8a8_q, aria_norm_quantize_act_int8, aria_round_act_int8 and aria_attention launch their
 *    first kernel as a PROGRAMMATIC DEPENDENT of whatever precedes it on `stream` (its prologue overlaps
 *    that kernel's tail); every kernel of this library executes griddepcontrol.wait -- which returns only when
 *    the preceding kernel has completed and its writes are visible -- before it reads or writes global
 *    memory.  This is ordinary stream order after any predecessor that was launched normally, and after
 *    this library's own kernels.  The one predecessor it is NOT safe after: a foreign kernel that was itself
 *    launched with the programmatic attribute and exits without cudaGridDependencySynchronize(): such a
 *    kernel can finish before ITS predecessor, and the wait here covers only the immediate predecessor.
 *    Put an event or a normally launched kernel in between in that case.  aria_quantize_weights_*,
 *    aria_linear_w4a16, aria_linear_w8a16, aria_steer and the first kernel of aria_denoiser_linears /
 *    aria_stack_plan_run are plain launches.
 *  - Return value: aria_status (0 = OK, negative = error).  On a validation error nothing is
 *    enqueued and no output is written.  Non-finite inputs are not checked (undefined).
 *  - Alignment: every data pointer must be 16-byte aligned.  K % 32 == 0, N % 8 == 0.
 *  - There is no CPU fallback: on a device that is not sm_100 every compute entry point
 *    returns ARIA_ERR_ARCH.
 */
#ifndef ARIA_H_
#define ARIA_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define ARIA_API __attribute__((visibility("default")))
#else
#define ARIA_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    ARIA_OK = 0,
    ARIA_ERR_NULL = -1,      /* a required pointer is NULL */
    ARIA_ERR_SHAPE = -2,     /* M,N,K <= 0, K % 32 != 0, N % 8 != 0, group != 32, n_layers <= 0 */
    ARIA_ERR_ALIGN = -3,     /* a pointer is not 16-byte aligned */
    ARIA_ERR_DTYPE = -4,     /* unknown / unsupported aria_dtype, aria_act or aria_mode */
    ARIA_ERR_ARCH = -5,      /* current device is not compute capability 10.x */
    ARIA_ERR_WORKSPACE = -6, /* ws is NULL or ws_bytes < aria_workspace_bytes(...) */
    ARIA_ERR_CUDA = -7       /* a CUDA runtime / driver call or a kernel launch failed */
} aria_status;

typedef enum { ARIA_F32 = 0, ARIA_BF16 = 1 } aria_dtype;
typedef enum { ARIA_ACT_NONE = 0, ARIA_ACT_GELU_ERF = 1 } aria_act;
typedef enum { ARIA_W8A8 = 0, ARIA_W4A16 = 1, ARIA_W8A16 = 2 } aria_mode;
typedef enum { ARIA_STEER_ADD = 0, ARIA_STEER_PROJECT = 1 } aria_steer_op;
typedef enum { ARIA_NORM_LAYER = 0, ARIA_NORM_RMS = 1 } aria_norm;

/* ---------------------------------------------------------------------------------------
 * S0 -- weight quantisation, once at load (configs C1-C3; readings R2-R4).
 * Per output channel n:  a = max_k |W[n,k]|;  w_scale[n] = a > 0 ? fl32(a/127) : 1;
 * Wq[n,k] = clamp(rint(fl32(W[n,k] / w_scale[n])), -127, 127)   (IEEE division, ties to even).
 * W: [N,K] of dtype `wt` (fp32 or bf16).  Wq: int8 [N,K].  w_scale: fp32 [N].            */
ARIA_API int aria_quantize_weights_int8(const void* W, int wt, int N, int K, int8_t* Wq, float* w_scale,
                               void* stream);

/* S0 -- int4 group quantisation (config C4; readings R3, R4, R7, R8).  Per group of `group`
 * (must be 32) consecutive k:  a = max |w|;  sg = fp16_rne(fl32(a/7)) (subnormals kept);
 * sg == 0 -> codes 0, else q = clamp(rint(fl32(w / float(sg))), -7, 7).
 * Wq4: uint8 [N,K/2], byte j of row n = (q[2j] & 0xF) | ((q[2j+1] & 0xF) << 4), 4-bit two's
 * complement (0x8 never produced).  g_scale: fp16 bit patterns [N,K/32].                   */
ARIA_API int aria_quantize_weights_int4(const void* W, int wt, int N, int K, int group, uint8_t* Wq4,
                               uint16_t* g_scale, void* stream);

/* S1 -- per-token dynamic activation quantisation ("quantizing activations
 * alongside weights"; configs C1-C3).  Same arithmetic as aria_quantize_weights_int8 with
 * rows = tokens.  X: [M,K] of dtype `xt`.  Xq: int8 [M,K].  x_scale: fp32 [M].             */
ARIA_API int aria_quantize_act_int8(const void* X, int xt, int M, int K, int8_t* Xq, float* x_scale,
                           void* stream);

/* S1+S2+S3 -- one W8A8 linear ("integer tensor cores"; configs C1-C3):
 *   Xq, sx = S1(X);  acc[m,n] = sum_k Xq[m,k] Wq[n,k]  (exact int32, tcgen05 kind::i8, TMEM);
 *   y = float(acc) * sx[m] * w_scale[n] + bias[n];  act == GELU_ERF: y = 0.5 y (1 + erf(y/sqrt2));
 *   Y = cast(y, yt).
 * bias: [N] of dtype `bt`, may be NULL.  ws: scratch of at least
 * aria_workspace_bytes(M, K, N, ARIA_W8A8) bytes (holds Xq and sx; the size covers the two
 * alternating buffers aria_denoiser_linears uses).                                           */
ARIA_API int aria_linear_w8a8(const void* X, int xt, int M, int K, const int8_t* Wq, const float* w_scale,
                     int N, const void* bias, int bt, int act, void* Y, int yt, void* ws,
                     size_t ws_bytes, void* stream);

/* The same W8A8 linear for callers that CANNOT ALLOCATE device memory and so have no `ws` to pass:
 *   - real-time threads (an audio callback of an on-device generator): cudaMalloc takes a
 *     process-wide lock, may synchronise the device and has no latency bound, so they never call it;
 *   - plug-ins inside a host or serving engine whose own pool already owns all GPU memory (cudaMalloc fails);
 *   - code handed raw device pointers by another runtime, with no allocator to ask.
 * The Xq / sx scratch is a fixed array of ARIA_STATIC_WS_BYTES inside the library's device image instead.  The
 * call allocates nothing: no cudaMalloc / cudaFree, no allocating library routine.  X, Wq, w_scale, bias and Y
 * are passed exactly as to aria_linear_w8a8 and the result is the same, bit for bit (same kernels, same launches).
 *  - Limit: round_up(M*K, 256) + round_up(4*M, 256) <= ARIA_STATIC_WS_BYTES (16 MiB: up to M = 2048 tokens at
 *    K = 6144, the largest linear of config C5).  A larger shape returns ARIA_ERR_WORKSPACE, nothing is enqueued
 *    and Y is not touched; use aria_linear_w8a8 with your own workspace there.  aria_static_ws_bytes() returns
 *    the limit of the library that is actually loaded.
 *  - Cost: every GPU on which this entry point has been called keeps the 16 MiB until the process exits.
 *  - First call on each device: looks up the array's device address (cudaGetSymbolAddress, which loads the
 *    module on that device; the address differs per GPU and is cached per device ordinal).  Make that first
 *    call with the device current and BEFORE starting any stream capture on it.
 *  - One array per device, shared by every call and every stream: two calls whose kernels may overlap on
 *    the GPU (different streams, no ordering between them) race on it and corrupt each other's codes.  Calls on
 *    one stream, or ordered by events, are safe.  The array keeps the previous call's bytes; nothing in it needs
 *    clearing, because S1 overwrites every code and scale the GEMM reads.                                       */
#define ARIA_STATIC_WS_BYTES (16u << 20)
ARIA_API int aria_linear_w8a8_static_ws(const void* X, int xt, int M, int K, const int8_t* Wq, const float* w_scale,
                                        int N, const void* bias, int bt, int act, void* Y, int yt, void* stream);
ARIA_API size_t aria_static_ws_bytes(void);

/* S2+S3 only -- the same linear for activations that are ALREADY quantised (a producer that
 * emitted int8 codes, or a caller reusing one S1 pass for several linears of the same input):
 * Xq int8 [M,K] and x_scale fp32 [M] as produced by aria_quantize_act_int8.  No workspace.     */
ARIA_API int aria_linear_w8a8_q(const int8_t* Xq, const float* x_scale, int M, int K, const int8_t* Wq,
                       const float* w_scale, int N, const void* bias, int bt, int act, void* Y,
                       int yt, void* stream);

/* S4 -- one W4A16 linear (config C4; reading R12):  w^[n,k] = bf16_rne(q[n,k] * sg[n,k/32])
 * dequantised on chip;  y = sum_k x[m,k] w^[n,k] (fp32 accumulate, tcgen05 kind::f16 bf16)
 * + bias[n]; optional GELU; Y = cast(y, yt).  X: bf16 [M,K].  Wq4/g_scale: canonical format
 * of aria_quantize_weights_int4.  bias: bf16 [N] or NULL.
 * ws: scratch for the split-K schedule that small-M shapes use to fill the GPU (fp32 partial sums +
 * tile counters, aria_workspace_bytes(M, K, N, ARIA_W4A16) bytes).  ws == NULL or a smaller ws is
 * accepted and selects the schedule WITHOUT split-K: same results within fp32 summation order,
 * but shapes with fewer than #SMs tiles (M <= 512 on a 6144 -> 1536 layer) then run several times
 * slower.  With split-K the kernel's CTAs wait on one another: see "Co-residency" below.          */
ARIA_API int aria_linear_w4a16(const void* X, int M, int K, const uint8_t* Wq4, const uint16_t* g_scale,
                      int group, int N, const void* bias, int act, void* Y, int yt, void* ws,
                      size_t ws_bytes, void* stream);

/* NEXT-1 -- one q8 weight-only ("W8A16") linear: PAPER.md L78, weights "compressed to 8-bit ...
 * integers (labelled q8)" with the arithmetic left in half precision; Table II col. q8 (L129-131).
 * Weights are the S0 int8 format of aria_quantize_weights_int8 (Wq int8 [N,K], w_scale fp32 [N]);
 * w^[n,k] = bf16(q[n,k] * w_scale[n]) dequantised on chip (the fp32 product rounded to bf16: equals the
 * definition's single rounding bf16_rne(q * sw) except when the fp32 rounding hits a bf16 tie, < 2^-16 of
 * the weights, by one ulp); y = sum_k x[m,k] w^[n,k] (fp32 accumulate, tcgen05 kind::f16 bf16) + bias[n];
 * optional GELU; Y = cast(y, yt).  X: bf16 [M,K].  bias: bf16 [N] or NULL.  ws: as aria_linear_w4a16
 * (aria_workspace_bytes(M, K, N, ARIA_W8A16)).                                                       */
ARIA_API int aria_linear_w8a16(const void* X, int M, int K, const int8_t* Wq, const float* w_scale, int N,
                               const void* bias, int act, void* Y, int yt, void* ws, size_t ws_bytes,
                               void* stream);

/* S5 -- one denoising step's stack of linears (PAPER.md L73 graph replay; config C5).
 * Layers run in array order on `stream`, each reading `in` [M,K] and writing `out` [M,N], both
 * of dtype `io` (bf16 or fp32; W4A16 requires bf16).  `in == NULL` chains the layer to the
 * previous layer's `out` (its N must equal this K).  mode W8A8: wq = int8 [N,K], w_scale = fp32
 * [N]; mode W4A16: wq = packed int4 [N,K/2], w_scale = fp16 bits [N,K/32]; mode W8A16: wq = int8 [N,K],
 * w_scale = fp32 [N], bf16 I/O.  bias has dtype `io`,
 * may be NULL.  Capturable: enqueue only.  Mode W8A8: the S1 pass of a layer whose input the
 * previous layer does not write is overlapped with that layer's GEMM (programmatic dependent
 * launch, two alternating Xq / sx buffers in `ws`); a layer whose output IS the next layer's input
 * (in == NULL, or in == the previous out) reduces the per-token absmax of what it stores in its own
 * epilogue, and the consumer's S1 pass only rounds (north_star: "activation-quantization pass fused
 * into the previous epilogue"); codes, scales and results are those of array order, bit for bit.   */
typedef struct {
    int K, N;
    int act; /* aria_act applied to this layer's output */
    const void* in;
    const void* wq;
    const void* w_scale;
    const void* bias;
    void* out;
} aria_layer;

ARIA_API int aria_denoiser_linears(const aria_layer* layers, int n_layers, int M, int mode, int io, void* ws,
                          size_t ws_bytes, void* stream);

/* S5 with a PLAN (SURVEY S8(b) "a plan variant that pre-encodes TMA tensor maps is allowed").
 * aria_stack_plan_create validates the list exactly like aria_denoiser_linears, copies it, and
 * ALLOCATES the plan's own device scratch (tensor maps, schedule, split-K partials, flags): it
 * may synchronise and is not capturable.  The plan keeps the layers' device pointers (weights,
 * scales, biases, in/out buffers), which must stay valid until aria_stack_plan_destroy.
 * aria_stack_plan_run only ENQUEUES one step on `stream` (capturable) and computes
 * the same linears in array order as aria_denoiser_linears, within the same tolerances (S4:
 * <= 2e-2 of max|y| against the definition with w^ = bf16_rne(q*sg) and with w^ = q*sg).
 *
 * For mode W4A16 with M <= 32, bf16 I/O, every K % 256 == 0, no output buffer overlapping another
 * output or an earlier input, and every input that touches an earlier output being exactly that
 * output, the step is ONE persistent weight-streaming kernel over all layers (HBM bound; layers
 * whose input is not an earlier layer's output may overlap).  Operand format there:
 *  - fp16 (aria_stack_plan_is_streaming == 1): w^ = fp16_rn((q + 8) * sg) - 8 * sg (offset-binary code
 *    scaled and rounded to fp16; the zero point is subtracted exactly by an extra tensor-core k-step)
 *    and the bf16 activations enter the same tcgen05 kind::f16 MMA converted to fp16.  Chosen at plan
 *    creation iff every group scale satisfies 1024 * sg <= 65504 (the scales are scanned once).  The
 *    ACTIVATIONS are checked on the device in every run: if any |x| or any 32-k group sum of x exceeds
 *    65504 (external inputs and chained outputs alike), or a whole input tensor has 0 < max|x| < 2^-7
 *    (fp16 subnormals would cost relative precision), the run raises a device flag and a second,
 *    otherwise empty launch recomputes the WHOLE list with exact bf16 operands (next item).  So every
 *    input aria_linear_w4a16 accepts gives results within the tolerances above; out-of-range inputs
 *    only cost time.  aria_stack_plan_fallback_fired reports whether the last run did that.
 *  - bf16 (aria_stack_plan_is_streaming == 2): w^ = bf16_rne(q * sg) and bf16 activations, exactly as
 *    aria_linear_w4a16.  Chosen when a scale fails the test above.
 * Any other list runs the per-layer path (aria_stack_plan_is_streaming == 0).  A plan's scratch serves
 * ONE step at a time: do not run the same plan concurrently on two streams.
 *
 * Co-residency.  The stream kernel's CTAs (and those of aria_linear_w4a16 with split-K) wait on
 * completion counters written by other CTAs of the same grid.  Every launch of the stream kernel -- the
 * fp16 launch AND the bf16 fallback launch that follows it in stream order -- is therefore a COOPERATIVE
 * launch of at most one CTA per SM, and so is every split-K launch of aria_linear_w4a16 /
 * aria_linear_w8a16: the grid starts only when all of it is resident (SMs held by another kernel delay
 * it, they cannot deadlock it), and a grid the device can never hold at once fails with ARIA_ERR_CUDA.
 * One step of a streaming plan enqueues one memset and one (bf16 plans) or two (fp16 plans) kernels.
 *
 * aria_stack_plan_fallback_fired: SYNCHRONOUS (copies one word from the device after the stream's work
 * has been synchronised by the caller); *fired = 0 if the last run stayed in the fp16 domain, else a
 * bit mask (1 = a value above the fp16 range, 2 = an input tensor below 2^-7).  Always 0 for plans that
 * do not use fp16 operands.                                                                        */
typedef struct aria_stack_plan aria_stack_plan;
ARIA_API int aria_stack_plan_create(const aria_layer* layers, int n_layers, int M, int mode, int io,
                                    aria_stack_plan** plan);
ARIA_API int aria_stack_plan_run(const aria_stack_plan* plan, void* stream);
ARIA_API int aria_stack_plan_is_streaming(const aria_stack_plan* plan);
ARIA_API int aria_stack_plan_fallback_fired(const aria_stack_plan* plan, int* fired);
ARIA_API void aria_stack_plan_destroy(aria_stack_plan* plan);

/* Same stack, but `in` / `out` of every layer are HOST pointers (pinned memory recommended):
 * each layer's input is copied host->device into `ws`, the layer runs, and its output is
 * copied device->host.  The copies run on two library-owned copy streams chained to `stream` by
 * events (double-buffered staging in `ws`), so the H2D / D2H transfers of neighbouring layers
 * overlap each other and the compute; the call returns after synchronising all three streams
 * (the copy streams are per device and shared by all calls: one _host call at a time per device).  Weights, scales and
 * biases stay DEVICE pointers (the compressed copy is resident).  ws must hold
 * aria_workspace_bytes_host(...) bytes.  Not capturable.                                    */
ARIA_API int aria_denoiser_linears_host(const aria_layer* layers, int n_layers, int M, int mode, int io,
                               void* ws, size_t ws_bytes, void* stream);

/* Scratch sizes in bytes (0 on invalid arguments). */
ARIA_API size_t aria_workspace_bytes(int M, int maxK, int maxN, int mode);
ARIA_API size_t aria_workspace_bytes_host(int M, int maxK, int maxN, int mode, int io);

/* Static string for a status code. */
ARIA_API const char* aria_status_string(int status);

/* Test hook for the bit-exact accumulator gate: acc[m,n] = sum_k Xq[m,k] Wq[n,k] as int32
 * [M,N], computed by the same tcgen05 kind::i8 kernel as aria_linear_w8a8.                   */
ARIA_API int aria_gemm_i8_i32(const int8_t* Xq, const int8_t* Wq, int M, int N, int K, int32_t* acc,
                     void* stream);

/* NEXT-3 -- in-graph activation steering of the residual stream, in place (eq. 2,
 * L94-98; projection variant L192 / L248).  H: [M,D] of dtype `ht` (a DiT block's output, row = token),
 * d: fp32 [D] direction (unit norm by eq. 1; not checked), strength: DEVICE pointer to one fp32 read at
 * run time -- a captured graph is replayed with a new strength without re-capture (L77).
 *   op ARIA_STEER_ADD:      h[t,:] <- h[t,:] + alpha * hbar_norm * d[:]     (eq. 2; hbar_norm = "the mean
 *                            baseline residual norm" of that block, a host scalar fixed at capture)
 *   op ARIA_STEER_PROJECT:  c_t = h[t,:] . d;  h[t,:] <- h[t,:] + beta * c_t * d[:]   (beta < 0 removes,
 *                            beta > 0 amplifies the component already present; hbar_norm ignored)
 * *strength == 0 leaves H untouched, bit for bit ("at strength 0 the output is bit-identical to the base
 * model", L77).  D % 8 == 0; fp32 arithmetic, one rounding to `ht`.  Enqueue only, capturable.        */
ARIA_API int aria_steer(void* H, int ht, int M, int D, const float* d, const float* strength, float hbar_norm,
                        int op, void* stream);

/* NEXT-2 ("producers/consumers around the linears") -- the two pieces of a DiT block that
 * sit between the quantized linears ("the diffusion transformer (DiT)"; L278 "the transformer's full
 * self-attention ... a fused attention kernel (FlashAttention-class) ... is the open lever"; L224).  The paper
 * gives neither formula; the textbook definitions are taken (R20-R22).
 *
 * aria_norm_quantize_act_int8 -- normalisation fused with S1: per token row,
 *   norm ARIA_NORM_LAYER:  mu = mean_k x;  var = mean_k (x - mu)^2;  n = (x - mu) / sqrt(var + eps) * gamma + beta
 *   norm ARIA_NORM_RMS:    n = x / sqrt(mean_k x^2 + eps) * gamma + beta
 *   n is rounded once to dtype `xt` (the tensor an unfused norm kernel would store), then S1 exactly as
 *   aria_quantize_act_int8:  x_scale = max|n| / 127 (1 for a zero row), Xq = clamp(rint(n / x_scale), +-127).
 * X: [M,K] of dtype `xt`; gamma: fp32 [K]; beta: fp32 [K] or NULL; eps >= 0.  Xq int8 [M,K], x_scale fp32 [M]
 * feed aria_linear_w8a8_q.  Xn: [M,K] of dtype `xt`, or NULL -- the normalised tensor is written only on request
 * (the fused path reads X once and writes one byte per element).  fp32 arithmetic (two-pass variance); codes and
 * scales are bit-identical to aria_quantize_act_int8 applied to Xn.  K % 32 == 0, K <= 24576.  Enqueue only.   */
ARIA_API int aria_norm_quantize_act_int8(const void* X, int xt, int M, int K, const float* gamma, const float* beta,
                                         int norm, float eps, void* Xn, int8_t* Xq, float* x_scale, void* stream);

/* aria_attention -- full (unmasked, non-causal) multi-head self-attention on the fused QKV projection's output:
 *   per sequence b, head h, query i:  s_j = scale * q_i . k_j;  p = softmax_j(s);  o_i = sum_j p_j v_j.
 * QKV: bf16 [B*S, 3*H*Dh], row = token b*S + i, columns [ q (H*Dh) | k (H*Dh) | v (H*Dh) ], head h at columns
 * h*Dh .. h*Dh+Dh-1 of its third.  O: bf16 [B*S, H*Dh] (the out-projection's input).  Dh must be 64; scale > 0
 * (1/sqrt(Dh) = 0.125 for the usual choice).  Scores and the output accumulate in fp32 on the tensor cores
 * (tcgen05 kind::f16, bf16 operands); the probabilities enter the second product rounded to bf16
 * (FlashAttention-class; R22 derives the tolerance).  row_absmax: NULL, or fp32 [B*S] that the caller
 * has ZEROED: the kernel reduces max_d |O[t, :]| over all heads into it (atomicMax on the stored bf16 values) --
 * the first half of a fused S1 for a W8A8 out-projection, finished by aria_round_act_int8.  Enqueue only.   */
ARIA_API int aria_attention(const void* QKV, int B, int S, int H, int Dh, float scale, void* O, float* row_absmax,
                            void* stream);

/* Second half of a fused S1 (north_star "activation-quantization pass fused into the previous epilogue"): the
 * per-token max|x| is already known (reduced by the kernel that produced X, e.g. aria_attention), so the pass
 * only rounds:  x_scale = absmax / 127 (1 if 0), Xq = clamp(rint(x / x_scale), +-127).  Bit-identical to
 * aria_quantize_act_int8 when absmax[m] == max_k |X[m,k]|.  absmax: fp32 [M]; clear != 0 resets absmax[m] to 0
 * once it has been read, so the buffer is ready for the next producer without a memset in the captured step.
 * A wrong absmax[m] gives the scale it implies, never a wrapped code: values above it saturate at +-127 (the
 * kernel compares what it holds against absmax[m]), and a NaN absmax[m] is treated as scale 1.               */
ARIA_API int aria_round_act_int8(const void* X, int xt, int M, int K, float* absmax, int clear, int8_t* Xq,
                                 float* x_scale, void* stream);

/* Measurement helper, NOT part of the hot path (SURVEY.md S7 hard part 2 / S8(d): "measure an int8
 * peak on the box first: a plain back-to-back tcgen05.mma kind::i8 issue loop with no memory
 * traffic"): every SM (ctas = 1) or SM pair (ctas = 2, cta_group::2) issues `iters` groups of four
 * 128*ctas x 256 x K tcgen05.mma (K = 32 for kind 0 = kind::i8 s8 x s8 -> s32, K = 16 for kind 1 =
 * kind::f16 bf16 x bf16 -> f32) on pseudo-random operands resident in shared memory, nothing loaded or
 * stored meanwhile.  The launch is repeated back to back for `seconds` (0: once after a warm-up) and
 * the LAST launch is reported: out[0] = operations per second (2 MNK per MMA, CUDA events), out[1] =
 * SM clock in MHz inside the loop (clock64 / globaltimer), out[2] = SM cycles per tcgen05.mma, out[3] =
 * launches made.  SYNCHRONOUS; allocates and frees a few hundred bytes of device memory.            */
ARIA_API int aria_tensor_peak(int kind, int ctas, int iters, double seconds, double* out, void* stream);

/* Host-only introspection of the launch plans (no device needed; used by the tests to prove that
 * every compiled tile variant is reached): the (BN, CTAS) tile of the W8A8 GEMM for an [M,N] output on
 * a device with `sms` SMs (BN in {64,128,192,256} output channels, CTAS = 2: tcgen05 cta_group::2
 * pairs computing 256 x BN), and the (token tile TT in {32,64,128,192,256}, split-K factor) of the
 * W4A16 / W8A16 GEMM.                                                                              */
ARIA_API int aria_w8a8_tile_plan(int M, int N, int sms, int* bn, int* ctas);
ARIA_API int aria_w4a16_tile_plan(int M, int N, int K, int sms, int* tt, int* splits);

/* Library build id ("aria-b200 <version> sm_100a"). */
ARIA_API const char* aria_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ARIA_H_ */
