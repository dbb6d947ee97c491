/*
 * twq.h -- C ABI of the B200 (sm_100a) TwinQuant dual-component 4-bit linear layer.
 *
 *     Y = deq( Q4(X*T) * R4^T ) + (X*L1)*L2
 *
 * PAPER.md = arxiv 2606.01556 (TwinQuant).  The operation is the inference form of
 * Eq. 3 (section 2): a 4-bit activation x 4-bit weight residual GEMM
 * (Eq. 2) with group scales along the reduction axis (L193, section 5.1) plus
 * a two-stage rank-r product, merged by one epilogue and one store (L179-181,
 * section 4.3).  The low-rank branch is the high-precision (FP16 factor) form that
 * BASELINE.json's north_star fixes ("keeps the low-rank path in FP16").
 *
 * Conventions
 *   - All data pointers are DEVICE pointers (cudaMalloc / torch CUDA tensors).  The
 *     library never allocates, frees or copies user buffers and never synchronises.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *     Every call is asynchronous with respect to the host.
 *   - All matrices are row-major.  M tokens, K in-features, N out-features,
 *     G group size along K, ng = K/G groups, r rank.
 *   - Errors are returned as twq_status; nothing throws or aborts.  Arguments are
 *     validated BEFORE any CUDA call, so invalid arguments are reported without a GPU.
 *   - Non-finite inputs give unspecified values, never a fault.
 *   - There is no CPU fallback: without an sm_100 device the compute entry points
 *     return TWQ_ERR_UNSUPPORTED / TWQ_ERR_CUDA.
 *   - One device per call: the current CUDA device (cudaSetDevice) at the time of the call.  Per-device facts and
 *     function attributes are cached per device; plans and TMA descriptors are cached per host thread.  Calls from
 *     several host threads are safe as long as two calls that share a workspace do not run concurrently.
 *
 * Stream-ordering contract (programmatic dependent launch)
 *   twq_quantize_act and twq_dual_linear are launched with the programmatic-stream-serialization attribute: a
 *   kernel may START while its stream predecessor is still running.  What each kernel does before / after its
 *   griddepcontrol.wait (= "the predecessor has completed and its writes are visible"):
 *     before the wait : reads of `packed` only (weights, scales, low-rank factors).  `packed` must therefore not be
 *                       written by the kernel that immediately precedes the call in the stream (pack once, offline).
 *     after the wait  : every read of X, Xq, sx and every write of Y, dbg_P, ws.  A predecessor -- a kernel of this
 *                       library or the caller's own, PDL-aware or not -- may produce X / Xq / sx up to its last
 *                       instruction.
 *   twq_quantize_act waits for its predecessor before it touches memory and only then lets its successor start.
 */
#ifndef TWQ_H_
#define TWQ_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    TWQ_OK = 0,
    TWQ_ERR_INVALID_ARG = 1,  /* null pointer, bad shape, bad alignment, buffer too small */
    TWQ_ERR_UNSUPPORTED = 2,  /* device is not sm_100, or a shape outside the built kernels */
    TWQ_ERR_WORKSPACE = 3,    /* ws_bytes < twq_workspace_bytes(...) */
    TWQ_ERR_CUDA = 4          /* a CUDA runtime / driver call or the launch failed */
} twq_status;

typedef enum { TWQ_OUT_BF16 = 0, TWQ_OUT_FP16 = 1, TWQ_OUT_FP32 = 2 } twq_out_dtype;

/* Shape rules shared by every entry point (checked, TWQ_ERR_INVALID_ARG otherwise):
 *   M >= 1; G in {64,128}; K >= G, K % G == 0; N >= 16, N % 16 == 0;
 *   0 <= r <= 256, r % 16 == 0 (r = 0: plain W4A4, no low-rank branch);
 *   pointers 16-byte aligned; leading dimensions >= row length and a multiple of 8 elements.
 */

/* Human-readable name of a status code (static string, never NULL). */
const char* twq_status_string(twq_status s);

/* ---------------------------------------------------------------------------
 * twq_packed_bytes -- size in bytes of the opaque kernel-native weight blob that
 * twq_pack_weights writes for one layer (0 if the shape is invalid).
 * Contents ("pre-processed offline"; L193 groups of G along K), each section 256-byte aligned:
 * 4-bit residual codes tiled [N/8][K/G][8][G/2] (N*K/2 bytes), FP16 group scales tiled the same way [N/8][K/G][8],
 * L1^T [r,K] FP16 (tcgen05 kernel), L1 in 32-wide K slabs [K/32][r][32] FP16 (small-batch kernel), L2^T [N,r] FP16.
 */
size_t twq_packed_bytes(int N, int K, int r, int G);

/* ---------------------------------------------------------------------------
 * twq_pack_weights -- offline re-layout of one layer's weights (step a0).
 *   Rq  [N,K]   int8   residual 4-bit codes, each in [-8,7] (two's complement INT4,
 *                      symmetric quantizer of Eq. 1; values outside
 *                      [-8,7] are truncated to their low 4 bits)
 *   sw  [N,K/G] fp16   residual group scales (one per G contiguous k, per out channel)
 *   L1  [K,r]   fp16   low-rank factor 1 (may be NULL iff r == 0)
 *   L2  [r,N]   fp16   low-rank factor 2 (may be NULL iff r == 0)
 *   packed      out    blob of twq_packed_bytes(N,K,r,G) bytes, 256-byte aligned
 * The packed 4-bit interchange layout inside the blob is R4[N,K/2]: byte j of a row
 * holds code k=2j in its low nibble and k=2j+1 in its high nibble.
 * Returns TWQ_ERR_INVALID_ARG if packed_bytes is too small.
 */
twq_status twq_pack_weights(const int8_t* Rq, const void* sw, const void* L1, const void* L2,
                            int N, int K, int r, int G,
                            void* packed, size_t packed_bytes, void* stream);

/* ---------------------------------------------------------------------------
 * twq_quantize_act -- online per-token group quantizer (steps a1-a2).
 * PAPER.md Eq. 1 (L43-47): Q_X = round(X/s_X), s_X = max|X|/q_max, q_max = 7;
 * activation-side diagonal transform X*diag(lambda)^-1 (L54-58); groups of G (L193).
 * Exact FP32 operation order (this order IS the specification; reading R8):
 *     x~  = (float)X[m,k] * tinv[k]       (one RN multiply; skipped when tinv == NULL)
 *     a   = max(max_{k in g} |x~|, 2^-30)
 *     s   = a / 7.0f  (RN divide)   -> sx[m,g]
 *     inv = 1.0f / s  (RN divide)
 *     q   = clamp(rint_even(x~ * inv), -7, 7)
 *   X    [M,ldx] bf16  activations (ldx >= K elements)
 *   tinv [K]     fp32  diagonal of T (1/lambda), or NULL for T = identity
 *   Xq   [M,K/2] u8    out: packed codes, low nibble = even k, two's complement
 *   sx   [M,K/G] fp32  out: group scales
 */
twq_status twq_quantize_act(const void* X, int M, int K, int ldx, const float* tinv, int G,
                            uint8_t* Xq, float* sx, void* stream);

/* Bytes of scratch twq_dual_linear needs for this shape (0 is a legal answer). */
size_t twq_workspace_bytes(int M, int N, int K, int r, int G);

/* ---------------------------------------------------------------------------
 * twq_dual_linear -- the fused dual-branch layer (steps a3-a7), ONE kernel launch.
 *   residual : P[m,g,n] = sum_{k in g} qx[m,k]*qw[n,k]   exact int32   (Eq. 2; L177)
 *              Yres     = sum_g sx[m,g]*sw[n,g]*P[m,g,n]  FP32          (L181 "folds the scale factors")
 *   low-rank : H = X*L1 (FP32 accumulate, kept on chip), Ylr = H*L2    (Eq. 3; L177-179)
 *              The 16-bit tensor-core product needs one operand format and L1 is FP16, so X (BF16) is rewritten to
 *              FP16 on chip: exact for 2^-14 <= |x| <= 65504, SATURATING at +-65504 above, and losing bits below
 *              2^-14 (flush to zero below 2^-24).  H is rounded once to FP16 (saturating) as the operand of the
 *              second product (readings R2, R12).  The residual branch reads X through Xq / sx only.
 *   epilogue : Y = round_out(Yres + Ylr), one store                    (L181)
 *   X      [M,ldx] bf16     raw activations (read by the low-rank branch; may be NULL iff r == 0)
 *   Xq,sx                   outputs of twq_quantize_act for the same X
 *   packed                  blob written by twq_pack_weights for (N,K,r,G)
 *   Y      [M,ldy]          out, dtype ydt (ldy >= N elements)
 *   ws, ws_bytes            scratch of at least twq_workspace_bytes(...) bytes, 256-byte aligned (may be
 *                           NULL when that is 0).  Only calls with few output tiles beyond the small-batch
 *                           kernel (64 < M, roughly M*N < 0.5 M outputs) need it: split-K partial sums of Y
 *                           and tile counters.  Small batches (M <= 64) and prefill-shaped calls need none,
 *                           and the on-chip intermediate H never passes through it.  The caller zero-fills it
 *                           ONCE after allocation; every call leaves the counters zero again, so it can be
 *                           reused without clearing -- by calls on ONE stream at a time (two calls that
 *                           share a workspace must not run concurrently).  Calls that use a workspace are
 *                           launched cooperatively (their CTAs wait for one another): the driver refuses the
 *                           launch (TWQ_ERR_CUDA) rather than let it hang if the grid cannot be co-resident.
 *   dbg_P  [M,K/G,N] int32  NULL, or receives the integer group accumulators P taken from the
 *                           same tensor-core path that feeds Y (parity evidence; slows the call)
 */
twq_status twq_dual_linear(const void* X, int ldx, const uint8_t* Xq, const float* sx,
                           const void* packed, int M, int N, int K, int r, int G,
                           void* Y, twq_out_dtype ydt, int ldy,
                           void* ws, size_t ws_bytes, int32_t* dbg_P, void* stream);

/* ---------------------------------------------------------------------------
 * twq_dual_linear_x -- the whole hot path (steps a1-a7) from the raw activations: quantizer + fused layer.
 * the kernel "quantizes the input activation tile once and reuses it for both components"; here the
 * quantized tile is produced once per thread-block cluster and reused by every CTA and channel tile of the call.
 *   M <= 64 (the small-batch kernel, when its shared-memory plan fits): ONE kernel launch; codes and scales never
 *     leave the chip unless Xq_out / sx_out ask for a copy.  Same FP32 operation order as twq_quantize_act: the codes
 *     and scales (and therefore P and Y) are bit-identical to the two-call path.
 *   otherwise: twq_quantize_act followed by twq_dual_linear (two launches), the quantizer's outputs going to
 *     Xq_out / sx_out if given, else to the front of the workspace.
 *   X      [M,ldx] bf16     raw activations (required)
 *   tinv   [K] fp32         diagonal of the activation-side transform, or NULL for identity
 *   Xq_out [M,K/2] u8       NULL, or receives the packed codes;  sx_out [M,K/G] fp32: NULL, or receives the scales
 *   ws, ws_bytes            at least twq_workspace_bytes_x(...) bytes, 256-byte aligned, zero-filled once (as for
 *                           twq_dual_linear); 0 bytes for the one-launch shapes
 * Other arguments, stream ordering and errors as for twq_dual_linear.
 */
size_t twq_workspace_bytes_x(int M, int N, int K, int r, int G);
twq_status twq_dual_linear_x(const void* X, int ldx, const float* tinv, const void* packed,
                             int M, int N, int K, int r, int G,
                             void* Y, twq_out_dtype ydt, int ldy,
                             void* ws, size_t ws_bytes, uint8_t* Xq_out, float* sx_out,
                             int32_t* dbg_P, void* stream);

/* ---------------------------------------------------------------------------
 * The paper's own, fully 4-bit low-rank branch (section 4.3, Eq. 4):
 *     Y = Q(X) [ Q(U) Q(V) + Q(R) ],   U = L1^T and V = L2^T both 4-bit with group scales.
 *   stage 1  : H[m,j]  = sum_g sx[m,g]*su[j,g]*P1[m,g,j],  P1 = sum_{k in g} qx[m,k]*qu[j,k] (exact int32).  The branch
 *              multiplies the SAME quantized activation tile as the residual (L179); H is summed in FP32 and never
 *              leaves the chip (L177-179).
 *   re-quantization on the fly (L181: "estimating an intermediate scale s_H from the INT32 accumulator and re-quantizing
 *              on the fly"): one scale per token and per group of gr consecutive rank indices, gr = r for r <= 128,
 *              else 128 (so r <= 128 or r == 256).  The quantizer of Eq. 1 in the FP32 operation order of
 *              twq_quantize_act:  s_H = max(amax|H|, 2^-30) / 7;  Q_H = clamp(rint(H * (1 / s_H)), -7, 7), packed
 *              4-bit in shared memory.
 *   stage 2  : Ylr[m,n] = sum_h s_H[m,h]*sv[n,h]*P2[m,h,n],  P2 = sum_{j in h} Q_H[m,j]*qv[n,j] (exact int32)
 *   epilogue : Y = round_out(Yres + Ylr), one store (L181); Yres as in twq_dual_linear.
 * DESIGN.md readings R18-R22.  The quantizer, both branches and the epilogue are ONE launch per slab of at most 64 tokens
 * (32 or 16 where the quantized activation tile of 64 tokens does not fit in shared memory: K > 4096 roughly).  Larger M:
 * consecutive slabs, one launch each; a tcgen05 path for prefill-shaped M is not written yet.
 *
 * twq_pack_weights_q4lr -- offline re-layout (step a0) into an opaque blob of twq_packed_bytes_q4lr(N,K,r,G) bytes:
 *   Rq  [N,K] int8, sw [N,K/G] fp16   the residual, as for twq_pack_weights
 *   Uq  [r,K] int8 codes in [-8,7],  su [r,K/G] fp16     groups of G along K
 *   Vq  [N,r] int8 codes in [-8,7],  sv [N,r/gr] fp16    groups of gr along r
 *   r: a multiple of 16 in [16,128], or 256.  All pointers device, 16-byte aligned; packed 256-byte aligned.
 *
 * twq_dual_linear_q4lr_x -- the whole path from the raw activations.
 *   X, ldx, tinv, Y, ydt, ldy, Xq_out, sx_out, dbg_P    as for twq_dual_linear_x (no workspace is ever needed)
 *   packed                  blob written by twq_pack_weights_q4lr for (N,K,r,G)
 *   dbg_H  [M,r] fp32       NULL, or receives H as the re-quantizer saw it
 *   dbg_QH [M,r] int8       NULL, or receives the codes Q_H;  dbg_sH [M,r/gr] fp32: NULL, or receives s_H
 *                           (parity evidence taken from the path that feeds Y; slows the call)
 * Returns TWQ_ERR_UNSUPPORTED when even a 16-token slab's shared-memory plan does not fit: the resident quantized tile
 * (16 tokens x K/2 bytes), the FP32 H and the weight rings share 227 KB, which excludes e.g. K = 25600 at r = 256 and
 * K = 8192 with N = 28672 at r = 256 (32 channel tiles per CTA).  Nothing is launched in that case.
 * Stream ordering and the other errors as for twq_dual_linear.
 */
size_t twq_packed_bytes_q4lr(int N, int K, int r, int G);
twq_status twq_pack_weights_q4lr(const int8_t* Rq, const void* sw, const int8_t* Uq, const void* su,
                                 const int8_t* Vq, const void* sv, int N, int K, int r, int G,
                                 void* packed, size_t packed_bytes, void* stream);
twq_status twq_dual_linear_q4lr_x(const void* X, int ldx, const float* tinv, const void* packed,
                                  int M, int N, int K, int r, int G,
                                  void* Y, twq_out_dtype ydt, int ldy,
                                  uint8_t* Xq_out, float* sx_out, int32_t* dbg_P,
                                  float* dbg_H, int8_t* dbg_QH, float* dbg_sH, void* stream);

/* ---------------------------------------------------------------------------
 * twq_dual_linear_noalloc -- twq_dual_linear for callers that cannot allocate device memory (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): no workspace argument.  The scratch that the few
 * shapes with a workspace need (64 < M with few output tiles, see twq_dual_linear) lives in a static device array of
 * TWQ_NOALLOC_MAX_WS bytes inside the library -- every GPU that loads the library holds these 8.5 MiB until the process
 * exits; it covers every workspace shape of BASELINE.json's configs (largest: 8 MiB + 256 B), while the largest workspace the
 * planner can ask for at all is about 9.5 MB (a few hundred tokens, few channels).  The call allocates nothing (no
 * cudaMalloc / cudaFree, no allocating library routine) and issues one small memset on `stream` (the tile counters) in
 * front of the kernel when the shape uses scratch.
 *   Arguments as for twq_dual_linear, without ws / ws_bytes / dbg_P.  Results are those of twq_dual_linear.
 *   TWQ_ERR_WORKSPACE  the shape needs more than TWQ_NOALLOC_MAX_WS bytes (twq_workspace_bytes(...) says how many):
 *                      nothing is launched; use twq_dual_linear with a caller workspace.
 *   All calls on a device share the one array: two calls that may overlap on the GPU (different streams without a
 *   dependency between them) race on it and must not be issued; calls ordered by a stream or by events are fine.
 */
#define TWQ_NOALLOC_MAX_WS (8u * 1024u * 1024u + 512u * 1024u)
size_t twq_noalloc_max_workspace(void);
twq_status twq_dual_linear_noalloc(const void* X, int ldx, const uint8_t* Xq, const float* sx,
                                   const void* packed, int M, int N, int K, int r, int G,
                                   void* Y, twq_out_dtype ydt, int ldy, void* stream);

/* Number of kernel launches the last successful twq_dual_linear(_x) / twq_quantize_act /
 * twq_pack_weights call on this thread issued (bench.py's gpu_launches accounting). */
int twq_last_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* TWQ_H_ */
