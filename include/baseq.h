/* libbaseq -- C ABI of the BASE-Q W4A4 linear hot path for NVIDIA B200 (sm_100a).
 *
 * The operation is the online quantised linear layer of BASE-Q (arxiv 2506.15689):
 *
 *   Y = Q_w(W s R) . Q_a( s^a R^-1 s^-1 x - b^c ) + (W R b^c + b)          (Eq. 15)
 *
 * split the way the paper deploys it (Fig. 6): a fused quantisation kernel
 * (online Hadamard, scale, bias, per-token int4), an int4 x int4 -> int32 GEMM, and a fused
 * de-quantisation (both scales + fused bias).  P:n below = PAPER.md line n, S:n = SPEC.md
 * line n, C-n = the readings listed in DESIGN.md.
 *
 * Conventions (all entry points)
 *  - plain C, no torch / C++ types; every pointer is a DEVICE pointer owned by the caller
 *    unless the argument name ends in _host;
 *  - the library never allocates, frees or synchronises (baseq_sync_status is the one call that
 *    blocks), and keeps no reference to any argument after the call returns; all work is enqueued
 *    on `stream` (a cudaStream_t passed as void*; NULL = the legacy default stream);
 *  - arguments are validated on the host before anything is launched or copied -- a call that
 *    returns an error has enqueued nothing; every call returns a baseq_status_t (no exceptions,
 *    no errno, nothing printed);
 *  - any host thread may call, with any device current (one process may drive several GPUs);
 *  - there is no CPU fallback: on a device that is not compute capability 10.x every compute
 *    entry point returns BASEQ_ERR_UNSUPPORTED;
 *  - CUDA launch failures are returned as BASEQ_ERR_CUDA by the enqueueing call;
 *    asynchronous faults surface at the caller's next synchronisation;
 *  - non-finite activations: behaviour unspecified (S:32 rejects them at construction).
 *
 * Shape rules (BASEQ_ERR_SHAPE): T >= 1 (empty input is an error, S:57 / S:225),
 * K % 128 == 0 and 128 <= K <= 32768 in EVERY entry point (a whole row stays in one CTA; the GEMM's
 * raw accumulator 256 * acc stays inside int32), N % 8 == 0 and N >= 8.  T need not be a multiple
 * of any tile.
 * Alignment (BASEQ_ERR_ALIGN): x, codes, y, packed blob 16-byte aligned (blob: 128);
 * ldx >= K, ldx % 8 == 0; ldy >= N, ldy % 8 == 0.
 */
#ifndef BASEQ_H_
#define BASEQ_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define BASEQ_API __attribute__((visibility("default")))
#else
#define BASEQ_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  BASEQ_OK = 0,
  BASEQ_ERR_NULL = 1,        /* a required pointer is NULL                               */
  BASEQ_ERR_SHAPE = 2,       /* T/K/N violate the shape rules above                      */
  BASEQ_ERR_ALIGN = 3,       /* pointer or leading-dimension alignment                   */
  BASEQ_ERR_PARAM = 4,       /* alpha / gamma / had_block out of range                   */
  BASEQ_ERR_WORKSPACE = 5,   /* workspace / scratch too small; from baseq_sync_status: a
                                packed blob did not match the (N, K) of a GEMM call       */
  BASEQ_ERR_UNSUPPORTED = 6, /* not an sm_100 device, or a combination that is not built */
  BASEQ_ERR_CUDA = 7         /* a CUDA runtime / driver call failed                      */
} baseq_status_t;

/* Static string for a status code. */
BASEQ_API const char* baseq_status_string(baseq_status_t s);
/* Library version (integer, increases with ABI changes). */
BASEQ_API int baseq_version(void);
/* The one blocking call: synchronises `stream`, then reads and clears the current device's status
 * word.  A packed blob lives in device memory, so no enqueue-only call can compare its header
 * with the (N, K) it is given; the GEMM kernels do (magic, N, K -- written by baseq_pack_weights):
 * on a mismatch the kernel does no work, writes nothing, and raises the word.  Returns
 * BASEQ_ERR_WORKSPACE if any GEMM of this device since the last call found such a blob,
 * BASEQ_ERR_CUDA if the synchronisation reports an asynchronous fault, else BASEQ_OK. */
BASEQ_API baseq_status_t baseq_sync_status(void* stream);

/* The per-quantizer parameters of Eq. 15 / BlockParams.
 *   u_k = g_k * h_k - b_k,  h = block-Hadamard(x) or x,  g_k = sa ? sa[k] : gamma    (C-1, C-2)
 *   s_t = max((alpha * max_k |u_k|) / 7, 1e-12)                                       (C-7, C-8, C-10)
 *   q_k = clamp(rne(u_k * (1 / s_t)), -8, 7)     product exact, one rounding     (C-5, C-6, C-17)
 * every line one correctly rounded fp32 operation. */
typedef struct {
  float alpha;      /* clip ratio, 0 < alpha <= 1, else BASEQ_ERR_PARAM; below
                       2^-16 a plain (slow) kernel takes over that clamps before it rounds -- the
                       same codes -- and baseq_quantize_act_tc returns BASEQ_ERR_UNSUPPORTED          */
  float gamma;      /* scalar s^a, used iff sa == NULL; must be finite and > 0                      */
  const float* sa;  /* [K] per-channel s^a, already divided by the paired scale s; or NULL          */
  const float* b;   /* [K] correction bias b^c in the scaled (and rotated) domain; NULL = 0         */
  int had_block;    /* 0 = none; else online Hadamard block size: a power of two in
                       [2, 256] dividing K, else BASEQ_ERR_PARAM                            */
} baseq_act_params_t;

/* ---- offline weight packer (P:241 per-channel symmetric int4; "fused bias" of Eq. 14) ----
 * Re-tiles int4 weights into the blob the GEMM streams with bulk-TMA copies, stores s_w and
 * computes the fused bias  fb[n] = s_w[n] * sum_k qw[n,k] * b[k] + layer_bias[n]  (fp64
 * accumulation, C-3: qw are the very integers the GEMM multiplies).
 *   w_nibbles   [N, K/2] bytes row-major, byte j of row n = (qw[n,2j] & 15) | ((qw[n,2j+1] & 15) << 4)
 *   w_scale     [N] fp32 per-output-channel step size s_w
 *   b           [K] fp32 or NULL (then fb = layer_bias)
 *   layer_bias  [N] fp32 or NULL
 *   packed_out  caller buffer of baseq_packed_weight_bytes(N, K) bytes, 128-byte aligned
 *   fused_bias_out  optional [N] copy of fb for inspection, or NULL
 * The blob is opaque, position independent (may be copied) and a pure function of the inputs.
 * Ordering: the GEMM kernels are enqueued with the programmatic-dependent-launch attribute and
 * read the blob's header and weight boxes BEFORE they wait for the preceding kernel of the stream.
 * Blobs written by baseq_pack_weights are safe by construction (header and boxes are followed by
 * a fully serialised kernel boundary inside the call; s_w / fb / wsum, which its last kernel and
 * baseq_set_fused_bias write, are read after the wait).  A blob the caller copies must be
 * complete in stream order through a memcpy or a plain kernel launch, not through a kernel that
 * triggers its dependents early. */
BASEQ_API size_t baseq_packed_weight_bytes(int N, int K);
BASEQ_API baseq_status_t baseq_pack_weights(const uint8_t* w_nibbles, const float* w_scale, const float* b,
                                  const float* layer_bias, int N, int K, void* packed_out,
                                  float* fused_bias_out, void* stream);
/* Replace the blob's fused bias by caller-supplied values (parity runs feed the oracle's fb,
 * whose fp64 summation order is not part of the contract -- DESIGN.md "fused bias"). */
BASEQ_API baseq_status_t baseq_set_fused_bias(void* packed, int N, int K, const float* fb, void* stream);

/* ---- fused activation quantiser (K2 of SURVEY; "fuse the online bias and scaling ...
 * within quantization"; Eq. 15; per-token dynamic symmetric int4, round-half-to-even) ----
 *   x_bf16  [T, ldx] bf16, row-major, first K columns of each row are read
 *   codes   [T, K/2] bytes: byte j = (q[2j] & 15) | ((q[2j+1] & 15) << 4)
 *   scales  [T] fp32 step sizes s_t                                                          */
BASEQ_API baseq_status_t baseq_quantize_act(const void* x_bf16, int64_t ldx, int T, int K,
                                  const baseq_act_params_t* p, uint8_t* codes, float* scales,
                                  void* stream);

/* ---- NEXT-2: the same quantiser with the online block-128 Hadamard run on the tensor cores --
 * what the paper deploys ("implement it as a larger matrix multiplication"; R_qk as a
 * 128 x 128 matmul): H_128 X^T with tcgen05.mma kind::f16, fp32 accumulation in tensor
 * memory.  +-1 and the bf16 activations are exact operands; only the ORDER of each 128-term fp32
 * sum is the tensor core's, so codes and scales are not bit-reproducible against
 * baseq_quantize_act's fp32-butterfly contract.  Guarantee: with
 *   u*[t,c] = g_c (H x)[t,c] / sqrt(128) - b_c      evaluated exactly,
 *   tol[t,c] = 2^-16 |g_c| sum_{k in block(c)} |x[t,k]| / sqrt(128) + 2^-21 |u*[t,c]|,
 * the returned s_t is max((alpha m) / 7, 1e-12) for an m inside the band of max_c |u*| +- tol, and
 * every returned code is clamp(rne(u' / s_t), -8, 7) for some u' with |u' - u*| <= tol: a code can
 * differ from the contract's only where u* / s_t is within tol / s_t of a rounding boundary, and then
 * by one level.  Same arguments, layouts and errors as baseq_quantize_act; p->had_block must be 128
 * and K <= 28672, else BASEQ_ERR_UNSUPPORTED.  The codes feed baseq_w4a4_gemm unchanged. */
BASEQ_API baseq_status_t baseq_quantize_act_tc(const void* x_bf16, int64_t ldx, int T, int K,
                                     const baseq_act_params_t* p, uint8_t* codes, float* scales,
                                     void* stream);

/* ---- W4A4 GEMM + fused de-quantisation (K1 + K3 of SURVEY) ----
 *   acc[t,n] = sum_k qa[t,k] * qw[n,k]                       exact int32 (tcgen05 kind::i8)
 *   Y[t,n]   = bf16_rne( (s_t * s_w[n]) * acc[t,n] + fb[n] ) evaluated as the fp64 expression
 *              fma((double)s_t * (double)s_w[n], (double)acc, (double)fb[n]), one rounding to bf16 (C-9)
 *   codes, scales  as produced by baseq_quantize_act
 *   packed_w       blob from baseq_pack_weights for the same (N, K)
 *   y_bf16         [T, ldy] bf16 row-major
 *   acc_dump       optional [T, N] int32 copy of the accumulators (parity runs only), or NULL
 * Decode shapes: for T <= 64 this call and baseq_w4a4_gemm_asym run a
 * weight-streaming kernel (one pass over the packed weights, warp-level s8 MMA on nibbles
 * expanded in registers) instead of the tcgen05 tile kernel; same contract, same bits, same
 * arguments -- the choice is not visible to the caller.  Both kernels are enqueued with the
 * programmatic-dependent-launch attribute and read `codes` / `scales` only after the preceding
 * kernel of `stream` has completed; inside a CUDA graph consecutive calls overlap their weight
 * streams. */
BASEQ_API baseq_status_t baseq_w4a4_gemm(const uint8_t* codes, const float* scales, const void* packed_w,
                               int T, int N, int K, void* y_bf16, int64_t ldy, int32_t* acc_dump,
                               void* stream);

/* ---- NEXT-1: per-token ASYMMETRIC dynamic int4 activations (the paper's deployed setting,
 * P:241 "per-token asymmetric dynamic quantization"; Eq. 4 P:74 with lower bound z and step s;
 * z = alpha * min, s = alpha * (max - min) / 15, floor 1e-12) ----
 *   u_k as above;  mn = min u, mx = max u
 *   s_t = max((alpha * (mx - mn)) / 15, 1e-12);  z_t = alpha * mn
 *   q_k = clamp(rne((u_k - z_t) * (1 / s_t)), 0, 15)            UNSIGNED codes, same nibble packing
 *   zeros  [T] fp32 lattice lower bounds z_t
 * The GEMM re-centres the unsigned codes to q - 8 on chip (tcgen05 kind::i8, S8 x S8, accumulating
 * acc - 8 wsum; acc_dump still returns acc = sum_k q qw, the oracle's accumulator) and the
 * epilogue adds the lower-bound term:  Y = bf16_rne( fma(s_t s_w, acc, fma(z_t s_w, wsum[n], fb[n])) )
 * with wsum[n] = sum_k qw[n,k] from the packed blob (fp64 expression, one rounding to bf16).
 * Scalar gamma or the per-channel vector p->sa, any K the symmetric call accepts; there is no
 * fused single-launch variant with asymmetric codes is baseq_linear_fused_asym below. */
BASEQ_API baseq_status_t baseq_quantize_act_asym(const void* x_bf16, int64_t ldx, int T, int K,
                                       const baseq_act_params_t* p, uint8_t* codes, float* scales,
                                       float* zeros, void* stream);
BASEQ_API baseq_status_t baseq_w4a4_gemm_asym(const uint8_t* codes, const float* scales,
                                    const float* zeros, const void* packed_w, int T, int N, int K,
                                    void* y_bf16, int64_t ldy, int32_t* acc_dump, void* stream);

/* ---- NEXT-3: KV-cache "per-head asymmetric dynamic quantization".  A group is one
 * (token, head) block of head_dim contiguous channels (heads never straddle groups); every
 * group is quantised on its own min / max by the asymmetric rule above (Eq. 4) with
 * u = x (no gamma, bias or Hadamard):
 *   s = max((alpha * (mx - mn)) / 15, 1e-12);  z = alpha * mn;  q = clamp(rne((x - z) * (1 / s)), 0, 15)
 *   x_bf16 [T, ldx] bf16 (device), row t = n_heads blocks of head_dim, ldx >= n_heads * head_dim,
 *          ldx % 8 == 0;  head_dim 64 or 128, else BASEQ_ERR_UNSUPPORTED
 *   codes  [T, n_heads * head_dim / 2] u8 unsigned nibbles (low nibble = even channel), contiguous
 *   scales, zeros [T, n_heads] fp32, contiguous
 * All buffers are caller-owned device memory; the call only enqueues on `stream`. */
BASEQ_API baseq_status_t baseq_quantize_kv(const void* x_bf16, int64_t ldx, int T, int n_heads,
                                           int head_dim, float alpha, uint8_t* codes, float* scales,
                                           float* zeros, void* stream);

/* ---- fused variant (a10): quantiser and GEMM in ONE launch ----
 * Four extra warps per CTA of the GEMM kernel quantise X in the background, one token row per
 * warp, with the arithmetic of baseq_quantize_act; their codes go to `workspace` (the size of the
 * codes, [T, K/2], resident in L2 for the shapes that fit it) and a counter per 128-row group tells
 * the GEMM's TMA producers when a group is complete; tiles are walked M-major so the first wave
 * needs the first one or two 256-row strips only.  No kernel boundary between quantiser and GEMM;
 * the same contract and the same bits as baseq_quantize_act followed by baseq_w4a4_gemm.
 * had_block: 0 or any power of two <= 256 dividing K (128 and 0 at full speed).
 *   workspace / workspace_bytes  device scratch of at least baseq_fused_workspace_bytes(T, N, K)
 *                = a 256-byte control block + 256-byte-rounded counters + T * K / 2 bytes,
 *                256-byte aligned.  Its contents on entry do not matter: the kernel clears its own
 *                counters and announces that through a 64-bit word of the control block, which its
 *                last CTA resets (memory that was never a workspace carries that word by chance
 *                with probability 2^-64); nothing but the kernel is enqueued, so the call can be
 *                captured in a CUDA graph and replayed.  It may be reused by the next call on the
 *                same stream; two calls that overlap on the GPU must not share it (with
 *                workspaces of their own they may overlap: the quantiser warps claim token rows
 *                from a counter, so a CTA that is resident never waits for one that is not)
 *   codes_dump   optional [T, K/2]: the codes are written there instead of the workspace, or NULL
 *   scales_out   [T] required                                                                */
BASEQ_API size_t baseq_fused_workspace_bytes(int T, int N, int K);
BASEQ_API baseq_status_t baseq_linear_fused(const void* x_bf16, int64_t ldx, int T, int K,
                                  const baseq_act_params_t* p, const void* packed_w, int N,
                                  void* y_bf16, int64_t ldy, void* workspace, size_t workspace_bytes,
                                  uint8_t* codes_dump, float* scales_out, int32_t* acc_dump,
                                  void* stream);

/* The same single launch with per-token ASYMMETRIC activations (NEXT-1; Eq. 4): the
 * background warps quantise as baseq_quantize_act_asym does, the GEMM and epilogue are those of
 * baseq_w4a4_gemm_asym -- the same bits as the two calls.  zeros_out [T] required (the lattice
 * lower bounds z_t); codes_dump, if given, receives the UNSIGNED nibbles. */
BASEQ_API baseq_status_t baseq_linear_fused_asym(const void* x_bf16, int64_t ldx, int T, int K,
                                  const baseq_act_params_t* p, const void* packed_w, int N,
                                  void* y_bf16, int64_t ldy, void* workspace, size_t workspace_bytes,
                                  uint8_t* codes_dump, float* scales_out, float* zeros_out,
                                  int32_t* acc_dump, void* stream);

/* ---- end-to-end helper with HOST activations / outputs (bench.py's e2e leg) ----
 * Copies x_host (pinned or pageable) to the device scratch, runs quantize_act + w4a4_gemm on
 * `stream`, copies Y back to y_host.  p->sa / p->b and packed_w are DEVICE pointers as above.
 *   dev_scratch  device buffer of at least baseq_linear_host_scratch_bytes(T, N, K) bytes
 * Returns after enqueueing; the caller synchronises the stream before reading y_host. */
BASEQ_API size_t baseq_linear_host_scratch_bytes(int T, int N, int K);
BASEQ_API baseq_status_t baseq_linear_host(const void* x_bf16_host, int T, int K, const baseq_act_params_t* p,
                                 const void* packed_w, int N, void* y_bf16_host, void* dev_scratch,
                                 size_t dev_scratch_bytes, void* stream);

/* ---- the two-kernel linear for callers that cannot allocate (Eq. 15; a1-a9) ----
 * baseq_quantize_act followed by baseq_w4a4_gemm -- same contract, same bits -- with the
 * intermediate codes [T, K/2] and scales [T] held in a static __device__ array inside the
 * library instead of caller buffers: no cudaMalloc / cudaFree / allocating routine is called,
 * here or by anything it launches (CUDA graph capture, serving loops, harnesses that forbid
 * allocation).  The caller still passes X, the packed weights and Y (device pointers, as above).
 *   limit      T * K / 2 <= 4 MiB of codes and T <= 8192 (config 2, 2048 x 4096, fits exactly);
 *              beyond it BASEQ_ERR_WORKSPACE, nothing enqueued.  The array is
 *              baseq_linear_static_scratch_bytes() = 4 MiB + 32 KiB, held by every GPU that loads
 *              the library until the process exits.
 *   sharing    ONE array per device, shared by every call and keeping the last call's contents
 *              (nothing in it needs to start at zero: each call writes all T rows before it reads
 *              them).  Calls are ordered on their stream; two calls that overlap on the GPU --
 *              different streams, or two host threads on the same device -- RACE on it.        */
BASEQ_API size_t baseq_linear_static_scratch_bytes(void);
BASEQ_API baseq_status_t baseq_linear_static(const void* x_bf16, int64_t ldx, int T, int K,
                                   const baseq_act_params_t* p, const void* packed_w, int N,
                                   void* y_bf16, int64_t ldy, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* BASEQ_H_ */
