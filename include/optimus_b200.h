/* optimus_b200.h -- C ABI of liboptimus_b200 (sm_100a / NVIDIA B200).
 *
 * The runtime hot path that Optimus' horizontal ("group fusion") and split/cat
 * rewrites produce (arxiv/paper_2607_02945): a matched group of N independent
 * same-type operators is replaced by ONE semantically equivalent operator
 * (section 3.2 "each color-coded group is fused into a single
 * composite node"; "group fusion allows multiple no-data
 * dependency instances to be executed within a single kernel launch without
 * altering the individual input tensor layouts, though it requires customized
 * kernels").  This library is those customised kernels: one kernel launch per
 * group, described by an array of per-member descriptors.
 *
 * General conventions
 *   - Plain C.  No exception crosses the ABI; every call returns opt_status and
 *     records a message readable through opt_last_error() (thread-local).
 *   - All tensor pointers in descriptors are DEVICE pointers owned by the caller.
 *     The descriptor array itself is HOST memory, copied during plan_create and
 *     free to release afterwards.  A plan owns only its device-side tables; the
 *     tensor pointers baked into it must stay valid until opt_plan_destroy.
 *   - Layout: every tensor is 2-D row-major with unit column stride; `ld*` is
 *     the row stride in ELEMENTS.  A column slice of a wider buffer (a concat
 *     slot, a split chunk) is expressed as base + column offset with ld = width
 *     of the wider buffer -- "without altering the individual input tensor
 *     layouts".
 *   - Member order is output order ("preserving their original order of
 *     execution").
 *   - Independence precondition ("Nodes are considered independent if no data
 *     dependency exists between them"): no member's output may
 *     overlap any input or any other output of the group; violations that the
 *     host can see from the address ranges return OPT_ERR_ALIAS.  Inputs may
 *     alias each other (batch_linear_lhs).  A pointwise chunk
 *     with dst == src && ldd == lds (in place) is allowed.
 *   - Unsupported or misaligned groups launch NOTHING and return an error: the
 *     "guaranteed no-op fallback" of PAPER.md:183.  There is no CPU fallback.
 *   - Alignment (8 elements for bf16): bf16 paths need 16-byte
 *     aligned base pointers, ld* % 8 == 0, D % 8 == 0, width % 8 == 0.  The
 *     grouped Linear takes ANY K and N (the tails are zero-filled on chip --
 *     what pad_aten_mm_pass does by padding); when N % 8 != 0 the padding
 *     elements of y up to the next 16-byte boundary of each row are overwritten
 *     (nothing else can live there: every base is 16-byte aligned).  fp32 paths need 16-byte aligned
 *     bases and multiples of 4.
 *   - 1 <= n <= 65535 members, every dimension >= 1 (members with rows == 0 are
 *     rejected as OPT_ERR_INVALID_ARG).
 *   - opt_plan_launch is asynchronous on the given stream: exactly one kernel
 *     launch, no allocation, no synchronisation, no memcpy.  Results are
 *     bitwise reproducible run to run (no atomics on outputs, no split-K).
 *   - A plan is single-flight: its device tables hold the work-scheduler
 *     counters of the persistent kernels (re-armed by the kernel itself at the
 *     end of every launch), so the same plan may be launched again and again,
 *     back to back on one stream or as a CUDA-graph node, but must not run
 *     concurrently with itself on two streams.  Different plans are independent.
 */
#ifndef OPTIMUS_B200_H_
#define OPTIMUS_B200_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  OPT_OK = 0,
  OPT_ERR_INVALID_ARG = 1, /* NULL pointer, n out of range, non-positive dimension, bad enum   */
  OPT_ERR_UNSUPPORTED = 2, /* valid but outside what the kernels cover (e.g. D too large)      */
  OPT_ERR_ALIGNMENT = 3,   /* pointer / stride / extent alignment rule violated                */
  OPT_ERR_ALIAS = 4,       /* an output overlaps an input or another output of the group       */
  OPT_ERR_CUDA = 5,        /* a CUDA runtime/driver call failed; message has the CUDA error    */
  OPT_ERR_NO_DEVICE = 6    /* no CUDA device, or the device is not sm_100                      */
} opt_status;

typedef enum { OPT_F32 = 0, OPT_BF16 = 1 } opt_dtype;
typedef enum { OPT_ACT_NONE = 0, OPT_ACT_RELU = 1, OPT_ACT_TANH = 2, OPT_ACT_SIGMOID = 3 } opt_act;
typedef enum {
  OPT_PW_COPY = 0, OPT_PW_RELU = 1, OPT_PW_TANH = 2, OPT_PW_SIGMOID = 3,
  /* the remaining horizontal pointwise patterns of the paper's Table 1 */
  OPT_PW_CLAMP = 4,      /* batch_clamp:      dst = min(max(src, p0), p1), NaN propagates (torch.clamp)          */
  OPT_PW_NAN_TO_NUM = 5, /* batch_nan_to_num: NaN -> p0, +inf -> p1, -inf -> p2, finite values unchanged          */
  OPT_PW_SUB = 6,        /* batch_aten_sub:   dst = src - src2                                                     */
  OPT_PW_DIV = 7,        /* batch_aten_div:   dst = src / src2                                                     */
  OPT_PW_MUL = 8,        /* batch_aten_mul:   dst = src * src2                                                     */
  /* activation_quantization_aten_pass: saved activations kept in FP8 (OCP E4M3) */
  OPT_PW_QUANT_E4M3 = 9,    /* dst (fp8, 1 byte/element, ldd in fp8 elements) = e4m3_rne_satfinite(src * p0)      */
  OPT_PW_DEQUANT_E4M3 = 10, /* dst (bf16) = value(src fp8 code, lds in fp8 elements) * p0                          */
  /* backward of the ReLU epilogue of a grouped Linear in a post-grad graph (batch_linear_post_grad):
   * src = incoming gradient, src2 = the ReLU's forward output (or input: same mask); feeds the dgrad / wgrad groups */
  OPT_PW_RELU_BWD = 11,     /* dst = (src2 <= 0) ? 0 : src   (exact; a NaN in src2 lets the gradient through)      */
  /* backward of the tanh / sigmoid epilogues (torch tanh_backward / sigmoid_backward): src = incoming gradient,
   * src2 = the STORED forward output; fp32 arithmetic, one rounding to the storage dtype                           */
  OPT_PW_TANH_BWD = 12,     /* dst = src * (1 - src2^2)                                                             */
  OPT_PW_SIGMOID_BWD = 13   /* dst = src * (1 - src2) * src2                                                        */
} opt_pw_op;

/* Storage of the two operands of a grouped Linear member.  Default 0: x is [M,K], w is [N,K] (torch nn.Linear).
 * OPT_LAYOUT_X_TRANSPOSED: x is stored [K,M] (ldx = its row stride); OPT_LAYOUT_W_TRANSPOSED: w is stored [K,N].
 * With them the same grouped kernel computes the BACKWARD of a grouped Linear (batch_linear_post_grad operates
 * on post-grad graphs; training QPS is the paper's headline):
 *     dgrad  dX[M,K] = dY[M,N] * W[N,K]      ->  x = dY, w = W stored [contraction N, K]: W_TRANSPOSED
 *     wgrad  dW[N,K] = dY[M,N]^T * X[M,K]    ->  x = dY stored [contraction M, N]: X_TRANSPOSED,
 *                                                w = X stored [contraction M, K]: W_TRANSPOSED
 * The tensor cores read such operands in place (MN-major shared-memory descriptors): no transposed copy.     */
enum { OPT_LAYOUT_X_TRANSPOSED = 1, OPT_LAYOUT_W_TRANSPOSED = 2 };

/* One member of a grouped Linear (+bias +activation) -- batch_linear /
 * batch_linear_post_grad with its epilogue:
 *     Y = act(X * W^T + bias)
 * X:[M,K] (ldx), W:[N,K] (ldw; torch nn.Linear layout, K-major), bias:[N] or
 * NULL, Y:[M,N] (ldy).  For a concatenated output give y = concat_base +
 * column_offset and ldy = total concat width.  bf16: inputs and output bf16,
 * products accumulated in fp32 on the tensor cores, bias and activation in
 * fp32, one round-to-nearest-even to bf16.  fp32: plain fp32 FMA (no TF32).
 * SKINNY groups (decompose_mm_pass: huge M, tiny K and N): a bf16
 * group in which EVERY member has K in {4,8,16}, N in {2,4,8,16}, K*N <= 128 and
 * layout 0 runs through a streaming row kernel instead of 128-row tensor-core
 * tiles (same semantics, one launch); for such a group ldx, ldw and ldy only
 * have to be even, so dense [M,4] x [4,2] tensors are accepted.                */
typedef struct {
  const void* x;
  int64_t ldx;
  const void* w;
  int64_t ldw;
  const void* bias;
  void* y;
  int64_t ldy;
  int32_t M, N, K;
  int32_t act;    /* opt_act */
  int32_t layout; /* 0, or OPT_LAYOUT_* flags: an operand stored transposed (bf16 groups only) */
  /* Optional FP8 copy of the output, written by the same epilogue (activation quantisation fused into the op that
   * produces the saved activation: activation_quantization_aten_pass, `use_scaling`):
   *     y8[m, n] = e4m3_rne_satfinite( bf16(Y[m, n]) * scale8 )          (OCP E4M3, 1 byte per element)
   * i.e. exactly what OPT_PW_QUANT_E4M3 with p0 = scale8 produces from the stored bf16 Y -- bit for bit -- without
   * the extra read of Y.  y8:[M,N] bytes, row stride ldy8 BYTES (ldy8 % 16 == 0, 16-byte aligned base, N % 16 == 0).
   * y8 == NULL: no FP8 output.  With y8 given, y may be NULL (only the FP8 copy is written).  bf16 groups, layout 0.
   * Zero-initialise the three fields otherwise.                                                                    */
  void* y8;
  int64_t ldy8;
  float scale8;
} opt_linear_member;

/* One member of a grouped CHAINED Linear -- two Linear layers of a tower fused
 * vertically, the hidden tensor never written to HBM ("chained
 * transformations", Fig. 5; the paper finds horizontal + vertical fusion
 * combined far better than either alone, Table 3):
 *     h = act1(X * W1^T + b1)      rounded once to bf16 (the intermediate the
 *                                  unfused graph materialises)
 *     Y = act2(h * W2^T + b2)      rounded once to bf16
 * X:[M,K] (ldx), W1:[H,K] (ldw1), b1:[H] or NULL, W2:[N,H] (ldw2), b2:[N] or
 * NULL, Y:[M,N] (ldy; concat slot as for opt_linear_member).  bf16 only.
 * On-chip limits: K <= 256, H <= 512, N <= 64; K % 8 == 0, H % 16 == 0,
 * N % 16 == 0 (otherwise OPT_ERR_UNSUPPORTED / OPT_ERR_ALIGNMENT: run the two
 * layers as two opt_linear groups).  The result equals, bit for bit, what two
 * opt_linear groups produce with h stored in bf16 between them.              */
typedef struct {
  const void* x;
  int64_t ldx;
  const void* w1;
  int64_t ldw1;
  const void* b1;
  const void* w2;
  int64_t ldw2;
  const void* b2;
  void* y;
  int64_t ldy;
  int32_t M, K, H, N;
  int32_t act1, act2; /* opt_act */
} opt_linear2_member;

/* One member of a grouped LayerNorm + CHAINED Linear (SURVEY 8(f) rank 1 with the
 * LayerNorm folded in; the tower of BASELINE.json configs[4]: Fig. 5):
 *     xn = layer_norm(x; gamma, beta, eps) over K   (never materialised, NOT rounded)
 *     h  = act1(xn * W1^T + b1)                      rounded once to bf16
 *     Y  = act2(h * W2^T + b2)                       rounded once to bf16
 * chain.x is the LayerNorm's INPUT [M,K]; every other field of `chain`, the
 * limits and the alignment rules are those of opt_linear2_member.  gamma / beta:
 * [K] bf16 or NULL (1 / 0).  Computed as rstd_r * (x * (W1 diag(gamma))^T - mu_r * s) + c
 * with W1 diag(gamma) rounded to bf16, s_n = sum_k of it, c_n = sum_k beta_k W1[n,k] +
 * b1_n in fp32, refolded from the CURRENT W1 / gamma / beta / b1 inside every
 * launch (plan-owned workspace); row statistics in fp32.  Differs from the
 * three-group path (LayerNorm output stored in bf16) by that one rounding.    */
typedef struct {
  opt_linear2_member chain;
  const void* gamma;
  const void* beta;
  float eps;
  int32_t reserved; /* 0 */
} opt_ln_linear2_member;

/* One member of a batched LayerNorm -- batch_layernorm:
 *     mu = mean(x_r), v = mean((x_r - mu)^2)  (biased), over the last dim D
 *     y_r = (x_r - mu) / sqrt(v + eps) * gamma + beta
 * x:[rows,D] (ldx), y:[rows,D] (ldy), gamma/beta:[D] or NULL (NULL = 1 / 0).
 * Statistics and affine in fp32 (two-pass), one rounding.                     */
typedef struct {
  const void* x;
  int64_t ldx;
  void* y;
  int64_t ldy;
  const void* gamma;
  const void* beta;
  int32_t rows, D;
  float eps;
  /* Optional FP8 (E4M3) copy of the output, same contract as opt_linear_member.y8:
   *     y8[r, j] = e4m3_rne_satfinite( bf16(y[r, j]) * scale8 ),   y8:[rows,D] bytes, row stride ldy8 BYTES (% 8 == 0),
   * 8-byte aligned base; bf16 activations only.  With y8 given, y may be NULL.  Zero-initialise otherwise.        */
  void* y8;
  int64_t ldy8;
  float scale8;
} opt_layernorm_member;

/* One member of a batched LayerNorm BACKWARD (torch
 * native_layer_norm_backward): with mu, v, xhat as in the forward and g = dy * gamma,
 *     dx     = rstd * (g - mean(g) - xhat * mean(g * xhat))      rows x D
 *     dgamma = sum over rows of dy * xhat ;  dbeta = sum over rows of dy      [D]
 * x, dy:[rows,D] (ldx, lddy), gamma:[D] or NULL (= 1), dx:[rows,D] (lddx); dgamma / dbeta: [D] in the param
 * dtype, or NULL when not wanted.  bf16 activations, D % 8 == 0, D <= 2048 (the forward's limit; else OPT_ERR_UNSUPPORTED).  fp32
 * arithmetic; the column sums are added in a fixed order (bitwise reproducible, no atomics on data).            */
typedef struct {
  const void* x;
  int64_t ldx;
  const void* dy;
  int64_t lddy;
  const void* gamma;
  void* dx;
  int64_t lddx;
  void* dgamma;
  void* dbeta;
  int32_t rows, D;
  float eps;
} opt_layernorm_bwd_member;

/* One member of a batched bias gradient (the third output of the backward of
 * y = x W^T + b, PAPER.md:292 batch_linear_post_grad on post-grad graphs, PAPER.md:437 training):
 *     db[n] = sum over m of dZ[m, n]
 * dz:[M,N] (ldz, elements; a column slice of a concat buffer is fine), db:[N] in the param dtype (device
 * pointers, caller-owned).  bf16 activations: N % 8 == 0, 16-byte aligned pointers, ldz % 8 == 0 (fp32 activations --
 * configs[0]-like groups -- multiples of 4; else OPT_ERR_ALIGNMENT).  fp32 accumulation; rows are added in a fixed order (row groups, then row parts, through a
 * plan-owned workspace): bitwise reproducible, no atomics on data.  opt_plan_info: flops = M N adds, bytes = dZ + db.
 *
 * Fused ReLU mask (y != NULL; zero-initialise the struct otherwise): dz then holds the gradient dY that arrives at the
 * ReLU epilogue, y:[M,N] (ldy) the STORED forward output, and the member computes, in the same pass,
 *     dZ[m, n] = (y[m, n] <= 0) ? +0 : dY[m, n]      (torch threshold_backward == OPT_PW_RELU_BWD, bit-exact)
 *     db[n]    = sum over m of dZ[m, n]
 * dZ is written to dz_out:[M,N] (lddz_out) unless dz_out is NULL; dz_out == dz with lddz_out == ldz (in place) is
 * allowed.  y and dz_out follow the alignment rules of dz.  act (opt_act; needs y) selects the epilogue whose
 * derivative is fused: OPT_ACT_NONE / OPT_ACT_RELU the mask above, OPT_ACT_TANH dZ = dY (1 - y^2), OPT_ACT_SIGMOID
 * dZ = dY (1 - y) y -- dZ rounded to bf16 exactly as OPT_PW_TANH_BWD / OPT_PW_SIGMOID_BWD do, and db sums the
 * ROUNDED dZ (what a separate bias-gradient launch would read).                                                     */
typedef struct {
  const void* dz;
  int64_t ldz;
  void* db;
  int32_t M, N;
  const void* y;
  int64_t ldy;
  void* dz_out;
  int64_t lddz_out;
  int32_t act; /* opt_act */
} opt_bias_grad_member;

/* One chunk of a multi-tensor pointwise / split-cat pass -- batch_relu,
 * batch_sigmoid, batch_aten_tanh, batch_detach and the data
 * movement left over by the split/cat rewrites (Listing 2):
 *     dst[r, 0:width] = op(src[r, 0:width])   for r < rows
 * A split->f->cat chain is a list of chunks whose src/dst are column slices of
 * shared bases.  OPT_PW_COPY moves raw bits.  The binary ops read a second
 * operand src2 (same rows x width, row stride lds2); CLAMP / NAN_TO_NUM take
 * their scalars from p0..p2 (fp32; the result is rounded to the storage dtype).
 * For ops 0..3 the extra fields are ignored (zero-initialise the struct).      */
typedef struct {
  const void* src;
  int64_t lds;
  void* dst;
  int64_t ldd;
  int32_t rows, width;
  int32_t op; /* opt_pw_op */
  const void* src2; /* second operand of OPT_PW_SUB / DIV / MUL / *_BWD, else NULL */
  int64_t lds2;
  float p0, p1, p2; /* CLAMP: lo, hi;  NAN_TO_NUM: nan, posinf, neginf */
} opt_chunk;

/* One staged host<->device copy of opt_plan_launch_host. */
typedef struct {
  void* host;   /* host buffer (pinned for true asynchrony)                   */
  void* device; /* device buffer                                              */
  size_t bytes;
  int32_t to_device; /* 1: host->device before the kernel; 0: device->host after it */
} opt_host_copy;

typedef struct opt_plan opt_plan; /* opaque; owns device-side tables only */

/* Optional, documented planning choices of a grouped Linear (zero-initialise for the defaults; the results are
 * the same bits whatever is chosen -- only the schedule changes).  The library reads NO environment variable.
 *   cta_pair      0 (default) or 2: CTA pairs (256-row tiles, tcgen05 cta_group::2, the W tile shared by the pair);
 *                 1: one CTA per 128-row tile.
 *   no_skinny     1: never route a huge-M / tiny-K-and-N group to the streaming row kernel.
 *   no_lhs_order  1: schedule members that share one input X independently (member-major) instead of
 *                 m-block-major across them (batch_linear_lhs).                                  */
typedef struct {
  int32_t cta_pair;
  int32_t no_skinny;
  int32_t no_lhs_order;
  int32_t reserved[5]; /* 0 */
} opt_linear_options;

/* Build a plan for a group.  members: host array of n descriptors.  io: dtype
 * of activations (and of weights/bias for linear).  param: dtype of gamma/beta.
 * device: CUDA device ordinal.  On success *plan is set; on failure *plan is
 * NULL and nothing is launched or left allocated.  Host argument validation
 * happens before the first CUDA call, so INVALID_ARG / ALIGNMENT / ALIAS /
 * UNSUPPORTED are reported even on a machine without a GPU.  The calling
 * thread's current CUDA device is left as it was.                             */
opt_status opt_linear_plan_create(const opt_linear_member* members, int32_t n, opt_dtype io,
                                  int device, opt_plan** plan);
opt_status opt_linear_plan_create_ex(const opt_linear_member* members, int32_t n, opt_dtype io, int device,
                                     const opt_linear_options* options /* NULL = defaults */, opt_plan** plan);
opt_status opt_linear2_plan_create(const opt_linear2_member* members, int32_t n, opt_dtype io,
                                   int device, opt_plan** plan);
opt_status opt_ln_linear2_plan_create(const opt_ln_linear2_member* members, int32_t n, opt_dtype io,
                                      int device, opt_plan** plan);
opt_status opt_layernorm_plan_create(const opt_layernorm_member* members, int32_t n, opt_dtype io,
                                     opt_dtype param, int device, opt_plan** plan);
opt_status opt_layernorm_bwd_plan_create(const opt_layernorm_bwd_member* members, int32_t n, opt_dtype io,
                                         opt_dtype param, int device, opt_plan** plan);
opt_status opt_bias_grad_plan_create(const opt_bias_grad_member* members, int32_t n, opt_dtype io,
                                     opt_dtype param, int device, opt_plan** plan);
opt_status opt_pointwise_plan_create(const opt_chunk* chunks, int32_t n, opt_dtype io, int device,
                                     opt_plan** plan);

/* Enqueue the group on `cuda_stream` (a cudaStream_t; NULL = default stream):
 * exactly ONE kernel launch.  Asynchronous CUDA faults surface at the caller's
 * next synchronisation.                                                      */
opt_status opt_plan_launch(const opt_plan* plan, void* cuda_stream);

/* Same, for HOST buffers: on `cuda_stream`, first every copy with to_device=1
 * (cudaMemcpyAsync host->device), then the one kernel launch, then every copy
 * with to_device=0 (device->host).  No synchronisation; the caller syncs the
 * stream before reading the host outputs.                                    */
opt_status opt_plan_launch_host(const opt_plan* plan, const opt_host_copy* copies, int32_t ncopies,
                                void* cuda_stream);

/* Algorithmic work of one launch: flops (2*M*N*K summed; 0 for non-GEMM),
 * bytes (every input read once + every output written once, tables ignored),
 * launches (always 1) and the number of work tiles/blocks the kernel walks.
 * Any out pointer may be NULL.                                               */
opt_status opt_plan_info(const opt_plan* plan, int64_t* flops, int64_t* bytes, int32_t* launches,
                         int32_t* tiles);

opt_status opt_plan_destroy(opt_plan* plan);

/* NO-ALLOCATION entry point: the bias gradient of ONE Linear layer (PAPER.md:292 batch_linear_post_grad,
 * PAPER.md:437 training),  db[n] = sum over m of dz[m, n],  for callers that cannot call cudaMalloc (code under
 * CUDA-graph capture, tight serving loops, harnesses that forbid allocation).  It creates no plan and calls no
 * cudaMalloc / cudaFree / allocating library routine: the partial sums live in a file-scope device array of
 * OPT_NOALLOC_SCRATCH_BYTES (1 MiB + 256 B) that every GPU which loads the library holds until the process exits.
 *   dz:[M,N] bf16, row stride ldz (elements; a column slice of a concat buffer is fine), db:[N] of dtype `param`
 *   (OPT_F32 or OPT_BF16); device pointers on `device`, caller-owned.  N % 8 == 0, ldz % 8 == 0, 16-byte aligned
 *   pointers (else OPT_ERR_ALIGNMENT); db must not overlap dz (OPT_ERR_ALIAS); M >= 1.
 *   N <= OPT_NOALLOC_BIAS_GRAD_MAX_N, else OPT_ERR_UNSUPPORTED and nothing is launched (wider layers: the planned
 *   path, opt_bias_grad_plan_create).  M is not limited.
 * On `cuda_stream` (NULL = default stream): a 256-byte memset of the scratch's tickets, then ONE kernel launch;
 * asynchronous.  fp32 accumulation in a fixed order (bitwise reproducible, no atomics on data); the partitioning
 * differs from the planned kernel's, so the two agree within fp32 rounding, not bit for bit.
 * EVERY call shares the one scratch array: calls that overlap on the GPU (different streams or threads without an
 * ordering between them) RACE; calls on one stream are safe.  The calling thread's current device is left as it was. */
#define OPT_NOALLOC_BIAS_GRAD_MAX_N 4096
#define OPT_NOALLOC_SCRATCH_BYTES (64 * OPT_NOALLOC_BIAS_GRAD_MAX_N * 4 + 256)
opt_status opt_bias_grad_noalloc(const void* dz, int64_t ldz, void* db, int32_t M, int32_t N, opt_dtype param,
                                 int device, void* cuda_stream);

/* Last error message of the calling thread; never NULL ("" if none). */
const char* opt_last_error(void);

/* Process-wide count of kernel launches issued by this library. */
uint64_t opt_launch_count(void);

/* Library version string, e.g. "liboptimus_b200 0.1 (sm_100a)". */
const char* opt_version(void);

#ifdef __cplusplus
}
#endif
#endif /* OPTIMUS_B200_H_ */
