// Grouped CHAINED Linear: N independent  Y_i = act2(act1(X_i W1_i^T + b1_i) W2_i^T + b2_i)  in ONE
// launch, the hidden tensor never leaving the SM -- vertical fusion of two horizontally fused Linear
// groups ("chained transformations", Fig. 5; PAPER.md:363 horizontal + vertical combined;
// SURVEY.md 8(f) rank 1; include/optimus_b200.h opt_linear2_member).
//
// Semantics = the unfused graph with its intermediate in bf16 (reading Q3):
//     h = bf16_rne(act1(x W1^T + b1))        fp32 accumulate, fp32 bias/activation, one rounding
//     y = bf16_rne(act2(h W2^T + b2))
// so the result is the one the two-launch path (two grouped GEMMs) produces, without the 2 x M x H x 2 bytes
// of HBM traffic for h.
//
// Kernel: persistent, one CTA per SM, 384 threads, per 128-row tile of a member:
//   warp 0  TMA producer: the X tile (K <= 256: up to four 128x64 k-blocks, resident for the whole tile), a
//           4-stage ring of W1 k-blocks (128 hidden units x 64), a 2-stage ring of W2 slices (N x 128);
//   warp 1  layer-1 MMA issuer: per hidden chunk c of 128 units  acc1[c&1] = X . W1_c^T  (M=128, N<=128); it
//           never waits for a hidden tile, so the tensor pipe has work while the epilogue turns acc1 into h;
//   warp 11 layer-2 MMA issuer: acc2 += h_c . W2_c^T (M=128, N<=64, K<=128) as soon as h_c is published
//           (two issuing threads: a single one was instruction-bound on these short MMAs);
//   warp 2  tile scheduler (dynamic, one atomic per 4 tiles; entry + b1 + b2 into a 4-deep queue);
//   warps 3..10  epilogue: acc1 chunk -> +b1, act1, RNE bf16 -> the hidden tile in shared memory, written
//           directly in the K-major 128-byte-swizzled layout MMA2 reads; a tile's acc2 is drained late (after the
//           next tile's first chunk): + b2, act2, RNE -> staging -> TMA store into the output / concat slot.
//   TMEM: acc1 2 x 128 columns, acc2 2 x 64 columns.
//
// LN = true (opt_ln_linear2_plan_create): a LayerNorm over K in front of the chain, folded in algebraically so that
// the normalised tensor never exists (reading Q25):
//     xn W1^T + b1 = rstd_r * (x W1g^T - mu_r * s + sigma_r * c),   W1g = W1 diag(gamma) (bf16), s_n = sum_k W1g[n,k],
//                                                 c_n = sum_k beta_k W1[n,k] + b1_n,  sigma_r = 1 / rstd_r
//   and the two rank-1 terms ride on the tensor core as ONE extra K=16 MMA step per hidden chunk: an augmented
//   A k-slice [-mu_h, -mu_h, -mu_l, sigma_h, sigma_h, sigma_l, 0...] per row against an augmented B k-slice
//   [s_h, s_l, s_h, c_h, c_l, c_h, 0...] per hidden unit (hi / lo bf16 splits: products exact in fp32, the dropped
//   lo x lo term is 2^-16 relative).  So:
//   * prologue: every CTA folds a share of the members (W1g and the augmented slice into the plan's workspace) and
//     publishes a per-member epoch flag; the scheduler warp waits for a member's flag before it queues one of its
//     tiles (no grid-wide barrier: a CTA only ever waits for a prologue, and prologues wait for nothing);
//   * the raw X tile feeds MMA1 with W1g; the epilogue warps compute mu_r, sigma_r of the 128 rows from the same
//     shared-memory tile WHILE the MMAs run (two threads per row, shifted single pass, fp32) and write the augmented
//     A slice (extra statistics warps would put > 12 warps on the SM: <= 128 registers, measured 30 us slower);
//   * epilogue 1 is h = act1(rstd_r * acc): no per-column operand at all.
#include <algorithm>
#include <cstdlib>

#include "sm100_ptx.h"

namespace optb {

// Pipeline trace build (-DOPTB_GEMM_TRACE: liboptimus_b200_trace.so only, see grouped_gemm_sm100.cuh): cycles each
// warp role spends blocked on each barrier, one record of 32 counters per CTA.
#ifdef OPTB_GEMM_TRACE
__device__ unsigned long long* g_l2_trace = nullptr;       // [gridDim.x][32] or NULL
#define T2_DECL(name) long long name = 0
#define T2_NOW(name) name = clock64()
#define T2_WAIT(acc, stmt) do { const long long t0__ = clock64(); stmt; acc += clock64() - t0__; } while (0)
#define T2_ADD(acc, val) acc += (val)
#define T2_STORE(slot, val) do { if (g_l2_trace) g_l2_trace[(size_t)blockIdx.x * 32 + (slot)] = (unsigned long long)(val); } while (0)
#else
#define T2_DECL(name)
#define T2_NOW(name) do { } while (0)
#define T2_WAIT(acc, stmt) do { stmt; } while (0)
#define T2_ADD(acc, val) do { } while (0)
#define T2_STORE(slot, val) do { } while (0)
#endif

constexpr int kT_BM = 128;            // tile rows
constexpr int kT_BK = 64;             // k-block: one 128-byte swizzle row of bf16
constexpr int kT_HC = 128;            // hidden chunk: UMMA N of layer 1, K of layer 2 per chunk
constexpr int kT_MaxK = 256;          // layer-1 K (input features): the X tile is at most 4 k-blocks
constexpr int kT_MaxH = 512;          // hidden width: b1 travels in the queue slot
constexpr int kT_MaxN = 64;           // layer-2 N
constexpr int kT_W1Stages = 6;
constexpr int kT_EpiWarps = 8;
constexpr int kT_FirstEpiWarp = 3;
constexpr int kT_Mma2Warp = kT_FirstEpiWarp + kT_EpiWarps;     // warp 11: layer-2 MMA issuer
constexpr int kT_KBlockBytes = kT_BM * kT_BK * 2;          // 16 KB: a 128 x 64 bf16 k-block
constexpr int kT_W2KBlockBytes = kT_MaxN * kT_BK * 2;      // 8 KB: a 64 x 64 k-block of W2
constexpr int kT_QDepth = 4;
constexpr int kT_FlagSpinLimit = 4096;   // polls of a member's fold flag before the scheduler warp folds the member itself
// shared-memory map
constexpr int kT_OffX = 0;
constexpr int kT_OffW1 = kT_OffX + (kT_MaxK / kT_BK) * kT_KBlockBytes;            //  64 KB
constexpr int kT_OffW2 = kT_OffW1 + kT_W1Stages * kT_KBlockBytes;                 // +96 KB
constexpr int kT_OffOut = kT_OffW2 + 2 * 2 * kT_W2KBlockBytes;                    // +32 KB
constexpr int kT_OffQ = kT_OffOut + 4 * 4096;                                     // +16 KB output staging (4 warps x 32 rows x 128 B)
template <bool LN>
struct L2Cfg {
  static constexpr int kThreads = 32 * (kT_Mma2Warp + 1);
  // LN: the augmented A k-slice (a 128 x 64 k-block in the swizzled layout, 16 columns used) sits before the queue
  static constexpr int kOffAug = kT_OffQ;
  static constexpr int kOffQ = kT_OffQ + (LN ? kT_KBlockBytes : 0);
  // queue slot:  b1 (widened to fp32) | b2 (fp32) | TileEntry2     or, LN (no room for more):  b2 (bf16) | TileEntry2
  static constexpr int kOffB2 = LN ? 0 : kT_MaxH * 4;
  static constexpr int kQEntryOff = kOffB2 + kT_MaxN * (LN ? 2 : 4);
  static constexpr int kQSlotBytes = kQEntryOff + 32;
  static constexpr int kOffStats = kOffQ + kT_QDepth * kQSlotBytes;               // LN: partial row sums, 2 halves x 128 rows x {sum, sumsq}
  static constexpr int kOffBar = kOffStats + (LN ? 2 * kT_BM * 8 : 0);
  static constexpr int kSmemBytes = kOffBar + 384;
  static_assert(kSmemBytes <= 227 * 1024, "chained-GEMM shared memory map exceeds 227 KB");
};
constexpr int kT_TmemCols = 512;      // acc1: columns [0,256), acc2: [256,384), hidden tile (bf16 pairs): [384,512)
constexpr uint32_t kT_TmemAcc2 = 256, kT_TmemH = 384;

struct alignas(128) L2Member {
  CUtensorMap tmX;       // X  [M,K]   box {64, 128}  load
  CUtensorMap tmW1;      // W1 [H,K]   box {64, 128}  load
  CUtensorMap tmW2;      // W2 [N,H]   box {64, N}    load
  CUtensorMap tmY;       // Y  [M,N]   box {64, 32}   store
  CUtensorMap tmAug;     // LN: augmented B slice [H,16], box {64, 128} (columns 16.. zero-filled)  load
};
static_assert(sizeof(L2Member) == 640, "L2Member keeps tensor maps 128-byte aligned");

struct alignas(16) TileEntry2 {       // member < 0: padding entry of a chunk
  int32_t member, m0;
  uint32_t shape;        // H | K blocks of layer 1 << 16 | K=16 steps in the last K block << 24
  uint32_t misc;         // act1 | act2 << 8 | N << 16
  const void* b1;        // [H] bf16 or NULL
  const void* b2;        // [N] bf16 or NULL
};
static_assert(sizeof(TileEntry2) == 32, "TileEntry2 is two 16-byte vectors");

struct alignas(16) L2Fold {            // LN: what the prologue needs to fold one member's LayerNorm affine into W1
  const uint16_t* w1; int64_t ldw1;
  const uint16_t* gamma; const uint16_t* beta; const uint16_t* b1;
  uint16_t* w1g;         // [H,K] dense bf16 (workspace)
  uint16_t* aug;         // [H,16] bf16: s_h, s_l, s_h, c_h, c_l, c_h, 0 ... (workspace)
  int32_t H, K;
  float eps; int32_t pad;
};
static_assert(sizeof(L2Fold) == 80, "L2Fold layout");

__device__ __forceinline__ uint32_t l2_idesc(int n) {   // kind::f16, bf16 x bf16 -> fp32, M = 128, K-major A and B
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(kT_BM >> 4) << 24);
}

// Epilogue math of one 32-row x 64-column piece held in v[64] (this thread: one row): + bias (fp32 in the tile's queue
// slot: the scheduler warp widened it once per tile), activation, RNE to bf16 -> 32 packed pairs.  Packed f32x2 adds:
// the same fp32 sums as the grouped GEMM's epilogue (bitwise), in a third of the instructions.
template <int ACT>
__device__ __forceinline__ void epi2_math(const uint32_t (&v)[64], uint32_t bias_addr, uint32_t (&p)[32]) {
#pragma unroll
  for (int j = 0; j < 16; ++j) {         // 4 columns per step
    const uint4 b = lds128(bias_addr + 16 * j);
    f32x2 s0, s1;
    asm("mov.b64 %0, {%1, %2};" : "=l"(s0) : "r"(v[4 * j]), "r"(v[4 * j + 1]));
    asm("mov.b64 %0, {%1, %2};" : "=l"(s1) : "r"(v[4 * j + 2]), "r"(v[4 * j + 3]));
    f32x2 b0, b1;
    asm("mov.b64 %0, {%1, %2};" : "=l"(b0) : "r"(b.x), "r"(b.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(b1) : "r"(b.z), "r"(b.w));
    s0 = add2(s0, b0); s1 = add2(s1, b1);
    float f0, f1, f2, f3;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(f0), "=f"(f1) : "l"(s0));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(f2), "=f"(f3) : "l"(s1));
    if (ACT == OPT_ACT_RELU) { p[2 * j] = pack_relu_bf16x2(f0, f1); p[2 * j + 1] = pack_relu_bf16x2(f2, f3); }
    else {
      p[2 * j] = pack_bf16x2(act_f32<true>(f0, ACT), act_f32<true>(f1, ACT));
      p[2 * j + 1] = pack_bf16x2(act_f32<true>(f2, ACT), act_f32<true>(f3, ACT));
    }
  }
}
__device__ __forceinline__ void epi_act_b16(const uint32_t (&v)[64], uint32_t bias_addr, int act, uint32_t (&p)[32]) {   // bf16 bias
  switch (act) {
    case OPT_ACT_RELU: epi_math<OPT_ACT_RELU>(v, bias_addr, p); break;
    case OPT_ACT_NONE: epi_math<OPT_ACT_NONE>(v, bias_addr, p); break;
    case OPT_ACT_TANH: epi_math<OPT_ACT_TANH>(v, bias_addr, p); break;
    default:           epi_math<OPT_ACT_SIGMOID>(v, bias_addr, p); break;
  }
}
__device__ __forceinline__ void epi_act(const uint32_t (&v)[64], uint32_t bias_addr, int act, uint32_t (&p)[32]) {
  switch (act) {
    case OPT_ACT_RELU: epi2_math<OPT_ACT_RELU>(v, bias_addr, p); break;
    case OPT_ACT_NONE: epi2_math<OPT_ACT_NONE>(v, bias_addr, p); break;
    case OPT_ACT_TANH: epi2_math<OPT_ACT_TANH>(v, bias_addr, p); break;
    default:           epi2_math<OPT_ACT_SIGMOID>(v, bias_addr, p); break;
  }
}

// LN, layer 1: h = act(rstd_r * acc) (this thread's row; the per-column terms were added by the tensor core).
template <int ACT>
__device__ __forceinline__ void epi_math_ln(const uint32_t (&v)[64], float A, uint32_t (&p)[32]) {
#pragma unroll
  for (int j = 0; j < 32; ++j) {
    const float f0 = A * __uint_as_float(v[2 * j]), f1 = A * __uint_as_float(v[2 * j + 1]);
    if (ACT == OPT_ACT_RELU) p[j] = pack_relu_bf16x2(f0, f1);
    else p[j] = pack_bf16x2(act_f32<true>(f0, ACT), act_f32<true>(f1, ACT));
  }
}
__device__ __forceinline__ void epi_act_ln(const uint32_t (&v)[64], float A, int act, uint32_t (&p)[32]) {
  switch (act) {
    case OPT_ACT_RELU: epi_math_ln<OPT_ACT_RELU>(v, A, p); break;
    case OPT_ACT_NONE: epi_math_ln<OPT_ACT_NONE>(v, A, p); break;
    case OPT_ACT_TANH: epi_math_ln<OPT_ACT_TANH>(v, A, p); break;
    default:           epi_math_ln<OPT_ACT_SIGMOID>(v, A, p); break;
  }
}

// LN prologue: fold one member.  A row n of W1 is handled by LP = pow2 >= K/8 lanes (one 16-byte vector each):
//   W1g[n,k] = bf16(W1[n,k] * gamma_k);  s_n = sum_k W1g[n,k];  c_n = sum_k beta_k W1[n,k] + b1_n   (fp32, fixed order)
//   aug[n, 0..5] = s_h, s_l, s_h, c_h, c_l, c_h  (v_h = bf16(v), v_l = bf16(v - v_h)), aug[n, 6..15] = 0
__device__ __forceinline__ void l2_fold_member(const L2Fold& f, int warp, int nwarps, int lane) {
  const int nv = f.K >> 3;
  int LP = 1;
  while (LP < nv) LP <<= 1;
  const int rows_per_pass = 32 / LP, sub = lane / LP, j = lane % LP;
  uint4 g = make_uint4(0x3F803F80u, 0x3F803F80u, 0x3F803F80u, 0x3F803F80u), be = make_uint4(0, 0, 0, 0);   // gamma = 1, beta = 0
  if (j < nv) {
    if (f.gamma) g = __ldg(reinterpret_cast<const uint4*>(f.gamma) + j);
    if (f.beta) be = __ldg(reinterpret_cast<const uint4*>(f.beta) + j);
  }
  const uint32_t gw[4] = {g.x, g.y, g.z, g.w}, bw[4] = {be.x, be.y, be.z, be.w};
  constexpr int kBatch = 16;               // rows in flight per lane: the fold is latency-bound (one L2 round trip per batch)
  const int stride = nwarps * rows_per_pass;
  for (int nb = warp * rows_per_pass; nb < f.H; nb += kBatch * stride) {
    uint4 w[kBatch];
#pragma unroll
    for (int b = 0; b < kBatch; ++b) {
      const int n = nb + b * stride + sub;
      w[b] = make_uint4(0, 0, 0, 0);
      if (n < f.H && j < nv) w[b] = __ldg(reinterpret_cast<const uint4*>(f.w1 + (int64_t)n * f.ldw1) + j);
    }
#pragma unroll
    for (int b = 0; b < kBatch; ++b) {
      const int n = nb + b * stride + sub;
      if (nb + b * stride >= f.H) break;                   // warp-uniform
      float ssum = 0.f, csum = 0.f;
      const uint32_t ww[4] = {w[b].x, w[b].y, w[b].z, w[b].w};
      uint32_t o[4];
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        o[t] = pack_bf16x2(bf16_lo(ww[t]) * bf16_lo(gw[t]), bf16_hi(ww[t]) * bf16_hi(gw[t]));
        ssum += bf16_lo(o[t]) + bf16_hi(o[t]);
        csum = fmaf(bf16_lo(ww[t]), bf16_lo(bw[t]), fmaf(bf16_hi(ww[t]), bf16_hi(bw[t]), csum));
      }
      if (n < f.H && j < nv) *(reinterpret_cast<uint4*>(f.w1g + (int64_t)n * f.K) + j) = make_uint4(o[0], o[1], o[2], o[3]);
      for (int d = LP >> 1; d >= 1; d >>= 1) {
        ssum += __shfl_xor_sync(0xffffffffu, ssum, d);
        csum += __shfl_xor_sync(0xffffffffu, csum, d);
      }
      if (n < f.H && j == 0) {
        if (f.b1) csum += __uint_as_float((uint32_t)__ldg(f.b1 + n) << 16);
        const uint32_t s2 = pack_bf16x2(ssum, 0.f), c2 = pack_bf16x2(csum, 0.f);                 // hi parts (low halves)
        const uint32_t sl = pack_bf16x2(ssum - bf16_lo(s2), 0.f), cl = pack_bf16x2(csum - bf16_lo(c2), 0.f);
        uint4* a = reinterpret_cast<uint4*>(f.aug + (int64_t)n * 16);
        a[0] = make_uint4((s2 & 0xFFFFu) | (sl << 16), (s2 & 0xFFFFu) | (c2 << 16), (cl & 0xFFFFu) | (c2 << 16), 0u);
        a[1] = make_uint4(0u, 0u, 0u, 0u);
      }
    }
  }
}

template <bool LN>
__global__ void __launch_bounds__(L2Cfg<LN>::kThreads, 1)
grouped_linear2_sm100_kernel(const L2Member* __restrict__ members, const uint4* __restrict__ chunks, int n_chunks,
                             int* __restrict__ counters, const L2Fold* __restrict__ folds, int* __restrict__ flags,
                             int n_members) {
  using Cfg = L2Cfg<LN>;
  constexpr int kT_QSlotBytes = Cfg::kQSlotBytes, kT_OffBar = Cfg::kOffBar;
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t sbase = smem_u32(smem);
  if ((sbase & 1023u) != 0) __trap();            // 128-byte-swizzle tiles need 1024-byte alignment
  const uint32_t bar_base = sbase + kT_OffBar;
  // barriers (8 bytes each)
  const uint32_t xa_full = bar_base, xa_empty = bar_base + 8;
  auto w1_full = [&](int s) { return bar_base + 16u + 8u * s; };
  auto w1_empty = [&](int s) { return bar_base + 16u + 8u * (kT_W1Stages + s); };
  constexpr uint32_t kB2 = 16u + 16u * kT_W1Stages;        // the two-entry barrier arrays follow
  auto w2_full = [&](int s) { return bar_base + kB2 + 8u * s; };
  auto w2_empty = [&](int s) { return bar_base + kB2 + 16u + 8u * s; };
  auto a1_full = [&](int s) { return bar_base + kB2 + 32u + 8u * s; };
  auto a1_empty = [&](int s) { return bar_base + kB2 + 48u + 8u * s; };
  auto h_full = [&](int s) { return bar_base + kB2 + 64u + 8u * s; };
  auto h_empty = [&](int s) { return bar_base + kB2 + 80u + 8u * s; };
  auto a2_full = [&](int s) { return bar_base + kB2 + 96u + 8u * s; };
  auto a2_empty = [&](int s) { return bar_base + kB2 + 112u + 8u * s; };
  auto q_full = [&](int s) { return bar_base + kB2 + 128u + 8u * s; };
  auto q_empty = [&](int s) { return bar_base + kB2 + 128u + 8u * (kT_QDepth + s); };
  const uint32_t tmem_ptr_addr = bar_base + kB2 + 128u + 16u * kT_QDepth;
  auto st_full = [&](int s) { return tmem_ptr_addr + 8u + 8u * s; };           // LN: the augmented A slice of a tile is written
  static_assert(16 + 16 * kT_W1Stages + 128 + 16 * kT_QDepth + 8 + 32 <= 384, "barrier area");
  auto q_slot = [&](int s) { return sbase + Cfg::kOffQ + (uint32_t)s * kT_QSlotBytes; };
  constexpr uint32_t kQEntryOff = Cfg::kQEntryOff, kOffB2 = Cfg::kOffB2;
  const uint32_t stats_base = sbase + Cfg::kOffStats, aug_base = sbase + Cfg::kOffAug;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    mbar_init(xa_full, 1); mbar_init(xa_empty, LN ? 1 + kT_EpiWarps : 1);       // LN: the epilogue warps read the X tile too (row statistics)
    if (LN) for (int s = 0; s < 2; ++s) mbar_init(st_full(s), kT_EpiWarps / 2);
    for (int s = 0; s < kT_W1Stages; ++s) { mbar_init(w1_full(s), 1); mbar_init(w1_empty(s), 1); }
    for (int s = 0; s < 2; ++s) {
      mbar_init(w2_full(s), 1); mbar_init(w2_empty(s), 1);
      mbar_init(a1_full(s), 1); mbar_init(a1_empty(s), kT_EpiWarps);
      mbar_init(h_full(s), kT_EpiWarps); mbar_init(h_empty(s), 1);
      mbar_init(a2_full(s), 1); mbar_init(a2_empty(s), kT_EpiWarps);
    }
    for (int s = 0; s < kT_QDepth; ++s) { mbar_init(q_full(s), 1); mbar_init(q_empty(s), 3 + kT_EpiWarps); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async_smem();
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                 ::"r"(tmem_ptr_addr), "n"(kT_TmemCols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_addr) : "memory");

  int epoch1 = 0;                                  // LN: value a member's flag carries once folded in THIS launch
  if (LN) {
    epoch1 = *reinterpret_cast<volatile int*>(counters + 2) + 1;
    for (int i = blockIdx.x; i < n_members; i += gridDim.x) {
      const L2Fold f = folds[i];
      l2_fold_member(f, warp, Cfg::kThreads / 32, lane);
    }
    asm volatile("fence.proxy.async;" ::: "memory");       // W1g is read back through TMA (async proxy)
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0)
      for (int i = blockIdx.x; i < n_members; i += gridDim.x)
        asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(flags + i), "r"(epoch1) : "memory");
  }

  if (warp == 2) {
    // ----------------------------------------------------- tile scheduler ----
    int qs = 0; uint32_t qph = 0;
    int c = blockIdx.x;
    while (c < n_chunks) {
      int nextc = 0;
      if (lane == 0) nextc = atomicAdd(counters, 1) + (int)gridDim.x;
      uint4 e = make_uint4(0xFFFFFFFFu, 0, 0, 0);
      if (lane < 8) e = __ldg(chunks + (size_t)c * 8 + lane);          // lane 2g, 2g+1: tile g of the chunk
      // per tile: bias slices -> registers (the loads of tile g+1 are in flight while tile g is published)
      uint4 b1a, b1b, b2v;
      auto fetch = [&](int g, int& member) {
        member = (int)__shfl_sync(0xffffffffu, e.x, 2 * g);
        const uint32_t shape = __shfl_sync(0xffffffffu, e.z, 2 * g), misc = __shfl_sync(0xffffffffu, e.w, 2 * g);
        const uint32_t p1l = __shfl_sync(0xffffffffu, e.x, 2 * g + 1), p1h = __shfl_sync(0xffffffffu, e.y, 2 * g + 1);
        const uint32_t p2l = __shfl_sync(0xffffffffu, e.z, 2 * g + 1), p2h = __shfl_sync(0xffffffffu, e.w, 2 * g + 1);
        const uint4* b1 = reinterpret_cast<const uint4*>(((uint64_t)p1h << 32) | p1l);
        const uint4* b2 = reinterpret_cast<const uint4*>(((uint64_t)p2h << 32) | p2l);
        const int H = (int)(shape & 0xFFFFu), N = (int)(misc >> 16);
        b1a = b1b = b2v = make_uint4(0, 0, 0, 0);
        if (member >= 0) {
          if (LN) {
            // the member's folded weights / s / c come from some CTA's prologue of THIS launch: wait for its flag
            int ready = 0;
            if (lane == 0) {
              int f;
              for (int spin = 0; spin < kT_FlagSpinLimit && !ready; ++spin) {
                asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(f) : "l"(flags + member) : "memory");
                ready = f == epoch1;
              }
            }
            ready = __shfl_sync(0xffffffffu, ready, 0);
            if (!ready) {
              // The owner's prologue has not run (its CTA is not resident: fewer SMs than the grid, e.g. a partitioned
              // context): fold the member here.  Folds are idempotent -- every writer stores the same bits.
              const L2Fold f = folds[member];
              l2_fold_member(f, 0, 1, lane);
              asm volatile("fence.proxy.async;" ::: "memory");
              __threadfence();
              __syncwarp();
              if (lane == 0) asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(flags + member), "r"(epoch1) : "memory");
            }
            __syncwarp();
          } else {
            if (b1 != nullptr && 8 * lane < H) b1a = __ldg(b1 + lane);
            if (b1 != nullptr && 8 * (lane + 32) < H) b1b = __ldg(b1 + lane + 32);
          }
          if (b2 != nullptr && 8 * lane < N) b2v = __ldg(b2 + lane);
          if (lane < (LN ? 5 : 4))
            asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<const char*>(members + member) + 128 * lane) : "memory");
          // the tile's X k-blocks -> L2 now: the X buffer is single (64 KB), its load can only be issued when the
          // previous tile's last MMA1 has retired, and should then find the data in L2 rather than in HBM
          const int nkb1 = (int)((shape >> 16) & 0xFFu), m0 = (int)__shfl_sync(0xffffffffu, e.y, 2 * g);
          if (lane < nkb1)
            asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global.tile [%0, {%1, %2}];"
                         ::"l"(&members[member].tmX), "r"(lane * kT_BK), "r"(m0) : "memory");
        }
      };
      int member;
      fetch(0, member);
#pragma unroll 1
      for (int g = 0; g < 4; ++g) {
        const uint4 c1a = b1a, c1b = b1b, c2 = b2v;
        const int cur = member;
        if (g + 1 < 4) fetch(g + 1, member);
        if (cur < 0) continue;             // warp-uniform
        mbar_wait(q_empty(qs), qph ^ 1);
        const uint32_t slot = q_slot(qs);
        auto widen = [](uint32_t a, uint32_t b) { return make_uint4(a << 16, a & 0xFFFF0000u, b << 16, b & 0xFFFF0000u); };
        if (!LN) {                           // 8 bf16 per lane -> 8 fp32: units [8 lane, 8 lane + 8) and 256 + the same
          sts128(slot + 32 * lane, widen(c1a.x, c1a.y));
          sts128(slot + 32 * lane + 16, widen(c1a.z, c1a.w));
          sts128(slot + 1024 + 32 * lane, widen(c1b.x, c1b.y));
          sts128(slot + 1024 + 32 * lane + 16, widen(c1b.z, c1b.w));
        }
        if (LN) {
          if (lane < kT_MaxN / 8) sts128(slot + kOffB2 + 16 * lane, c2);
        } else if (lane < kT_MaxN / 8) {
          sts128(slot + kOffB2 + 32 * lane, widen(c2.x, c2.y));
          sts128(slot + kOffB2 + 32 * lane + 16, widen(c2.z, c2.w));
        }
        if ((lane >> 1) == g) sts128(slot + kQEntryOff + 16 * (lane & 1), e);
        __syncwarp();
        if (lane == 0) mbar_arrive(q_full(qs));
        if (++qs == kT_QDepth) { qs = 0; qph ^= 1; }
      }
      c = __shfl_sync(0xffffffffu, nextc, 0);
    }
    mbar_wait(q_empty(qs), qph ^ 1);
    if (lane == 0) {      // end marker; the last CTA to finish re-arms the counters for the next launch
      sts128(q_slot(qs) + kQEntryOff, make_uint4(0xFFFFFFFFu, 0, 0, 0));
      mbar_arrive(q_full(qs));
      __threadfence();
      if (atomicAdd(counters + 1, 1) == (int)gridDim.x - 1) {
        counters[0] = 0; counters[1] = 0;
        if (LN) counters[2] = epoch1;      // the next launch's flags carry the next epoch
        __threadfence();
      }
    }
  } else if (warp == 0) {
    // ------------------------------------------------------- TMA producer ----
    // Issue order = the order the MMA warp consumes: X(t); per chunk c: W1 k-blocks of c, then W2 of c-1; W2 of
    // the last chunk.  (A producer that follows the consumer's order cannot deadlock on the three rings.)
    if (lane == 0) {
      int qs = 0; uint32_t qph = 0;
      int w1s = 0; uint32_t w1ph = 0;
      uint32_t gt = 0, gh = 0;                       // tiles / hidden chunks issued so far
      T2_DECL(tr_t0); T2_DECL(tr_q); T2_DECL(tr_xe); T2_DECL(tr_w1e); T2_DECL(tr_w2e);
      T2_NOW(tr_t0);
      for (;;) {
        T2_WAIT(tr_q, mbar_wait(q_full(qs), qph));
        const uint4 e0 = lds128(q_slot(qs) + kQEntryOff);
        mbar_arrive(q_empty(qs));
        if (++qs == kT_QDepth) { qs = 0; qph ^= 1; }
        if ((int)e0.x < 0) break;
        const L2Member* m = members + (int)e0.x;
        const int m0 = (int)e0.y;
        const int H = (int)(e0.z & 0xFFFFu), nkb1 = (int)((e0.z >> 16) & 0xFFu);
        const int N = (int)(e0.w >> 16);
        const int nch = (H + kT_HC - 1) / kT_HC;
        if (LN) asm volatile("fence.proxy.async;" ::: "memory");   // W1g: generic-proxy writes of this launch -> TMA reads
        // X tile: resident for the whole tile, reloaded when the last MMA1 of the previous tile has retired
        T2_WAIT(tr_xe, mbar_wait(xa_empty, (gt & 1u) ^ 1u));
        mbar_expect_tx(xa_full, (uint32_t)nkb1 * kT_KBlockBytes);
        for (int kb = 0; kb < nkb1; ++kb) tma_load_2d(sbase + kT_OffX + kb * kT_KBlockBytes, &m->tmX, xa_full, kb * kT_BK, m0);
        ++gt;
        auto load_w2 = [&](int c, uint32_t g) {       // chunk c's slice of W2: [N, 128] = up to two 64-wide k-blocks
          const int s = (int)(g & 1u);
          const int bn = min(kT_HC, H - c * kT_HC), nkb2 = (bn + kT_BK - 1) / kT_BK;
          T2_WAIT(tr_w2e, mbar_wait(w2_empty(s), ((g >> 1) & 1u) ^ 1u));
          mbar_expect_tx(w2_full(s), (uint32_t)(nkb2 * N * kT_BK * 2));
          for (int j = 0; j < nkb2; ++j)
            tma_load_2d(sbase + kT_OffW2 + s * 2 * kT_W2KBlockBytes + j * kT_W2KBlockBytes, &m->tmW2, w2_full(s),
                        c * kT_HC + j * kT_BK, 0);
        };
        for (int c = 0; c < nch; ++c) {
          if (c >= 1) load_w2(c - 1, gh + c - 1);        // before W1 of chunk c: this thread may block on the W1 ring, and MMA2 of chunk c - 1 must not wait for its (small) W2 slice behind that
          for (int kb = 0; kb < nkb1; ++kb) {
            T2_WAIT(tr_w1e, mbar_wait(w1_empty(w1s), w1ph ^ 1));
            mbar_expect_tx(w1_full(w1s), kT_KBlockBytes);
            tma_load_2d(sbase + kT_OffW1 + w1s * kT_KBlockBytes, &m->tmW1, w1_full(w1s), kb * kT_BK, c * kT_HC);
            if (++w1s == kT_W1Stages) { w1s = 0; w1ph ^= 1; }
          }
          if (LN) {                                    // the chunk's augmented slice travels through the same ring
            mbar_wait(w1_empty(w1s), w1ph ^ 1);
            mbar_expect_tx(w1_full(w1s), kT_KBlockBytes);
            tma_load_2d(sbase + kT_OffW1 + w1s * kT_KBlockBytes, &m->tmAug, w1_full(w1s), 0, c * kT_HC);
            if (++w1s == kT_W1Stages) { w1s = 0; w1ph ^= 1; }
          }
        }
        load_w2(nch - 1, gh + nch - 1);
        gh += (uint32_t)nch;
      }
      T2_STORE(0, clock64() - tr_t0); T2_STORE(1, tr_q); T2_STORE(2, tr_xe); T2_STORE(3, tr_w1e); T2_STORE(4, tr_w2e);
    }
  } else if (warp == 1) {
    // ------------------------------------------ MMA issuer, layer 1 ----
    // acc1[g & 1] = X . W1_c^T for every hidden chunk; never waits for the hidden tile, so the tensor pipe always
    // has layer-1 work queued while the epilogue warps convert the previous chunk.
    if (lane == 0) {
      int qs = 0; uint32_t qph = 0;
      int w1s = 0; uint32_t w1ph = 0;
      uint32_t gt = 0, g = 0;
      const uint64_t xd0 = umma_desc_sw128(sbase + kT_OffX), wd0 = umma_desc_sw128(sbase + kT_OffW1);
      constexpr uint64_t kKB = kT_KBlockBytes >> 4;            // descriptor address units (16 bytes) per k-block
      T2_DECL(tr_t0); T2_DECL(tr_q); T2_DECL(tr_a1e); T2_DECL(tr_xf); T2_DECL(tr_w1f); T2_DECL(tr_tiles); T2_DECL(tr_tc);
      T2_NOW(tr_t0);
      for (;;) {
        T2_WAIT(tr_q, mbar_wait(q_full(qs), qph));
        const uint4 e0 = lds128(q_slot(qs) + kQEntryOff);
        mbar_arrive(q_empty(qs));
        if (++qs == kT_QDepth) { qs = 0; qph ^= 1; }
        if ((int)e0.x < 0) break;
        const int H = (int)(e0.z & 0xFFFFu), nkb1 = (int)((e0.z >> 16) & 0xFFu), klast1 = (int)(e0.z >> 24);
        const int nch = (H + kT_HC - 1) / kT_HC;
        for (int c = 0; c < nch; ++c, ++g) {
          const uint32_t s = g & 1u;
          const uint32_t idesc1 = l2_idesc(min(kT_HC, H - c * kT_HC));
          T2_WAIT(tr_a1e, mbar_wait(a1_empty(s), ((g >> 1) & 1u) ^ 1u));      // epilogue has drained this acc1 stage
          if (c == 0) T2_WAIT(tr_xf, mbar_wait(xa_full, gt & 1u));
          T2_ADD(tr_tc, (min(kT_HC, H - c * kT_HC) / 2) * ((nkb1 - 1) * 4 + klast1) + (min(kT_HC, H - c * kT_HC) / 16) * ((int)(e0.w >> 16) / 2));
          tc_fence_after();
          const uint32_t acc1 = tmem_base + s * 128u;
          for (int kb = 0; kb < nkb1; ++kb) {
            T2_WAIT(tr_w1f, mbar_wait(w1_full(w1s), w1ph));
            tc_fence_after();
            const uint64_t adesc = xd0 + (uint64_t)kb * kKB, bdesc = wd0 + (uint64_t)w1s * kKB;
            if (kb + 1 < nkb1) {                             // +32 bytes (= +2 encoded) per K=16 step
              tc_mma_bf16(acc1, adesc, bdesc, idesc1, kb != 0);
              tc_mma_bf16(acc1, adesc + 2, bdesc + 2, idesc1, 1);
              tc_mma_bf16(acc1, adesc + 4, bdesc + 4, idesc1, 1);
              tc_mma_bf16(acc1, adesc + 6, bdesc + 6, idesc1, 1);
            } else {
              for (int k = 0; k < klast1; ++k) tc_mma_bf16(acc1, adesc + 2 * k, bdesc + 2 * k, idesc1, (kb | k) != 0);
            }
            tc_commit(w1_empty(w1s));
            if (++w1s == kT_W1Stages) { w1s = 0; w1ph ^= 1; }
          }
          if (LN) {                                          // + (-mu_r s_n + sigma_r c_n): one K=16 step
            if (c == 0) mbar_wait(st_full(gt & 1u), (gt >> 1) & 1u);   // the epilogue warps have written the A slice
            mbar_wait(w1_full(w1s), w1ph);
            tc_fence_after();
            tc_mma_bf16(acc1, umma_desc_sw128(aug_base), wd0 + (uint64_t)w1s * kKB, idesc1, 1);
            tc_commit(w1_empty(w1s));
            if (++w1s == kT_W1Stages) { w1s = 0; w1ph ^= 1; }
          }
          tc_commit(a1_full(s));
          if (c == nch - 1) tc_commit(xa_empty);             // the X tile may be replaced
        }
        ++gt;
        T2_ADD(tr_tiles, 1);
      }
      T2_STORE(5, clock64() - tr_t0); T2_STORE(6, tr_q); T2_STORE(7, tr_a1e); T2_STORE(8, tr_xf); T2_STORE(9, tr_w1f);
      T2_STORE(10, tr_tiles); T2_STORE(11, tr_tc);
    }
  } else if (warp == kT_Mma2Warp) {
    // ------------------------------------------ MMA issuer, layer 2 ----
    // acc2 (+)= h_c . W2_c^T as soon as the epilogue has published the hidden tile of chunk c.
    if (lane == 0) {
      int qs = 0; uint32_t qph = 0;
      uint32_t gt = 0, g = 0;
      const uint64_t w2d0 = umma_desc_sw128(sbase + kT_OffW2);
      constexpr uint64_t kW2KB = kT_W2KBlockBytes >> 4;
      T2_DECL(tr_t0); T2_DECL(tr_q); T2_DECL(tr_a2e); T2_DECL(tr_w2f); T2_DECL(tr_hf);
      T2_NOW(tr_t0);
      for (;;) {
        T2_WAIT(tr_q, mbar_wait(q_full(qs), qph));
        const uint4 e0 = lds128(q_slot(qs) + kQEntryOff);
        mbar_arrive(q_empty(qs));
        if (++qs == kT_QDepth) { qs = 0; qph ^= 1; }
        if ((int)e0.x < 0) break;
        const int H = (int)(e0.z & 0xFFFFu), N = (int)(e0.w >> 16);
        const int nch = (H + kT_HC - 1) / kT_HC;
        const uint32_t acc2 = tmem_base + kT_TmemAcc2 + (gt & 1u) * 64u;
        const uint32_t idesc2 = l2_idesc(N);
        T2_WAIT(tr_a2e, mbar_wait(a2_empty(gt & 1u), ((gt >> 1) & 1u) ^ 1u));   // the epilogue has drained this acc2 stage
        for (int c = 0; c < nch; ++c, ++g) {
          const uint32_t s = g & 1u;
          const int ksteps = min(kT_HC, H - c * kT_HC) / 16;
          T2_WAIT(tr_hf, mbar_wait(h_full(s), (g >> 1) & 1u));
          T2_WAIT(tr_w2f, mbar_wait(w2_full(s), (g >> 1) & 1u));
          tc_fence_after();
          const uint64_t wd = w2d0 + (uint64_t)s * 2 * kW2KB;
          const uint32_t ht = tmem_base + kT_TmemH + s * 64u;                // A operand: 8 TMEM columns per K=16 step
          for (int k = 0; k < ksteps; ++k) {
            const uint64_t j = (uint64_t)(k >> 2), kk = (uint64_t)(k & 3);   // k-block of W2, K=16 step inside it
            tc_mma_bf16_ts(acc2, ht + 8u * (uint32_t)k, wd + j * kW2KB + 2 * kk, idesc2, (c | k) != 0);
          }
          tc_commit(h_empty(s));
          tc_commit(w2_empty(s));
        }
        tc_commit(a2_full(gt & 1u));
        ++gt;
      }
      T2_STORE(12, clock64() - tr_t0); T2_STORE(13, tr_q); T2_STORE(14, tr_a2e); T2_STORE(15, tr_w2f); T2_STORE(16, tr_hf);
    }
  } else {
    // ----------------------------------------------------------- epilogue ----
    // Per hidden chunk: acc1 -> registers -> + b1, act1, RNE -> the hidden tile in shared memory (layer-2 A operand).
    // The layer-2 accumulator of a row tile is drained LATE, after the first hidden chunk of the NEXT tile has been
    // published: by then its MMAs have long retired, so the warps never sit waiting for them.
    const int ew = warp - kT_FirstEpiWarp;
    const int quad = warp & 3;               // TMEM lane quadrant this warp may read
    const int half = ew >> 2;                // which 64-column half of a 128-wide hidden chunk
    const uint32_t lane_off = (uint32_t)(quad * 32) << 16;
    int qs = 0; uint32_t qph = 0;
    uint32_t gt = 0, gh = 0;
    // the tile whose layer-2 accumulator is still to be drained
    bool pend = false;
    uint32_t p_slot = 0, p_gt = 0;
    int p_qs = 0, p_act2 = 0, p_m0 = 0;
    const L2Member* p_m = nullptr;
    const uint32_t sbuf = sbase + kT_OffOut + (uint32_t)quad * 4096u;  // output staging (warps with half == 0)
    T2_DECL(tr_t0); T2_DECL(tr_q); T2_DECL(tr_a1f); T2_DECL(tr_he); T2_DECL(tr_a2f); T2_DECL(tr_st); T2_DECL(tr_drain); T2_DECL(tr_xf);
    T2_DECL(tr_s_ld); T2_DECL(tr_s_math); T2_DECL(tr_s_sts); T2_DECL(tr_s_fence); T2_DECL(tr_chunks);
    T2_NOW(tr_t0);
    auto drain = [&]() {
      T2_DECL(tr_d0); T2_NOW(tr_d0);
      const uint32_t s2 = p_gt & 1u;
      T2_WAIT(tr_a2f, mbar_wait(a2_full(s2), (p_gt >> 1) & 1u));
      tc_fence_after();
      uint32_t v[64], p[32];
      {
        const uint32_t t = tmem_base + lane_off + kT_TmemAcc2 + s2 * 64u;
        tc_ld_32x32(t, *reinterpret_cast<uint32_t(*)[32]>(&v[0]));
        tc_ld_32x32(t + 32, *reinterpret_cast<uint32_t(*)[32]>(&v[32]));
        tc_wait_ld();
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(a2_empty(s2));
      if (half == 0) {
        if constexpr (LN) epi_act_b16(v, p_slot + kOffB2, p_act2, p);
        else epi_act(v, p_slot + kOffB2, p_act2, p);
      }
      if (half == 0) {
        T2_WAIT(tr_st, if (lane == 0) tma_store_wait_read<0>());       // this warp's previous store has read the staging tile
        __syncwarp();
#pragma unroll
        for (int j = 0; j < 8; ++j)
          sts128(sbuf + lane * 128 + ((j ^ (lane & 7)) << 4), make_uint4(p[4 * j], p[4 * j + 1], p[4 * j + 2], p[4 * j + 3]));
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
          tma_store_2d(&p_m->tmY, sbuf, 0, p_m0 + quad * 32);
          tma_store_commit();
        }
      }
      __syncwarp();                          // every lane has read the slot's b2
      if (lane == 0) mbar_arrive(q_empty(p_qs));
      T2_ADD(tr_drain, clock64() - tr_d0);
    };
    for (;;) {
      T2_WAIT(tr_q, mbar_wait(q_full(qs), qph));
      const uint32_t slot = q_slot(qs);
      const uint4 e0 = lds128(slot + kQEntryOff);
      if ((int)e0.x < 0) break;
      const L2Member* m = members + (int)e0.x;
      const int m0 = (int)e0.y;
      const int H = (int)(e0.z & 0xFFFFu);
      const int act1 = (int)(e0.w & 0xFFu), act2 = (int)((e0.w >> 8) & 0xFFu);
      const int nch = (H + kT_HC - 1) / kT_HC;
      float lnA = 0.f;                                // LN: rstd of this thread's row
      if constexpr (LN) {
        // Row statistics from the resident X tile while MMA1 runs on it: the two threads of a row (the warps of one
        // TMEM quadrant) take alternate 16-byte pieces, shifted single pass (shift = the row's first element),
        // partial sums exchanged through shared memory; the half-0 thread writes the row's augmented A slice
        // (-mu_h, -mu_h, -mu_l, sigma_h, sigma_h, sigma_l, 0...).
        const uint4 e1 = lds128(slot + kQEntryOff + 16);           // LN: the b1 field holds K | eps << 32 (no global load on the per-tile chain)
        const int K = (int)e1.x;
        const float eps = __uint_as_float(e1.y);
        const uint32_t ss = gt & 1u;
        T2_WAIT(tr_xf, mbar_wait(xa_full, gt & 1u));
        const int r0 = quad * 32 + lane;
        const uint32_t a0 = sbase + kT_OffX + (uint32_t)r0 * 128u;
        const uint32_t x7 = (uint32_t)(lane & 7);                   // r0 & 7
        const float s0 = bf16_lo(lds128(a0 + (x7 << 4)).x);
        const f32x2 ns = pk2(-s0, -s0);
        f32x2 sumA = pk2(0.f, 0.f), sumB = sumA, sqA = sumA, sqB = sumA;
        const int nv = K >> 3;
#pragma unroll 4
        for (int c = half; c < nv; c += 2) {
          const uint4 u = lds128(a0 + (uint32_t)(c >> 3) * kT_KBlockBytes + ((((uint32_t)c & 7u) ^ x7) << 4));
          const f32x2 d0 = add2(bf2_to_f2(u.x), ns), d1 = add2(bf2_to_f2(u.y), ns);
          const f32x2 d2 = add2(bf2_to_f2(u.z), ns), d3 = add2(bf2_to_f2(u.w), ns);
          sumA = add2(sumA, d0); sqA = fma2(d0, d0, sqA);
          sumB = add2(sumB, d1); sqB = fma2(d1, d1, sqB);
          sumA = add2(sumA, d2); sqA = fma2(d2, d2, sqA);
          sumB = add2(sumB, d3); sqB = fma2(d3, d3, sqB);
        }
        float psum = sum2(add2(sumA, sumB)), psq = sum2(add2(sqA, sqB));
        const uint32_t mine_addr = stats_base + ((uint32_t)half * kT_BM + (uint32_t)r0) * 8u;
        const uint32_t peer_addr = stats_base + ((uint32_t)(half ^ 1) * kT_BM + (uint32_t)r0) * 8u;
        asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(mine_addr), "f"(psum), "f"(psq) : "memory");
        asm volatile("bar.sync %0, 64;" ::"r"(1 + quad) : "memory");
        float osum, osq;
        asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(osum), "=f"(osq) : "r"(peer_addr) : "memory");
        asm volatile("bar.sync %0, 64;" ::"r"(1 + quad) : "memory");    // both have read before either writes the next tile's
        // same order in both threads: (half 0) + (half 1)
        const float tsum = half ? osum + psum : psum + osum, tsq = half ? osq + psq : psq + osq;
        const float inv = 1.f / (float)K;
        const float m0 = tsum * inv;
        const float sig = sqrtf(fmaxf(fmaf(-m0, m0, tsq * inv), 0.f) + eps), nmu = -(s0 + m0);
        lnA = 1.f / sig;
        if (half == 0) {
          const uint32_t mh = pack_bf16x2(nmu, 0.f) & 0xFFFFu, gh2 = pack_bf16x2(sig, 0.f) & 0xFFFFu;
          const uint32_t ml = pack_bf16x2(nmu - bf16_lo(mh), 0.f) & 0xFFFFu, gl = pack_bf16x2(sig - bf16_lo(gh2), 0.f) & 0xFFFFu;
          const uint32_t arow = aug_base + (uint32_t)r0 * 128u;
          // (single-buffered: X(t+1) only lands after every MMA1 of tile t, the slice's last reader, has retired)
          sts128(arow + (x7 << 4), make_uint4(mh | (mh << 16), ml | (gh2 << 16), gh2 | (gl << 16), 0u));
          sts128(arow + ((1u ^ x7) << 4), make_uint4(0u, 0u, 0u, 0u));
          fence_proxy_async_smem();                    // the A slice is read by the tensor core
        }
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(xa_empty);
          if (half == 0) mbar_arrive(st_full(ss));
        }
      }
      for (int c = 0; c < nch; ++c) {
        const uint32_t g = gh + (uint32_t)c;
        const int s = (int)(g & 1u);
        const uint32_t ph = (g >> 1) & 1u;
        const int bn = min(kT_HC, H - c * kT_HC);
        const bool mine = half * 64 < bn;            // this warp's 64 columns exist in the chunk
        T2_WAIT(tr_a1f, mbar_wait(a1_full(s), ph));
        tc_fence_after();
        const uint32_t t = tmem_base + lane_off + (uint32_t)s * 128u + (uint32_t)half * 64u;
        {                                              // (columns past the chunk's width hold stale data: never used)
          uint32_t v[64], p[32];
          T2_DECL(tq0); T2_DECL(tq1); T2_DECL(tq2); T2_DECL(tq3); T2_DECL(tq4);
          T2_NOW(tq0);
          tc_ld_32x32(t, *reinterpret_cast<uint32_t(*)[32]>(&v[0]));
          tc_ld_32x32(t + 32, *reinterpret_cast<uint32_t(*)[32]>(&v[32]));
          tc_wait_ld();
          T2_NOW(tq1);
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(a1_empty(s));     // acc1 stage is in registers: MMA1 of chunk c+2 may overwrite it
          if constexpr (LN) epi_act_ln(v, lnA, act1, p);
          else epi_act(v, slot + (uint32_t)(c * kT_HC + half * 64) * 4u, act1, p);
          T2_NOW(tq2);
          // the hidden tile lives in TENSOR MEMORY (two buffers of 64 columns: a column holds two consecutive hidden
          // units of this thread's row): MMA2 of chunk c-2 has long retired
          T2_WAIT(tr_he, mbar_wait(h_empty(s), ph ^ 1u));
          T2_NOW(tq3);
          tc_fence_after();
          if (mine) tc_st_32x32(tmem_base + lane_off + kT_TmemH + (uint32_t)s * 64u + (uint32_t)half * 32u, p);
          tc_wait_st();
          T2_NOW(tq4);
          T2_ADD(tr_s_ld, tq1 - tq0); T2_ADD(tr_s_math, tq2 - tq1); T2_ADD(tr_s_sts, tq4 - tq3);
        }
        T2_DECL(tq5); T2_NOW(tq5);
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(h_full(s));
        T2_ADD(tr_s_fence, clock64() - tq5); T2_ADD(tr_chunks, 1);
        if (c == 0 && pend) { drain(); pend = false; }
      }
      gh += (uint32_t)nch;
      pend = true;
      p_slot = slot; p_gt = gt; p_qs = qs; p_act2 = act2; p_m0 = m0; p_m = m;
      ++gt;
      if (++qs == kT_QDepth) { qs = 0; qph ^= 1; }
    }
    if (pend) drain();
    if (lane == 0) tma_store_wait_all();
    if (ew == 0 && lane == 0) {
      T2_STORE(17, clock64() - tr_t0); T2_STORE(18, tr_q); T2_STORE(19, tr_a1f); T2_STORE(20, tr_he); T2_STORE(21, tr_a2f);
      T2_STORE(22, tr_st); T2_STORE(23, tr_drain); T2_STORE(24, tr_xf);
      T2_STORE(25, tr_s_ld); T2_STORE(26, tr_s_math); T2_STORE(27, tr_s_sts); T2_STORE(28, tr_s_fence); T2_STORE(29, tr_chunks);
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kT_TmemCols) : "memory");
  }
}

#ifdef OPTB_GEMM_TRACE
// trace build only: where the chained kernel writes its per-CTA wait-cycle records ([grid][32] uint64), or NULL
extern "C" int opt_trace_set_linear2_buffer(void* device_buffer) {
  unsigned long long* p = static_cast<unsigned long long*>(device_buffer);
  return (int)cudaMemcpyToSymbol(optb::g_l2_trace, &p, sizeof p);
}
#endif

cudaError_t launch_linear2(const opt_plan* p, cudaStream_t s) {
  char* base = static_cast<char*>(p->dev_tables);
  const L2Member* mem = reinterpret_cast<const L2Member*>(base + p->off0);
  const uint4* chunks = reinterpret_cast<const uint4*>(base + p->off1);
  int* counters = reinterpret_cast<int*>(base + p->off2);
  if (p->kind == kPlanLnLinear2)       // counters (256 B) | per-member flags | fold table
    grouped_linear2_sm100_kernel<true><<<p->grid, p->block, p->smem, s>>>(
        mem, chunks, p->n_chunks, counters, reinterpret_cast<const L2Fold*>(base + p->off3), counters + 64, p->n_members);
  else
    grouped_linear2_sm100_kernel<false><<<p->grid, p->block, p->smem, s>>>(mem, chunks, p->n_chunks, counters, nullptr, nullptr, 0);
  return cudaGetLastError();
}

}  // namespace optb

using namespace optb;

namespace {
// one planner for both entry points: lnm == nullptr -> plain chain (members), else LayerNorm + chain (lnm[i].chain)
opt_status create_linear2(const opt_linear2_member* members, const opt_ln_linear2_member* lnm, int32_t n, opt_dtype io,
                          int device, opt_plan** plan) {
  const bool LN = lnm != nullptr;
  auto M_ = [&](int32_t i) -> const opt_linear2_member& { return LN ? lnm[i].chain : members[i]; };
  if (plan) *plan = nullptr;
  if (!plan || (!members && !lnm)) return fail(OPT_ERR_INVALID_ARG, "opt_linear2_plan_create: NULL argument");
  if (n < 1 || n > 65535) return fail(OPT_ERR_INVALID_ARG, "n = %d outside [1, 65535]", n);
  if (io != OPT_F32 && io != OPT_BF16) return fail(OPT_ERR_INVALID_ARG, "bad io dtype %d", (int)io);
  if (io != OPT_BF16) return fail(OPT_ERR_UNSUPPORTED, "chained Linear is implemented for bf16 groups only");
  std::vector<Region> regions;
  int64_t flops = 0, bytes = 0, tiles = 0;
  for (int32_t i = 0; i < n; ++i) {
    const opt_linear2_member& m = M_(i);
    if (!m.x || !m.w1 || !m.w2 || !m.y) return fail(OPT_ERR_INVALID_ARG, "member %d: NULL pointer", i);
    if (m.M < 1 || m.K < 1 || m.H < 1 || m.N < 1)
      return fail(OPT_ERR_INVALID_ARG, "member %d: M=%d K=%d H=%d N=%d must be >= 1", i, m.M, m.K, m.H, m.N);
    if (m.act1 < OPT_ACT_NONE || m.act1 > OPT_ACT_SIGMOID || m.act2 < OPT_ACT_NONE || m.act2 > OPT_ACT_SIGMOID)
      return fail(OPT_ERR_INVALID_ARG, "member %d: bad activation", i);
    if ((m.M > 1 && (m.ldx < m.K || m.ldy < m.N)) || (m.H > 1 && m.ldw1 < m.K) || (m.N > 1 && m.ldw2 < m.H))
      return fail(OPT_ERR_INVALID_ARG, "member %d: row stride smaller than the row", i);
    if (!aligned16(m.x) || !aligned16(m.w1) || !aligned16(m.w2) || !aligned16(m.y) || !aligned16(m.b1) || !aligned16(m.b2))
      return fail(OPT_ERR_ALIGNMENT, "member %d: pointers must be 16-byte aligned", i);
    if (m.K % 8 || m.ldx % 8 || m.ldw1 % 8 || m.ldw2 % 8 || m.ldy % 8)
      return fail(OPT_ERR_ALIGNMENT, "member %d: K and the row strides must be multiples of 8 (PAPER.md:445)", i);
    if (m.H % 16 || m.N % 16)
      return fail(OPT_ERR_ALIGNMENT, "member %d: H=%d and N=%d must be multiples of 16 (tensor-core N / K granularity)", i, m.H, m.N);
    if (m.K > kT_MaxK || m.H > kT_MaxH || m.N > kT_MaxN)
      return fail(OPT_ERR_UNSUPPORTED, "member %d: K=%d H=%d N=%d outside the on-chip limits K<=%d H<=%d N<=%d", i, m.K, m.H,
                  m.N, kT_MaxK, kT_MaxH, kT_MaxN);
    regions.push_back({(uintptr_t)m.x, m.ldx * 2, (int64_t)m.K * 2, m.M, false, i});
    regions.push_back({(uintptr_t)m.w1, m.ldw1 * 2, (int64_t)m.K * 2, m.H, false, i});
    regions.push_back({(uintptr_t)m.w2, m.ldw2 * 2, (int64_t)m.H * 2, m.N, false, i});
    if (m.b1) regions.push_back({(uintptr_t)m.b1, 0, (int64_t)m.H * 2, 1, false, i});
    if (m.b2) regions.push_back({(uintptr_t)m.b2, 0, (int64_t)m.N * 2, 1, false, i});
    regions.push_back({(uintptr_t)m.y, m.ldy * 2, (int64_t)m.N * 2, m.M, true, i});
    if (LN) {
      const opt_ln_linear2_member& l = lnm[i];
      if (!aligned16(l.gamma) || !aligned16(l.beta)) return fail(OPT_ERR_ALIGNMENT, "member %d: pointers must be 16-byte aligned", i);
      if (!(l.eps >= 0.f)) return fail(OPT_ERR_INVALID_ARG, "member %d: eps must be >= 0", i);
      if (l.gamma) regions.push_back({(uintptr_t)l.gamma, 0, (int64_t)m.K * 2, 1, false, i});
      if (l.beta) regions.push_back({(uintptr_t)l.beta, 0, (int64_t)m.K * 2, 1, false, i});
      bytes += ((l.gamma ? m.K : 0) + (l.beta ? m.K : 0)) * 2;
      flops += 2ll * m.H * m.K;                              // the fold: W1 diag(gamma), s, c
    }
    flops += 2ll * m.M * m.H * (m.K + m.N);
    bytes += ((int64_t)m.M * m.K + (int64_t)m.H * m.K + (m.b1 ? m.H : 0) + (int64_t)m.N * m.H + (m.b2 ? m.N : 0) +
              (int64_t)m.M * m.N) * 2;
    tiles += (m.M + kT_BM - 1) / kT_BM;
  }
  if (tiles > INT32_MAX / 2) return fail(OPT_ERR_UNSUPPORTED, "too many tiles");
  if (opt_status st = check_independent(regions, /*allow_inplace_self=*/false)) return st;

  int num_sms = 0;
  DeviceGuard device_guard;      // the caller's current device is restored on return
  if (opt_status st = open_device(device, &num_sms)) return st;
  EncodeTiledFn enc = nullptr;
  if (opt_status st = get_encoder(&enc)) return st;
  auto align_up = [](size_t x) { return (x + 255) & ~size_t(255); };
  // LN: workspace = per member  W1g [H,K] bf16 | augmented slice [H,16] bf16
  std::vector<L2Fold> folds(LN ? n : 0);
  char* ws = nullptr;
  if (LN) {
    size_t wbytes = 0;
    std::vector<size_t> offs(n);
    for (int32_t i = 0; i < n; ++i) {
      offs[i] = wbytes;
      wbytes += align_up((size_t)M_(i).H * M_(i).K * 2) + align_up((size_t)M_(i).H * 32);
    }
    cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&ws), wbytes);
    if (e != cudaSuccess) return fail(OPT_ERR_CUDA, "workspace allocation (%zu bytes) failed: %s", wbytes, cudaGetErrorString(e));
    for (int32_t i = 0; i < n; ++i) {
      const opt_linear2_member& m = M_(i);
      L2Fold& f = folds[i];
      memset(&f, 0, sizeof f);
      f.w1 = static_cast<const uint16_t*>(m.w1); f.ldw1 = m.ldw1;
      f.gamma = static_cast<const uint16_t*>(lnm[i].gamma); f.beta = static_cast<const uint16_t*>(lnm[i].beta);
      f.b1 = static_cast<const uint16_t*>(m.b1);
      f.w1g = reinterpret_cast<uint16_t*>(ws + offs[i]);
      f.aug = reinterpret_cast<uint16_t*>(ws + offs[i] + align_up((size_t)m.H * m.K * 2));
      f.H = m.H; f.K = m.K; f.eps = lnm[i].eps;
    }
  }
  struct WsGuard { char* p; ~WsGuard() { if (p) cudaFree(p); } } ws_guard{ws};     // freed on every error path
  std::vector<L2Member> tab(n);
  memset(tab.data(), 0, tab.size() * sizeof(L2Member));
  std::vector<TileEntry2> flat;
  flat.reserve((size_t)tiles);
  for (int32_t i = 0; i < n; ++i) {
    const opt_linear2_member& m = M_(i);
    L2Member& t = tab[i];
    opt_status st;
    if ((st = encode_2d(enc, &t.tmX, m.x, m.M, m.K, m.ldx, kT_BK, kT_BM, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, "X", i)) ||
        (st = encode_2d(enc, &t.tmW1, LN ? (const void*)folds[i].w1g : m.w1, m.H, m.K, LN ? (int64_t)m.K : m.ldw1, kT_BK, kT_HC,
                        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, "W1", i)) ||
        (st = encode_2d(enc, &t.tmW2, m.w2, m.N, m.H, m.ldw2, kT_BK, m.N, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, "W2", i)) ||
        (st = encode_2d(enc, &t.tmY, m.y, m.M, m.N, m.ldy, 64, 32, CU_TENSOR_MAP_L2_PROMOTION_NONE, "Y", i)) ||
        (LN && (st = encode_2d(enc, &t.tmAug, folds[i].aug, m.H, 16, 16, kT_BK, kT_HC, CU_TENSOR_MAP_L2_PROMOTION_NONE, "aug", i))))
      return st;
    const int nkb1 = (m.K + kT_BK - 1) / kT_BK, klast1 = (m.K - (nkb1 - 1) * kT_BK + 15) / 16;
    for (int mb = 0; mb < (m.M + kT_BM - 1) / kT_BM; ++mb) {
      TileEntry2 e;
      e.member = i; e.m0 = mb * kT_BM;
      e.shape = (uint32_t)m.H | ((uint32_t)nkb1 << 16) | ((uint32_t)klast1 << 24);
      e.misc = (uint32_t)m.act1 | ((uint32_t)m.act2 << 8) | ((uint32_t)m.N << 16);
      e.b2 = m.b2;
      if (LN) {      // no b1 operand (folded into c): the slot carries K and eps for the row statistics
        uint32_t eps_bits;
        memcpy(&eps_bits, &folds[i].eps, 4);
        e.b1 = reinterpret_cast<const void*>((uintptr_t)((uint64_t)(uint32_t)m.K | ((uint64_t)eps_bits << 32)));
      } else {
        e.b1 = m.b1;
      }
      flat.push_back(e);
    }
  }
  // chunks of 4 tiles (one table line, one atomic), strided so that neighbouring CTAs work on neighbouring row tiles
  // of one member (its W1 / W2 stay hot in L2); the last 3 waves one tile per chunk
  TileEntry2 pad_entry;
  memset(&pad_entry, 0, sizeof pad_entry);
  pad_entry.member = -1;
  const size_t tail = std::min(flat.size(), (size_t)3 * num_sms);
  const size_t body = flat.size() - tail;
  const size_t nC = (body + 3) / 4;
  std::vector<TileEntry2> chunked;
  for (size_t c = 0; c < nC; ++c)
    for (int g = 0; g < 4; ++g) {
      const size_t k = (size_t)g * nC + c;
      chunked.push_back(k < body ? flat[k] : pad_entry);
    }
  for (size_t k = body; k < flat.size(); ++k) {
    chunked.push_back(flat[k]);
    for (int g = 1; g < 4; ++g) chunked.push_back(pad_entry);
  }
  const int64_t n_chunks = (int64_t)(chunked.size() / 4);

  opt_plan* p = new opt_plan();
  p->kind = LN ? kPlanLnLinear2 : kPlanLinear2; p->device = device; p->io = io; p->n_members = n; p->flops = flops; p->bytes = bytes;
  p->off0 = 0;
  p->off1 = align_up(tab.size() * sizeof(L2Member));
  p->off2 = p->off1 + align_up(chunked.size() * sizeof(TileEntry2));
  // scheduler counters (256 bytes: chunk, done, LN epoch), then LN: per-member flags, fold table; zero-initialised
  p->off3 = p->off2 + 256 + align_up((size_t)(LN ? n : 0) * 4);
  const size_t total = p->off3 + folds.size() * sizeof(L2Fold);
  std::vector<char> blob(total, 0);
  if (LN) memcpy(blob.data() + p->off3, folds.data(), folds.size() * sizeof(L2Fold));
  memcpy(blob.data(), tab.data(), tab.size() * sizeof(L2Member));
  memcpy(blob.data() + p->off1, chunked.data(), chunked.size() * sizeof(TileEntry2));
  if (opt_status st = upload_tables(p, blob.data(), total)) { delete p; return st; }
  const int smem_bytes = LN ? L2Cfg<true>::kSmemBytes : L2Cfg<false>::kSmemBytes;
  // (per instantiation, a compile-time constant: every plan of this kernel sets the same value)
  cudaError_t e = LN ? cudaFuncSetAttribute(grouped_linear2_sm100_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes)
                     : cudaFuncSetAttribute(grouped_linear2_sm100_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
  if (e != cudaSuccess) {
    cudaFree(p->dev_tables); delete p;
    return fail(OPT_ERR_CUDA, "cudaFuncSetAttribute(max dynamic smem %d) failed: %s", smem_bytes, cudaGetErrorString(e));
  }
  p->grid = dim3((unsigned)std::min<int64_t>(n_chunks, num_sms));
  p->block = dim3(LN ? L2Cfg<true>::kThreads : L2Cfg<false>::kThreads); p->smem = smem_bytes;
  p->total_tiles = (int32_t)tiles; p->n_chunks = (int32_t)n_chunks;
  p->workspace = ws; ws_guard.p = nullptr;
  *plan = p;
  return OPT_OK;
}
}  // namespace

extern "C" opt_status opt_linear2_plan_create(const opt_linear2_member* members, int32_t n, opt_dtype io, int device,
                                              opt_plan** plan) {
  return create_linear2(members, nullptr, n, io, device, plan);
}

extern "C" opt_status opt_ln_linear2_plan_create(const opt_ln_linear2_member* members, int32_t n, opt_dtype io, int device,
                                                 opt_plan** plan) {
  if (!members) { if (plan) *plan = nullptr; return fail(OPT_ERR_INVALID_ARG, "opt_ln_linear2_plan_create: NULL argument"); }
  return create_linear2(nullptr, members, n, io, device, plan);
}
