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
#include <algorithm>
#include <cstdlib>

#include "sm100_ptx.h"

namespace optb {

constexpr int kT_BM = 128;            // tile rows
constexpr int kT_BK = 64;             // k-block: one 128-byte swizzle row of bf16
constexpr int kT_HC = 128;            // hidden chunk: UMMA N of layer 1, K of layer 2 per chunk
constexpr int kT_MaxK = 256;          // layer-1 K (input features): the X tile is at most 4 k-blocks
constexpr int kT_MaxH = 512;          // hidden width: b1 travels in the queue slot
constexpr int kT_MaxN = 64;           // layer-2 N
constexpr int kT_W1Stages = 4;
constexpr int kT_EpiWarps = 8;
constexpr int kT_FirstEpiWarp = 3;
constexpr int kT_Mma2Warp = kT_FirstEpiWarp + kT_EpiWarps;     // warp 11: layer-2 MMA issuer
constexpr int kT_Threads = 32 * (kT_Mma2Warp + 1);
constexpr int kT_KBlockBytes = kT_BM * kT_BK * 2;          // 16 KB: a 128 x 64 bf16 k-block
constexpr int kT_W2KBlockBytes = kT_MaxN * kT_BK * 2;      // 8 KB: a 64 x 64 k-block of W2
constexpr int kT_QDepth = 4;
constexpr int kT_QSlotBytes = kT_MaxH * 2 + kT_MaxN * 2 + 32;     // b1 | b2 | TileEntry2
// shared-memory map
constexpr int kT_OffX = 0;
constexpr int kT_OffW1 = kT_OffX + (kT_MaxK / kT_BK) * kT_KBlockBytes;            //  64 KB
constexpr int kT_OffH = kT_OffW1 + kT_W1Stages * kT_KBlockBytes;                  // +96 KB
constexpr int kT_OffW2 = kT_OffH + 2 * kT_KBlockBytes;                            // +32 KB (one hidden tile: 2 k-blocks)
constexpr int kT_OffOut = kT_OffW2 + 2 * 2 * kT_W2KBlockBytes;                    // +32 KB
constexpr int kT_OffQ = kT_OffOut + 4 * 4096;                                     // +16 KB output staging (4 warps x 32 rows x 128 B)
constexpr int kT_OffBar = kT_OffQ + kT_QDepth * kT_QSlotBytes;
constexpr int kT_SmemBytes = kT_OffBar + 512;
static_assert(kT_SmemBytes <= 227 * 1024, "chained-GEMM shared memory map exceeds 227 KB");
constexpr int kT_TmemCols = 512;      // acc1: columns [0,256), acc2: [256,384)

struct alignas(128) L2Member {
  CUtensorMap tmX;       // X  [M,K]   box {64, 128}  load
  CUtensorMap tmW1;      // W1 [H,K]   box {64, 128}  load
  CUtensorMap tmW2;      // W2 [N,H]   box {64, N}    load
  CUtensorMap tmY;       // Y  [M,N]   box {64, 32}   store
};
static_assert(sizeof(L2Member) == 512, "L2Member keeps tensor maps 128-byte aligned");

struct alignas(16) TileEntry2 {       // member < 0: padding entry of a chunk
  int32_t member, m0;
  uint32_t shape;        // H | K blocks of layer 1 << 16 | K=16 steps in the last K block << 24
  uint32_t misc;         // act1 | act2 << 8 | N << 16
  const void* b1;        // [H] bf16 or NULL
  const void* b2;        // [N] bf16 or NULL
};
static_assert(sizeof(TileEntry2) == 32, "TileEntry2 is two 16-byte vectors");

__device__ __forceinline__ uint32_t l2_idesc(int n) {   // kind::f16, bf16 x bf16 -> fp32, M = 128, K-major A and B
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(kT_BM >> 4) << 24);
}

__device__ __forceinline__ void epi_act(const uint32_t (&v)[64], uint32_t bias_addr, int act, uint32_t (&p)[32]) {
  switch (act) {
    case OPT_ACT_RELU: epi_math<OPT_ACT_RELU>(v, bias_addr, p); break;
    case OPT_ACT_NONE: epi_math<OPT_ACT_NONE>(v, bias_addr, p); break;
    case OPT_ACT_TANH: epi_math<OPT_ACT_TANH>(v, bias_addr, p); break;
    default:           epi_math<OPT_ACT_SIGMOID>(v, bias_addr, p); break;
  }
}

__global__ void __launch_bounds__(kT_Threads, 1)
grouped_linear2_sm100_kernel(const L2Member* __restrict__ members, const uint4* __restrict__ chunks, int n_chunks,
                             int* __restrict__ counters) {
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
  static_assert(16 + 16 * kT_W1Stages + 128 + 16 * kT_QDepth + 4 <= 512, "barrier area");
  auto q_slot = [&](int s) { return sbase + kT_OffQ + (uint32_t)s * kT_QSlotBytes; };
  constexpr uint32_t kQEntryOff = kT_MaxH * 2 + kT_MaxN * 2;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    mbar_init(xa_full, 1); mbar_init(xa_empty, 1);
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
          if (b1 != nullptr && 8 * lane < H) b1a = __ldg(b1 + lane);
          if (b1 != nullptr && 8 * (lane + 32) < H) b1b = __ldg(b1 + lane + 32);
          if (b2 != nullptr && 8 * lane < N) b2v = __ldg(b2 + lane);
          if (lane < 4)
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
        sts128(slot + 16 * lane, c1a);
        sts128(slot + 512 + 16 * lane, c1b);
        if (lane < kT_MaxN / 8) sts128(slot + kT_MaxH * 2 + 16 * lane, c2);
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
      if (atomicAdd(counters + 1, 1) == (int)gridDim.x - 1) { counters[0] = 0; counters[1] = 0; __threadfence(); }
    }
  } else if (warp == 0) {
    // ------------------------------------------------------- TMA producer ----
    // Issue order = the order the MMA warp consumes: X(t); per chunk c: W1 k-blocks of c, then W2 of c-1; W2 of
    // the last chunk.  (A producer that follows the consumer's order cannot deadlock on the three rings.)
    if (lane == 0) {
      int qs = 0; uint32_t qph = 0;
      int w1s = 0; uint32_t w1ph = 0;
      uint32_t gt = 0, gh = 0;                       // tiles / hidden chunks issued so far
      for (;;) {
        mbar_wait(q_full(qs), qph);
        const uint4 e0 = lds128(q_slot(qs) + kQEntryOff);
        mbar_arrive(q_empty(qs));
        if (++qs == kT_QDepth) { qs = 0; qph ^= 1; }
        if ((int)e0.x < 0) break;
        const L2Member* m = members + (int)e0.x;
        const int m0 = (int)e0.y;
        const int H = (int)(e0.z & 0xFFFFu), nkb1 = (int)((e0.z >> 16) & 0xFFu);
        const int N = (int)(e0.w >> 16);
        const int nch = (H + kT_HC - 1) / kT_HC;
        // X tile: resident for the whole tile, reloaded when the last MMA1 of the previous tile has retired
        mbar_wait(xa_empty, (gt & 1u) ^ 1u);
        mbar_expect_tx(xa_full, (uint32_t)nkb1 * kT_KBlockBytes);
        for (int kb = 0; kb < nkb1; ++kb) tma_load_2d(sbase + kT_OffX + kb * kT_KBlockBytes, &m->tmX, xa_full, kb * kT_BK, m0);
        ++gt;
        auto load_w2 = [&](int c, uint32_t g) {       // chunk c's slice of W2: [N, 128] = up to two 64-wide k-blocks
          const int s = (int)(g & 1u);
          const int bn = min(kT_HC, H - c * kT_HC), nkb2 = (bn + kT_BK - 1) / kT_BK;
          mbar_wait(w2_empty(s), ((g >> 1) & 1u) ^ 1u);
          mbar_expect_tx(w2_full(s), (uint32_t)(nkb2 * N * kT_BK * 2));
          for (int j = 0; j < nkb2; ++j)
            tma_load_2d(sbase + kT_OffW2 + s * 2 * kT_W2KBlockBytes + j * kT_W2KBlockBytes, &m->tmW2, w2_full(s),
                        c * kT_HC + j * kT_BK, 0);
        };
        for (int c = 0; c < nch; ++c) {
          for (int kb = 0; kb < nkb1; ++kb) {
            mbar_wait(w1_empty(w1s), w1ph ^ 1);
            mbar_expect_tx(w1_full(w1s), kT_KBlockBytes);
            tma_load_2d(sbase + kT_OffW1 + w1s * kT_KBlockBytes, &m->tmW1, w1_full(w1s), kb * kT_BK, c * kT_HC);
            if (++w1s == kT_W1Stages) { w1s = 0; w1ph ^= 1; }
          }
          if (c >= 1) load_w2(c - 1, gh + c - 1);
        }
        load_w2(nch - 1, gh + nch - 1);
        gh += (uint32_t)nch;
      }
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
      for (;;) {
        mbar_wait(q_full(qs), qph);
        const uint4 e0 = lds128(q_slot(qs) + kQEntryOff);
        mbar_arrive(q_empty(qs));
        if (++qs == kT_QDepth) { qs = 0; qph ^= 1; }
        if ((int)e0.x < 0) break;
        const int H = (int)(e0.z & 0xFFFFu), nkb1 = (int)((e0.z >> 16) & 0xFFu), klast1 = (int)(e0.z >> 24);
        const int nch = (H + kT_HC - 1) / kT_HC;
        for (int c = 0; c < nch; ++c, ++g) {
          const uint32_t s = g & 1u;
          const uint32_t idesc1 = l2_idesc(min(kT_HC, H - c * kT_HC));
          mbar_wait(a1_empty(s), ((g >> 1) & 1u) ^ 1u);      // epilogue has drained this acc1 stage
          if (c == 0) mbar_wait(xa_full, gt & 1u);
          tc_fence_after();
          const uint32_t acc1 = tmem_base + s * 128u;
          for (int kb = 0; kb < nkb1; ++kb) {
            mbar_wait(w1_full(w1s), w1ph);
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
          tc_commit(a1_full(s));
          if (c == nch - 1) tc_commit(xa_empty);             // the X tile may be replaced
        }
        ++gt;
      }
    }
  } else if (warp == kT_Mma2Warp) {
    // ------------------------------------------ MMA issuer, layer 2 ----
    // acc2 (+)= h_c . W2_c^T as soon as the epilogue has published the hidden tile of chunk c.
    if (lane == 0) {
      int qs = 0; uint32_t qph = 0;
      uint32_t gt = 0, g = 0;
      const uint64_t hd0 = umma_desc_sw128(sbase + kT_OffH), w2d0 = umma_desc_sw128(sbase + kT_OffW2);
      constexpr uint64_t kKB = kT_KBlockBytes >> 4, kW2KB = kT_W2KBlockBytes >> 4;
      for (;;) {
        mbar_wait(q_full(qs), qph);
        const uint4 e0 = lds128(q_slot(qs) + kQEntryOff);
        mbar_arrive(q_empty(qs));
        if (++qs == kT_QDepth) { qs = 0; qph ^= 1; }
        if ((int)e0.x < 0) break;
        const int H = (int)(e0.z & 0xFFFFu), N = (int)(e0.w >> 16);
        const int nch = (H + kT_HC - 1) / kT_HC;
        const uint32_t acc2 = tmem_base + 256u + (gt & 1u) * 64u;
        const uint32_t idesc2 = l2_idesc(N);
        mbar_wait(a2_empty(gt & 1u), ((gt >> 1) & 1u) ^ 1u);   // the epilogue has drained this acc2 stage
        for (int c = 0; c < nch; ++c, ++g) {
          const uint32_t s = g & 1u;
          const int ksteps = min(kT_HC, H - c * kT_HC) / 16;
          mbar_wait(w2_full(s), (g >> 1) & 1u);
          mbar_wait(h_full(0), g & 1u);
          tc_fence_after();
          const uint64_t wd = w2d0 + (uint64_t)s * 2 * kW2KB;
          for (int k = 0; k < ksteps; ++k) {
            const uint64_t j = (uint64_t)(k >> 2), kk = (uint64_t)(k & 3);   // k-block, K=16 step inside it
            tc_mma_bf16(acc2, hd0 + j * kKB + 2 * kk, wd + j * kW2KB + 2 * kk, idesc2, (c | k) != 0);
          }
          tc_commit(h_empty(0));
          tc_commit(w2_empty(s));
        }
        tc_commit(a2_full(gt & 1u));
        ++gt;
      }
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
    const uint32_t row_off = (uint32_t)(quad * 32 + lane) * 128u;      // this thread's row inside a k-block
    int qs = 0; uint32_t qph = 0;
    uint32_t gt = 0, gh = 0;
    // the tile whose layer-2 accumulator is still to be drained
    bool pend = false;
    uint32_t p_slot = 0, p_gt = 0;
    int p_qs = 0, p_act2 = 0, p_m0 = 0;
    const L2Member* p_m = nullptr;
    const uint32_t sbuf = sbase + kT_OffOut + (uint32_t)quad * 4096u;  // output staging (warps with half == 0)
    auto drain = [&]() {
      const uint32_t s2 = p_gt & 1u;
      mbar_wait(a2_full(s2), (p_gt >> 1) & 1u);
      tc_fence_after();
      uint32_t v[64], p[32];
      {
        const uint32_t t = tmem_base + lane_off + 256u + s2 * 64u;
        tc_ld_32x32(t, *reinterpret_cast<uint32_t(*)[32]>(&v[0]));
        tc_ld_32x32(t + 32, *reinterpret_cast<uint32_t(*)[32]>(&v[32]));
        tc_wait_ld();
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(a2_empty(s2));
      if (half == 0) {
        epi_act(v, p_slot + kT_MaxH * 2, p_act2, p);
        if (lane == 0) tma_store_wait_read<0>();       // this warp's previous store has read the staging tile
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
    };
    for (;;) {
      mbar_wait(q_full(qs), qph);
      const uint32_t slot = q_slot(qs);
      const uint4 e0 = lds128(slot + kQEntryOff);
      if ((int)e0.x < 0) break;
      const L2Member* m = members + (int)e0.x;
      const int m0 = (int)e0.y;
      const int H = (int)(e0.z & 0xFFFFu);
      const int act1 = (int)(e0.w & 0xFFu), act2 = (int)((e0.w >> 8) & 0xFFu);
      const int nch = (H + kT_HC - 1) / kT_HC;
      for (int c = 0; c < nch; ++c) {
        const uint32_t g = gh + (uint32_t)c;
        const int s = (int)(g & 1u);
        const uint32_t ph = (g >> 1) & 1u;
        const int bn = min(kT_HC, H - c * kT_HC);
        const bool mine = half * 64 < bn;            // this warp's 64 columns exist in the chunk
        mbar_wait(a1_full(s), ph);
        tc_fence_after();
        uint32_t v[64], p[32];
        {                                              // (columns past the chunk's width hold stale data: never used)
          const uint32_t t = tmem_base + lane_off + (uint32_t)s * 128u + (uint32_t)half * 64u;
          tc_ld_32x32(t, *reinterpret_cast<uint32_t(*)[32]>(&v[0]));
          tc_ld_32x32(t + 32, *reinterpret_cast<uint32_t(*)[32]>(&v[32]));
          tc_wait_ld();
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(a1_empty(s));       // acc1 stage is in registers: MMA1 of chunk c+2 may overwrite it
        epi_act(v, slot + (uint32_t)(c * kT_HC + half * 64) * 2u, act1, p);
        // the hidden tile is single-buffered: MMA2 of chunk c-1 has normally retired by the time this chunk's
        // accumulator has been read and converted
        mbar_wait(h_empty(0), (g & 1u) ^ 1u);
        if (mine) {
          const uint32_t hrow = sbase + kT_OffH + (uint32_t)half * kT_KBlockBytes + row_off;
#pragma unroll
          for (int j = 0; j < 8; ++j)                  // K-major, 128-byte swizzle: 16-byte piece j of row r sits at j ^ (r & 7)
            sts128(hrow + ((j ^ (lane & 7)) << 4), make_uint4(p[4 * j], p[4 * j + 1], p[4 * j + 2], p[4 * j + 3]));
        }
        fence_proxy_async_smem();                      // generic-proxy writes -> visible to the tensor core's reads
        __syncwarp();
        if (lane == 0) mbar_arrive(h_full(0));
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
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kT_TmemCols) : "memory");
  }
}

cudaError_t launch_linear2(const opt_plan* p, cudaStream_t s) {
  char* base = static_cast<char*>(p->dev_tables);
  grouped_linear2_sm100_kernel<<<p->grid, p->block, p->smem, s>>>(
      reinterpret_cast<const L2Member*>(base + p->off0), reinterpret_cast<const uint4*>(base + p->off1), p->n_chunks,
      reinterpret_cast<int*>(base + p->off2));
  return cudaGetLastError();
}

}  // namespace optb

using namespace optb;

extern "C" opt_status opt_linear2_plan_create(const opt_linear2_member* members, int32_t n, opt_dtype io, int device,
                                              opt_plan** plan) {
  if (plan) *plan = nullptr;
  if (!plan || !members) return fail(OPT_ERR_INVALID_ARG, "opt_linear2_plan_create: NULL argument");
  if (n < 1 || n > 65535) return fail(OPT_ERR_INVALID_ARG, "n = %d outside [1, 65535]", n);
  if (io != OPT_F32 && io != OPT_BF16) return fail(OPT_ERR_INVALID_ARG, "bad io dtype %d", (int)io);
  if (io != OPT_BF16) return fail(OPT_ERR_UNSUPPORTED, "chained Linear is implemented for bf16 groups only");
  std::vector<Region> regions;
  int64_t flops = 0, bytes = 0, tiles = 0;
  for (int32_t i = 0; i < n; ++i) {
    const opt_linear2_member& m = members[i];
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
    flops += 2ll * m.M * m.H * (m.K + m.N);
    bytes += ((int64_t)m.M * m.K + (int64_t)m.H * m.K + (m.b1 ? m.H : 0) + (int64_t)m.N * m.H + (m.b2 ? m.N : 0) +
              (int64_t)m.M * m.N) * 2;
    tiles += (m.M + kT_BM - 1) / kT_BM;
  }
  if (tiles > INT32_MAX / 2) return fail(OPT_ERR_UNSUPPORTED, "too many tiles");
  if (opt_status st = check_independent(regions, /*allow_inplace_self=*/false)) return st;

  int num_sms = 0;
  if (opt_status st = open_device(device, &num_sms)) return st;
  EncodeTiledFn enc = nullptr;
  if (opt_status st = get_encoder(&enc)) return st;
  auto align_up = [](size_t x) { return (x + 255) & ~size_t(255); };
  std::vector<L2Member> tab(n);
  memset(tab.data(), 0, tab.size() * sizeof(L2Member));
  std::vector<TileEntry2> flat;
  flat.reserve((size_t)tiles);
  for (int32_t i = 0; i < n; ++i) {
    const opt_linear2_member& m = members[i];
    L2Member& t = tab[i];
    opt_status st;
    if ((st = encode_2d(enc, &t.tmX, m.x, m.M, m.K, m.ldx, kT_BK, kT_BM, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, "X", i)) ||
        (st = encode_2d(enc, &t.tmW1, m.w1, m.H, m.K, m.ldw1, kT_BK, kT_HC, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, "W1", i)) ||
        (st = encode_2d(enc, &t.tmW2, m.w2, m.N, m.H, m.ldw2, kT_BK, m.N, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, "W2", i)) ||
        (st = encode_2d(enc, &t.tmY, m.y, m.M, m.N, m.ldy, 64, 32, CU_TENSOR_MAP_L2_PROMOTION_NONE, "Y", i)))
      return st;
    const int nkb1 = (m.K + kT_BK - 1) / kT_BK, klast1 = (m.K - (nkb1 - 1) * kT_BK + 15) / 16;
    for (int mb = 0; mb < (m.M + kT_BM - 1) / kT_BM; ++mb) {
      TileEntry2 e;
      e.member = i; e.m0 = mb * kT_BM;
      e.shape = (uint32_t)m.H | ((uint32_t)nkb1 << 16) | ((uint32_t)klast1 << 24);
      e.misc = (uint32_t)m.act1 | ((uint32_t)m.act2 << 8) | ((uint32_t)m.N << 16);
      e.b1 = m.b1; e.b2 = m.b2;
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
  p->kind = kPlanLinear2; p->device = device; p->io = io; p->n_members = n; p->flops = flops; p->bytes = bytes;
  p->off0 = 0;
  p->off1 = align_up(tab.size() * sizeof(L2Member));
  p->off2 = p->off1 + align_up(chunked.size() * sizeof(TileEntry2));
  const size_t total = p->off2 + 256;                         // two int32 scheduler counters, zero-initialised
  std::vector<char> blob(total, 0);
  memcpy(blob.data(), tab.data(), tab.size() * sizeof(L2Member));
  memcpy(blob.data() + p->off1, chunked.data(), chunked.size() * sizeof(TileEntry2));
  if (opt_status st = upload_tables(p, blob.data(), total)) { delete p; return st; }
  cudaError_t e = cudaFuncSetAttribute(grouped_linear2_sm100_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kT_SmemBytes);
  if (e != cudaSuccess) {
    cudaFree(p->dev_tables); delete p;
    return fail(OPT_ERR_CUDA, "cudaFuncSetAttribute(max dynamic smem %d) failed: %s", kT_SmemBytes, cudaGetErrorString(e));
  }
  p->grid = dim3((unsigned)std::min<int64_t>(n_chunks, num_sms)); p->block = dim3(kT_Threads); p->smem = kT_SmemBytes;
  p->total_tiles = (int32_t)tiles; p->n_chunks = (int32_t)n_chunks;
  *plan = p;
  return OPT_OK;
}
