// Grouped Linear (+bias +activation): N independent  Y_i = act_i(X_i W_i^T + b_i)
// in ONE launch -- batch_linear / batch_linear_post_grad with the epilogue
// fused (PAPER.md:292, :148 group fusion; include/optimus_b200.h).
//
// Two kernels:
//   grouped_gemm_sm100_kernel  bf16 in/out, fp32 accumulate.  Persistent, one CTA
//       per SM; by default the CTAs work as PAIRS (cluster of 2, tcgen05
//       cta_group::2) on 256 x BN tiles -- each CTA stages its 128 rows of X and
//       half of the W tile, the leader issues the MMAs for both, so W crosses
//       L2->SM once per pair.  Warp-specialised:
//         warp 0      TMA producer: cp.async.bulk.tensor 2-D loads of a 128x64 X
//                     tile and a BNx64 W tile (128-byte swizzle) into a shared-
//                     memory ring (4..8 stages, sized per plan) guarded by
//                     full/empty mbarriers;
//         warp 1      TMEM allocator + MMA issuer: one elected lane issues
//                     tcgen05.mma.cta_group::1.kind::f16 (M=128, N=BN, K=16) four
//                     times per stage into a TMEM accumulator, tcgen05.commit
//                     releases the stage / publishes the accumulator;
//         warp 2      device-side tile scheduler: one atomicAdd per chunk of up
//                     to 4 tiles (one 128-byte line of the plan's tile table),
//                     copies each tile's 32-byte entry and its bias slice into a
//                     4-deep shared-memory queue, prefetches the member's tensor
//                     maps; the last CTA to finish re-arms the counter;
//         warps 3..10 epilogue, two warps per TMEM lane quadrant taking alternate
//                     64-column chunks: tcgen05.ld (32 lanes x 32 columns), + bias
//                     (from the queue slot: no global load in the epilogue),
//                     activation (ReLU folded into cvt.rn.relu.bf16x2), RNE to
//                     bf16, swizzled st.shared, TMA store (cp.async.bulk.tensor,
//                     64x32 boxes) into the member's output or its slot of the
//                     concatenated output.
//       TMEM holds two accumulator stages (2 x 256 columns) so the epilogue of
//       tile t overlaps the MMAs of tile t+1.  Tiles of one X row-panel are
//       adjacent in the schedule so its re-reads hit L2.  Deterministic: the
//       scheduler only decides WHICH CTA computes a tile, never how.
//   grouped_gemm_f32_kernel    plain fp32 FFMA (no TF32) 32x32 tiles for fp32
//       groups (configs[0]); same tile scheduler, accurate tanhf/expf epilogue.
#include <algorithm>
#include <map>
#include <set>
#include <tuple>
#include <cstdlib>

#include "sm100_ptx.h"

namespace optb {

// =========================================================== fp32 SIMT path ==
struct F32Member {
  const float* x; const float* w; const float* bias; float* y;
  int64_t ldx, ldw, ldy;
  int32_t M, N, K, act;
  int32_t nbn;        // n-blocks per m-block
  int32_t pad;
};

constexpr int kF32Tile = 32, kF32BK = 32, kF32Threads = 256;

__device__ __forceinline__ int find_member(const int32_t* __restrict__ starts, int n, int tile) {
  int lo = 0, hi = n;   // starts[lo] <= tile < starts[hi]
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(starts + mid) <= tile) lo = mid; else hi = mid;
  }
  return lo;
}

// fp32 groups are tiny and latency-bound (configs[0]: 8.5e5 flop): 32x32 output tiles so that the group spreads
// over more SMs, a 32-deep K slice per step, and the NEXT slice's global loads issued before the current slice is
// multiplied, so only the first load latency is exposed.  Thread t owns outputs (ty + 8i, tx) for i < 4.
__global__ void __launch_bounds__(kF32Threads)
grouped_gemm_f32_kernel(const F32Member* __restrict__ members, const int32_t* __restrict__ starts, int n_members) {
  __shared__ float As[kF32BK][kF32Tile + 1];
  __shared__ float Bs[kF32BK][kF32Tile + 1];
  const int tile = blockIdx.x;
  const int mi = find_member(starts, n_members, tile);
  const F32Member m = members[mi];
  const int local = tile - __ldg(starts + mi);
  const int m0 = (local / m.nbn) * kF32Tile, n0 = (local % m.nbn) * kF32Tile;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  // loader mapping: element (row lr + 8j, k lk) of the A and B slices, j < 4
  const int lk = threadIdx.x & 31, lr = threadIdx.x >> 5;
  float ra[4], rb[4];
  auto fetch = [&](int k0) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int r = lr + 8 * j;
      ra[j] = (m0 + r < m.M && k0 + lk < m.K) ? __ldg(m.x + (int64_t)(m0 + r) * m.ldx + k0 + lk) : 0.f;
      rb[j] = (n0 + r < m.N && k0 + lk < m.K) ? __ldg(m.w + (int64_t)(n0 + r) * m.ldw + k0 + lk) : 0.f;
    }
  };
  float acc[4] = {0.f, 0.f, 0.f, 0.f};
  fetch(0);
  for (int k0 = 0; k0 < m.K; k0 += kF32BK) {
#pragma unroll
    for (int j = 0; j < 4; ++j) { As[lk][lr + 8 * j] = ra[j]; Bs[lk][lr + 8 * j] = rb[j]; }
    __syncthreads();
    if (k0 + kF32BK < m.K) fetch(k0 + kF32BK);        // in flight while this slice is multiplied
#pragma unroll
    for (int k = 0; k < kF32BK; ++k) {
      const float b = Bs[k][tx];
#pragma unroll
      for (int i = 0; i < 4; ++i) acc[i] = fmaf(As[k][ty + 8 * i], b, acc[i]);
    }
    __syncthreads();
  }
  const int c = n0 + tx;
  if (c < m.N) {
    const float bias = m.bias ? __ldg(m.bias + c) : 0.f;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int r = m0 + ty + 8 * i;
      if (r < m.M) m.y[(int64_t)r * m.ldy + c] = act_f32<false>(acc[i] + bias, m.act);
    }
  }
}

cudaError_t launch_linear_f32(const opt_plan* p, cudaStream_t s) {
  const char* base = static_cast<const char*>(p->dev_tables);
  grouped_gemm_f32_kernel<<<p->grid, p->block, 0, s>>>(reinterpret_cast<const F32Member*>(base + p->off0),
                                                      reinterpret_cast<const int32_t*>(base + p->off1), p->n_members);
  return cudaGetLastError();
}

// ===================================================== bf16 tcgen05 path =====
constexpr int kBM = 128;           // tile rows (UMMA M, cta_group::1)
constexpr int kBK = 64;            // K per stage = one 128-byte swizzle row of bf16
constexpr int kMaxBN = 256;        // widest tile (UMMA N)
constexpr int kMaxStages = 8;      // smem ring depth is chosen per plan (stage = A tile + widest W tile of the group)
constexpr int kAccStages = 2;
constexpr int kTmemCols = 512;     // 2 accumulator stages x 256 fp32 columns
constexpr int kEpiWarps = 8;       // two per TMEM lane quadrant, alternating 64-column chunks
constexpr int kFirstEpiWarp = 3;   // warp 0 TMA, warp 1 MMA, warp 2 tile scheduler, warps 3..10 epilogue
constexpr int kGemmThreads = 32 * (kFirstEpiWarp + kEpiWarps);
constexpr int kABytes = kBM * kBK * 2;          // 16 KB
constexpr int kEpiBufBytes = 32 * 128;          // one warp's 32 rows x 64 bf16 staging tile
constexpr int kQDepth = 4;                      // tile queue: scheduler warp -> TMA / MMA / epilogue warps
constexpr int kQBiasBytes = kMaxBN * 2;         // the tile's bias slice, bf16
constexpr int kQSlotBytes = kQBiasBytes + 32;   // + the tile's 32-byte TileEntry
constexpr int kTilesPerChunk = 4;               // tiles fetched per atomic (one 128-byte table line)
constexpr int kSmemMax = 227 * 1024;
constexpr uint32_t kTransX = 1u << 28, kTransW = 1u << 29;   // TileEntry::misc flags: operand stored transposed
constexpr int kSmemFixed = kEpiWarps * kEpiBufBytes + kQDepth * kQSlotBytes + 256;   // staging + queue + barriers

struct alignas(128) GemmMember {
  CUtensorMap tmA;       // X [M,K]   box {64, 128}   load
  CUtensorMap tmB;       // W [N,K]   box {64, BN}    load
  CUtensorMap tmY;       // Y [M,N]   box {64, 32}    store
  CUtensorMap tmB2;      // W [N,K]   box {64, BN/2}  load (CTA-pair kernel: each CTA holds half of the W tile)
};
static_assert(sizeof(GemmMember) == 512, "GemmMember must keep tensor maps 128-byte aligned");

// One output tile, everything the three warp roles need (built by the planner, copied into shared
// memory by the scheduler warp).  member < 0: padding entry of a chunk (skipped).
struct alignas(16) TileEntry {
  int32_t member, m0, n0;
  uint32_t idesc;        // tcgen05 instruction descriptor (M=128, N=bn, bf16 x bf16 -> fp32)
  uint32_t bn_nkb;       // tile width | K blocks << 16
  uint32_t misc;         // K=16 steps in the last K block | act << 8 | valid columns (min(bn, N-n0)) << 16
  const void* bias;      // bias + n0 (bf16) or NULL
};
static_assert(sizeof(TileEntry) == 32, "TileEntry is two 16-byte vectors");

// Kernel-wide shared-memory map (dynamic, 1024-byte aligned base):
//   [0, nstages*stage_bytes)   operand ring: per stage a 128x64 X tile then the CTA's W tile (128B swizzle)
//   + 8 x 4 KB                 epilogue staging tiles (one per epilogue warp)
//   + kQDepth x 544 B          tile queue slots: 512 B bias slice (bf16) + 32 B TileEntry
//   + 256 B                    mbarriers: full[8] empty[8] tfull[2] tempty[2] qfull[4] qempty[4], TMEM base
//
// NCTA = 1: one CTA per tile (128 x BN).  NCTA = 2: a CTA PAIR (cluster of 2, cta_group::2) per 256 x BN tile:
// CTA r holds rows [128r, 128r+128) of X and rows [r*BN/2, (r+1)*BN/2) of the W tile, the leader (rank 0) issues
// the MMAs for both and runs the one scheduler of the pair, each CTA drains its own 128 accumulator rows.  W
// crosses L2->SM once per pair instead of once per CTA (configs[2] is bound by that traffic).
template <int NCTA>
__global__ void __launch_bounds__(kGemmThreads, 1)
grouped_gemm_sm100_kernel(const GemmMember* __restrict__ members, const uint4* __restrict__ chunks, int n_chunks,
                          int* __restrict__ counters, int nstages, int stage_bytes) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t sbase = smem_u32(smem);
  if ((sbase & 1023u) != 0) __trap();            // 128-byte-swizzle tiles need 1024-byte alignment
  const uint32_t epi_base = sbase + (uint32_t)(nstages * stage_bytes);
  const uint32_t q_base = epi_base + kEpiWarps * kEpiBufBytes;
  const uint32_t bar_base = q_base + kQDepth * kQSlotBytes;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (kMaxStages + s); };
  auto tfull_bar = [&](int s) { return bar_base + 8u * (2 * kMaxStages + s); };
  auto tempty_bar = [&](int s) { return bar_base + 8u * (2 * kMaxStages + kAccStages + s); };
  auto qfull_bar = [&](int s) { return bar_base + 8u * (2 * kMaxStages + 2 * kAccStages + s); };
  auto qempty_bar = [&](int s) { return bar_base + 8u * (2 * kMaxStages + 2 * kAccStages + kQDepth + s); };
  auto q_slot = [&](int s) { return q_base + (uint32_t)s * kQSlotBytes; };
  const uint32_t tmem_ptr_addr = bar_base + 8u * (2 * kMaxStages + 2 * kAccStages + 2 * kQDepth);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = NCTA == 2 ? cluster_ctarank() : 0u;     // 0 = leader
  // barriers that live in the LEADER (the peer arrives on them remotely): tempty, qempty
  auto leader = [&](uint32_t bar) { return NCTA == 2 ? mapa(bar, 0) : bar; };
  auto arrive_leader = [&](uint32_t bar) { if (NCTA == 2) mbar_arrive_cluster(mapa(bar, 0)); else mbar_arrive(bar); };
  auto wait_q = [&](uint32_t bar, uint32_t parity) { mbar_wait(bar, parity); };

  if (warp == 0 && lane == 0) {
    for (int s = 0; s < nstages; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int s = 0; s < kAccStages; ++s) { mbar_init(tfull_bar(s), 1); mbar_init(tempty_bar(s), NCTA * kEpiWarps); }
    // queue consumers: TMA + epilogue warps of every CTA of the pair, MMA issuer of the leader
    for (int s = 0; s < kQDepth; ++s) { mbar_init(qfull_bar(s), 1); mbar_init(qempty_bar(s), NCTA * (1 + kEpiWarps) + 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async_smem();
  }
  if (warp == 1) {
    if (NCTA == 2) {
      asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;"
                   ::"r"(tmem_ptr_addr), "n"(kTmemCols) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    } else {
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                   ::"r"(tmem_ptr_addr), "n"(kTmemCols) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
  }
  tc_fence_before();
  if (NCTA == 2) cluster_sync_all(); else __syncthreads();      // the peer's barriers are initialised too
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_addr) : "memory");

  if (warp == 2) {
    // ----------------------------------------------------- tile scheduler ----
    // Dynamic: one atomic per CHUNK of up to 4 tiles (one 128-byte table line); the next chunk id is
    // fetched while this chunk is published.  Per tile: entry + bias slice -> queue slot -> qfull.
    // CTA pair: the leader's scheduler serves both CTAs (remote shared-memory stores + remote arrive).
    if (rank == 0) {
      const int n_sched = NCTA == 2 ? (int)num_clusters_x() : (int)gridDim.x;
      int qs = 0; uint32_t qph = 0;
      int c = NCTA == 2 ? (int)cluster_id_x() : (int)blockIdx.x;
      // queue slot `qs` of both CTAs: local st.shared + arrive; peer: st.async pieces counted on ITS qfull
      auto publish = [&](int qs_, uint32_t off, uint4 v) {
        sts128(q_slot(qs_) + off, v);
        if (NCTA == 2) st_async128(mapa(q_slot(qs_) + off, 1), v, mapa(qfull_bar(qs_), 1));
      };
      auto signal_full = [&](int qs_, uint32_t peer_bytes) {
        mbar_arrive(qfull_bar(qs_));
        if (NCTA == 2) mbar_expect_tx_cluster(mapa(qfull_bar(qs_), 1), peer_bytes);
      };
      while (c < n_chunks) {
        int nextc = 0;
        if (lane == 0) nextc = atomicAdd(counters, 1) + n_sched;
        uint4 e = make_uint4(0xFFFFFFFFu, 0, 0, 0);
        if (lane < 2 * kTilesPerChunk) e = __ldg(chunks + (size_t)c * (2 * kTilesPerChunk) + lane);   // lane 2g, 2g+1: tile g
        uint4 bias_v[kTilesPerChunk];
        int member[kTilesPerChunk];
#pragma unroll
        for (int g = 0; g < kTilesPerChunk; ++g) {
          member[g] = (int)__shfl_sync(0xffffffffu, e.x, 2 * g);
          const uint32_t misc = __shfl_sync(0xffffffffu, e.y, 2 * g + 1);
          const uint32_t blo = __shfl_sync(0xffffffffu, e.z, 2 * g + 1), bhi = __shfl_sync(0xffffffffu, e.w, 2 * g + 1);
          const uint4* bp = reinterpret_cast<const uint4*>(((uint64_t)bhi << 32) | blo);
          bias_v[g] = make_uint4(0, 0, 0, 0);
          if (member[g] >= 0) {
            const int nvalid = (int)((misc >> 16) & 0x1FFu);
            if (bp != nullptr && 8 * lane + 8 <= nvalid) {
              bias_v[g] = __ldg(bp + lane);
            } else if (bp != nullptr && 8 * lane < nvalid) {       // ragged N: the last piece element by element
              const unsigned short* be = reinterpret_cast<const unsigned short*>(bp + lane);
              uint32_t w[4] = {0, 0, 0, 0};
              for (int t = 0; t < nvalid - 8 * lane; ++t) w[t >> 1] |= (uint32_t)__ldg(be + t) << (16 * (t & 1));
              bias_v[g] = make_uint4(w[0], w[1], w[2], w[3]);
            }
            if (lane < 4)   // warm the descriptor cache for the member's tensor maps
              asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<const char*>(members + member[g]) + 128 * lane) : "memory");
          }
        }
#pragma unroll
        for (int g = 0; g < kTilesPerChunk; ++g) {
          if (member[g] < 0) continue;       // warp-uniform
          wait_q(qempty_bar(qs), qph ^ 1);
          publish(qs, 16 * lane, bias_v[g]);
          if ((lane >> 1) == g) publish(qs, kQBiasBytes + 16 * (lane & 1), e);
          __syncwarp();
          if (lane == 0) signal_full(qs, kQSlotBytes);
          if (++qs == kQDepth) { qs = 0; qph ^= 1; }
        }
        c = __shfl_sync(0xffffffffu, nextc, 0);
      }
      // end marker, then the last scheduler to get here re-arms the counters for the next launch of this plan
      wait_q(qempty_bar(qs), qph ^ 1);
      if (lane == 0) {
        publish(qs, kQBiasBytes, make_uint4(0xFFFFFFFFu, 0, 0, 0));
        signal_full(qs, 16);
        __threadfence();
        if (atomicAdd(counters + 1, 1) == n_sched - 1) {
          counters[0] = 0;
          counters[1] = 0;
          __threadfence();
        }
      }
    }
  } else if (warp == 0) {
    // ------------------------------------------------------- TMA producer ----
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      int qs = 0; uint32_t qph = 0;
      for (;;) {
        wait_q(qfull_bar(qs), qph);
        const uint4 e0 = lds128(q_slot(qs) + kQBiasBytes);
        const uint4 e1 = lds128(q_slot(qs) + kQBiasBytes + 16);
        arrive_leader(qempty_bar(qs));
        if (++qs == kQDepth) { qs = 0; qph ^= 1; }
        if ((int)e0.x < 0) break;
        const GemmMember* m = members + (int)e0.x;
        const int bn = (int)(e1.x & 0xFFFFu), nkb = (int)(e1.x >> 16);
        const int m0 = (int)e0.y + (int)rank * kBM;              // this CTA's 128 rows of the (pair) tile
        const int n0 = (int)e0.z + (int)rank * (bn / NCTA);      // this CTA's rows of the W tile
        const uint32_t b_bytes = (uint32_t)(bn / NCTA) * (kBK * 2);
        const CUtensorMap* tmB = NCTA == 2 ? &m->tmB2 : &m->tmB;
        for (int kb = 0; kb < nkb; ++kb) {
          mbar_wait(empty_bar(stage), phase ^ 1);
          const uint32_t sa = sbase + stage * stage_bytes;
          if (NCTA == 2) {
            // the leader's barrier counts the bytes of both CTAs
            if (rank == 0) mbar_expect_tx(full_bar(stage), 2 * (kABytes + b_bytes));
            const uint32_t lb = mapa(full_bar(stage), 0);
            tma_load_2d_pair(sa, &m->tmA, lb, kb * kBK, m0);
            tma_load_2d_pair(sa + kABytes, tmB, lb, kb * kBK, n0);
          } else {
            mbar_expect_tx(full_bar(stage), kABytes + b_bytes);
            if (e1.y & kTransX) {                    // stored [K, M]: two 64x64 boxes (contraction rows, M contiguous)
              tma_load_2d(sa, &m->tmA, full_bar(stage), m0, kb * kBK);
              tma_load_2d(sa + 8192, &m->tmA, full_bar(stage), m0 + 64, kb * kBK);
            } else {
              tma_load_2d(sa, &m->tmA, full_bar(stage), kb * kBK, m0);
            }
            if (e1.y & kTransW) {                    // stored [K, N]: BN/64 boxes
              for (int j = 0; j < bn / 64; ++j) tma_load_2d(sa + kABytes + j * 8192, tmB, full_bar(stage), n0 + 64 * j, kb * kBK);
            } else {
              tma_load_2d(sa + kABytes, tmB, full_bar(stage), kb * kBK, n0);
            }
          }
          if (++stage == nstages) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------- MMA issuer (leader only) ----
    if (lane == 0 && rank == 0) {
      int stage = 0; uint32_t phase = 0;
      int as = 0; uint32_t aphase = 0;
      int qs = 0; uint32_t qph = 0;
      for (;;) {
        wait_q(qfull_bar(qs), qph);
        const uint4 e0 = lds128(q_slot(qs) + kQBiasBytes);
        const uint4 e1 = lds128(q_slot(qs) + kQBiasBytes + 16);
        arrive_leader(qempty_bar(qs));
        if (++qs == kQDepth) { qs = 0; qph ^= 1; }
        if ((int)e0.x < 0) break;
        const uint32_t idesc = e0.w;
        const int nkb = (int)(e1.x >> 16), klast = (int)(e1.y & 0xFFu);
        wait_q(tempty_bar(as), aphase ^ 1);         // the epilogues (of both CTAs) have drained this accumulator stage
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + as * kMaxBN;
        for (int kb = 0; kb < nkb; ++kb) {
          mbar_wait(full_bar(stage), phase);
          tc_fence_after();
          const uint32_t sa = sbase + stage * stage_bytes;
          const bool tx = NCTA == 1 && (e1.y & kTransX), tw = NCTA == 1 && (e1.y & kTransW);
          const uint64_t adesc = tx ? umma_desc_sw128_mn(sa) : umma_desc_sw128(sa);
          const uint64_t bdesc = tw ? umma_desc_sw128_mn(sa + kABytes) : umma_desc_sw128(sa + kABytes);
          // per K=16 step: K-major +32 bytes inside the swizzle row (+2 encoded); MN-major +2 groups of 8 rows (+128)
          const uint64_t astep = tx ? 128 : 2, bstep = tw ? 128 : 2;
          const int ksteps = kb + 1 < nkb ? kBK / 16 : klast;
          for (int k = 0; k < ksteps; ++k) {
            if (NCTA == 2) tc_mma_bf16_pair(d_tmem, adesc + 2 * k, bdesc + 2 * k, idesc, (kb | k) != 0);
            else tc_mma_bf16(d_tmem, adesc + astep * k, bdesc + bstep * k, idesc, (kb | k) != 0);
          }
          // frees the smem stage (in both CTAs) when these MMAs retire
          if (NCTA == 2) tc_commit_pair(empty_bar(stage)); else tc_commit(empty_bar(stage));
          if (++stage == nstages) { stage = 0; phase ^= 1; }
        }
        if (NCTA == 2) tc_commit_pair(tfull_bar(as)); else tc_commit(tfull_bar(as));   // accumulator complete
        if (++as == kAccStages) { as = 0; aphase ^= 1; }
      }
    }
  } else {
    // ----------------------------------------------------------- epilogue ----
    const int ew = warp - kFirstEpiWarp;
    const int quad = warp & 3;               // TMEM lane quadrant this warp may read
    const int half = ew >> 2;                // 0: even 64-column chunks, 1: odd ones
    const uint32_t sbuf = epi_base + (uint32_t)ew * kEpiBufBytes;
    const uint32_t srow = sbuf + lane * 128;
    int as = 0; uint32_t aphase = 0;
    int qs = 0; uint32_t qph = 0;
    for (;;) {
      wait_q(qfull_bar(qs), qph);
      const uint32_t slot = q_slot(qs);
      const uint4 e0 = lds128(slot + kQBiasBytes);
      const uint4 e1 = lds128(slot + kQBiasBytes + 16);
      if ((int)e0.x < 0) break;
      const GemmMember* m = members + (int)e0.x;
      const int m0 = (int)e0.y + (int)rank * kBM, n0 = (int)e0.z;
      const int bn = (int)(e1.x & 0xFFFFu), act = (int)((e1.y >> 8) & 0xFFu);
      mbar_wait(tfull_bar(as), aphase);
      tc_fence_after();
      const uint32_t t_row = tmem_base + ((uint32_t)(quad * 32) << 16) + as * kMaxBN;
      const int nchunks = (bn + 63) >> 6;
      bool released = false;
      for (int c = half; c < nchunks; c += 2) {
        uint32_t v[64];
        tc_ld_32x32(t_row + c * 64, *reinterpret_cast<uint32_t(*)[32]>(&v[0]));
        tc_ld_32x32(t_row + c * 64 + 32, *reinterpret_cast<uint32_t(*)[32]>(&v[32]));
        tc_wait_ld();
        if (c + 2 >= nchunks) {              // this warp's part of the accumulator is in registers
          tc_fence_before();
          __syncwarp();
          if (lane == 0) arrive_leader(tempty_bar(as));
          released = true;
        }
        uint32_t p[32];
        const uint32_t bias_addr = slot + (uint32_t)c * 128;
        switch (act) {
          case OPT_ACT_RELU: epi_math<OPT_ACT_RELU>(v, bias_addr, p); break;
          case OPT_ACT_NONE: epi_math<OPT_ACT_NONE>(v, bias_addr, p); break;
          case OPT_ACT_TANH: epi_math<OPT_ACT_TANH>(v, bias_addr, p); break;
          default:           epi_math<OPT_ACT_SIGMOID>(v, bias_addr, p); break;
        }
        // staging buffer free? (the previous TMA store of this warp has read it) -- checked after the math so
        // that the store engine's read of the previous chunk overlaps it
        if (lane == 0) tma_store_wait_read<0>();
        __syncwarp();
#pragma unroll
        for (int j = 0; j < 8; ++j)            // 16-byte pieces at their 128B-swizzled position
          sts128(srow + ((j ^ (lane & 7)) << 4), make_uint4(p[4 * j], p[4 * j + 1], p[4 * j + 2], p[4 * j + 3]));
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
          tma_store_2d(&m->tmY, sbuf, n0 + c * 64, m0 + quad * 32);
          tma_store_commit();
        }
      }
      if (!released) {                       // no chunk for this warp in a narrow tile: still hand the stage back
        tc_fence_before();
        __syncwarp();
        if (lane == 0) arrive_leader(tempty_bar(as));
      }
      __syncwarp();                          // every lane has read the slot's bias
      if (lane == 0) arrive_leader(qempty_bar(qs));
      if (++qs == kQDepth) { qs = 0; qph ^= 1; }
      if (++as == kAccStages) { as = 0; aphase ^= 1; }
    }
    if (lane == 0) tma_store_wait_all();
  }

  tc_fence_before();
  if (NCTA == 2) cluster_sync_all(); else __syncthreads();      // the peer may still be reading this CTA's W half
  if (warp == 1) {
    tc_fence_after();
    if (NCTA == 2)
      asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols) : "memory");
    else
      asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols) : "memory");
  }
}

cudaError_t launch_linear_bf16(const opt_plan* p, cudaStream_t s) {
  char* base = static_cast<char*>(p->dev_tables);
  auto* members = reinterpret_cast<const GemmMember*>(base + p->off0);
  auto* chunks = reinterpret_cast<const uint4*>(base + p->off1);
  int* counters = reinterpret_cast<int*>(base + p->off2);
  if (p->ncta == 2) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = p->grid; cfg.blockDim = p->block; cfg.dynamicSmemBytes = p->smem; cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, grouped_gemm_sm100_kernel<2>, members, chunks, (int)p->n_chunks, counters,
                              (int)p->nstages, (int)p->stage_bytes);
  }
  grouped_gemm_sm100_kernel<1><<<p->grid, p->block, p->smem, s>>>(members, chunks, p->n_chunks, counters, p->nstages,
                                                                 p->stage_bytes);
  return cudaGetLastError();
}

static int choose_bn(int N) {
  if (N <= kMaxBN) return (N + 15) / 16 * 16;          // one n-block, UMMA N multiple of 16
  // several n-blocks: multiples of 64 only (epilogue chunks must not spill into the next block)
  int best = 256, best_pad = INT32_MAX;
  for (int bn : {256, 192, 128}) {
    const int pad = (N + bn - 1) / bn * bn - N;
    if (pad < best_pad) { best_pad = pad; best = bn; }
  }
  return best;
}

}  // namespace optb

using namespace optb;

extern "C" opt_status opt_linear_plan_create(const opt_linear_member* members, int32_t n, opt_dtype io, int device,
                                             opt_plan** plan) {
  return opt_linear_plan_create_ex(members, n, io, device, nullptr, plan);
}

extern "C" opt_status opt_linear_plan_create_ex(const opt_linear_member* members, int32_t n, opt_dtype io, int device,
                                                const opt_linear_options* options, opt_plan** plan) {
  if (plan) *plan = nullptr;
  if (!plan || !members) return fail(OPT_ERR_INVALID_ARG, "opt_linear_plan_create: NULL argument");
  opt_linear_options opts;
  memset(&opts, 0, sizeof opts);
  if (options) opts = *options;
  if (opts.cta_pair < 0 || opts.cta_pair > 2) return fail(OPT_ERR_INVALID_ARG, "options.cta_pair = %d outside {0, 1, 2}", opts.cta_pair);
  for (int32_t r : opts.reserved) if (r != 0) return fail(OPT_ERR_INVALID_ARG, "options.reserved must be zero");
  if (n < 1 || n > 65535) return fail(OPT_ERR_INVALID_ARG, "n = %d outside [1, 65535]", n);
  if (io != OPT_F32 && io != OPT_BF16) return fail(OPT_ERR_INVALID_ARG, "bad io dtype %d", (int)io);
  const int esz = elem_size(io), V = vec_elems(io);
  std::vector<Region> regions;
  int64_t flops = 0, bytes = 0;
  std::set<std::tuple<const void*, int64_t, int32_t, int32_t>> seen_x;
  // huge-M / tiny-K-and-N groups (decompose_mm_pass) stream through the SIMT row kernel (linear_skinny.cu)
  bool skinny = io == OPT_BF16 && !opts.no_skinny;
  for (int32_t i = 0; skinny && i < n; ++i) skinny = skinny_linear_member(members[i]);
  for (int32_t i = 0; i < n; ++i) {
    const opt_linear_member& m = members[i];
    if (!m.x || !m.w || !m.y) return fail(OPT_ERR_INVALID_ARG, "member %d: NULL pointer", i);
    if (m.M < 1 || m.N < 1 || m.K < 1) return fail(OPT_ERR_INVALID_ARG, "member %d: M=%d N=%d K=%d must be >= 1", i, m.M, m.N, m.K);
    if (m.act < OPT_ACT_NONE || m.act > OPT_ACT_SIGMOID) return fail(OPT_ERR_INVALID_ARG, "member %d: bad activation %d", i, m.act);
    if (m.layout & ~(OPT_LAYOUT_X_TRANSPOSED | OPT_LAYOUT_W_TRANSPOSED)) return fail(OPT_ERR_INVALID_ARG, "member %d: bad layout flags %d", i, m.layout);
    const bool tx = m.layout & OPT_LAYOUT_X_TRANSPOSED, tw = m.layout & OPT_LAYOUT_W_TRANSPOSED;
    if ((tx || tw) && io != OPT_BF16) return fail(OPT_ERR_UNSUPPORTED, "member %d: transposed operands are implemented for bf16 groups only", i);
    // stored shapes: x [M,K] or (transposed) [K,M]; w [N,K] or (transposed) [K,N]
    const int32_t x_rows = tx ? m.K : m.M, x_cols = tx ? m.M : m.K, w_rows = tw ? m.K : m.N, w_cols = tw ? m.N : m.K;
    if ((x_rows > 1 && m.ldx < x_cols) || (m.M > 1 && m.ldy < m.N) || (w_rows > 1 && m.ldw < w_cols))
      return fail(OPT_ERR_INVALID_ARG, "member %d: row stride smaller than the row", i);
    if (!aligned16(m.x) || !aligned16(m.w) || !aligned16(m.y) || !aligned16(m.bias))
      return fail(OPT_ERR_ALIGNMENT, "member %d: pointers must be 16-byte aligned", i);
    // bf16: K and N need NOT be multiples of 8 -- TMA zero-fills the K / N tails of the operand tiles and clips the
    // store, which is what pad_aten_mm_pass achieves by padding; only bases and row strides must be
    // 16-byte aligned.  fp32 (SIMT path): multiples of 4.
    if (io == OPT_F32 && (m.K % V || m.N % V))
      return fail(OPT_ERR_ALIGNMENT, "member %d: K=%d and N=%d must be multiples of %d", i, m.K, m.N, V);
    if (skinny) {      // rows are read and written as 4-byte words
      if (m.ldx % 2 || m.ldw % 2 || m.ldy % 2)
        return fail(OPT_ERR_ALIGNMENT, "member %d: row strides must be even (4-byte words)", i);
    } else if (m.ldx % V || m.ldw % V || m.ldy % V) {
      return fail(OPT_ERR_ALIGNMENT, "member %d: row strides must be multiples of %d elements", i, V);
    }
    regions.push_back({(uintptr_t)m.x, m.ldx * esz, (int64_t)x_cols * esz, x_rows, false, i});
    regions.push_back({(uintptr_t)m.w, m.ldw * esz, (int64_t)w_cols * esz, w_rows, false, i});
    if (m.bias) regions.push_back({(uintptr_t)m.bias, 0, (int64_t)m.N * esz, 1, false, i});
    regions.push_back({(uintptr_t)m.y, m.ldy * esz, (int64_t)m.N * esz, m.M, true, i});
    flops += 2ll * m.M * m.N * m.K;
    // an input shared by several members (batch_linear_lhs) is read once
    const bool first_use_of_x = seen_x.insert(std::make_tuple(m.x, m.ldx, m.M, tx ? -m.K : m.K)).second;
    bytes += ((first_use_of_x ? (int64_t)m.M * m.K : 0) + (int64_t)m.N * m.K + (m.bias ? m.N : 0) + (int64_t)m.M * m.N) * esz;
  }
  if (opt_status st = check_independent(regions, /*allow_inplace_self=*/false)) return st;

  int num_sms = 0;
  DeviceGuard device_guard;      // the caller's current device is restored on return
  if (opt_status st = open_device(device, &num_sms)) return st;
  auto align_up = [](size_t x) { return (x + 255) & ~size_t(255); };
  opt_plan* p = new opt_plan();
  p->device = device; p->io = io; p->n_members = n; p->flops = flops; p->bytes = bytes;
  std::vector<int32_t> starts(n + 1);
  int64_t tiles = 0;

  if (skinny) {
    if (opt_status st = plan_skinny_linear(members, n, p)) { delete p; return st; }
    *plan = p;
    return OPT_OK;
  }

  if (io == OPT_F32) {
    std::vector<F32Member> tab(n);
    for (int32_t i = 0; i < n; ++i) {
      const opt_linear_member& m = members[i];
      F32Member& t = tab[i];
      t.x = (const float*)m.x; t.w = (const float*)m.w; t.bias = (const float*)m.bias; t.y = (float*)m.y;
      t.ldx = m.ldx; t.ldw = m.ldw; t.ldy = m.ldy; t.M = m.M; t.N = m.N; t.K = m.K; t.act = m.act;
      t.nbn = (m.N + kF32Tile - 1) / kF32Tile; t.pad = 0;
      starts[i] = (int32_t)tiles;
      tiles += (int64_t)((m.M + kF32Tile - 1) / kF32Tile) * t.nbn;
      if (tiles > INT32_MAX) { delete p; return fail(OPT_ERR_UNSUPPORTED, "too many tiles"); }
    }
    starts[n] = (int32_t)tiles;
    p->kind = kPlanLinearF32;
    p->off0 = 0; p->off1 = align_up(tab.size() * sizeof(F32Member));
    const size_t total = p->off1 + align_up(starts.size() * sizeof(int32_t));
    std::vector<char> blob(total, 0);
    memcpy(blob.data(), tab.data(), tab.size() * sizeof(F32Member));
    memcpy(blob.data() + p->off1, starts.data(), starts.size() * sizeof(int32_t));
    if (opt_status st = upload_tables(p, blob.data(), total)) { delete p; return st; }
    p->grid = dim3((unsigned)tiles); p->block = dim3(kF32Threads); p->smem = 0;
    p->total_tiles = (int32_t)tiles;
    *plan = p;
    return OPT_OK;
  }

  EncodeTiledFn enc = nullptr;
  if (opt_status st = get_encoder(&enc)) { delete p; return st; }
  std::vector<GemmMember> tab(n);
  memset(tab.data(), 0, tab.size() * sizeof(GemmMember));
  // CTA pair (256-row tiles, W shared by the pair) or single CTA (128-row tiles)
  int ncta = opts.cta_pair == 1 ? 1 : 2;
  for (int32_t i = 0; i < n; ++i)
    if (members[i].layout) {                   // MN-major (transposed) operand tiles are built per CTA: single-CTA kernel
      if (opts.cta_pair == 2) { delete p; return fail(OPT_ERR_UNSUPPORTED, "options.cta_pair = 2: member %d has a transposed operand (single-CTA tiles only)", i); }
      ncta = 1;
    }
  const int tile_m = kBM * ncta;
  struct MemberTiling { int bn, nbn, nkb, klast; uint32_t idesc, flags; };
  std::vector<MemberTiling> tiling(n);
  int max_bn = 16;
  for (int32_t i = 0; i < n; ++i) {
    const opt_linear_member& m = members[i];
    GemmMember& t = tab[i];
    const bool tx = m.layout & OPT_LAYOUT_X_TRANSPOSED, tw = m.layout & OPT_LAYOUT_W_TRANSPOSED;
    int bn = choose_bn(m.N);
    if (tw) bn = (bn + 63) / 64 * 64;          // MN-major W tiles are rows of 64x64 boxes
    opt_status st;
    // K-major operand: box {64 k, rows};  transposed operand (stored [K, out]): box {64 out, 64 k}
    st = tx ? encode_2d(enc, &t.tmA, m.x, m.K, m.M, m.ldx, 64, kBK, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, "X^T", i)
            : encode_2d(enc, &t.tmA, m.x, m.M, m.K, m.ldx, kBK, kBM, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, "X", i);
    if (!st) st = tw ? encode_2d(enc, &t.tmB, m.w, m.K, m.N, m.ldw, 64, kBK, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, "W^T", i)
                     : encode_2d(enc, &t.tmB, m.w, m.N, m.K, m.ldw, kBK, bn, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, "W", i);
    if (!st) st = encode_2d(enc, &t.tmY, m.y, m.M, m.N, m.ldy, 64, 32, CU_TENSOR_MAP_L2_PROMOTION_NONE, "Y", i);
    if (!st && !tw) st = encode_2d(enc, &t.tmB2, m.w, m.N, m.K, m.ldw, kBK, bn / 2, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, "W/2", i);
    if (st) {
      delete p;
      return st;
    }
    MemberTiling& tl = tiling[i];
    tl.bn = bn; tl.nbn = (m.N + bn - 1) / bn; tl.nkb = (m.K + kBK - 1) / kBK;
    tl.klast = (m.K - (tl.nkb - 1) * kBK + 15) / 16;
    // tcgen05 instruction descriptor, kind::f16: D fp32 (bits 4-5 = 1), A bf16 (bits 7-9 = 1), B bf16
    // (bits 10-12 = 1), A and B K-major (bits 15, 16 = 0), N>>3 at bits 17-22, M>>4 at bits 24-28.
    tl.idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)tx << 15) | ((uint32_t)tw << 16) | ((uint32_t)(bn >> 3) << 17) |
               ((uint32_t)(tile_m >> 4) << 24);
    tl.flags = (tx ? kTransX : 0u) | (tw ? kTransW : 0u);
    max_bn = std::max(max_bn, bn);
    const int nmb = (m.M + tile_m - 1) / tile_m;
    tiles += (int64_t)nmb * tl.nbn;
    if (tiles > INT32_MAX / 2) { delete p; return fail(OPT_ERR_UNSUPPORTED, "too many tiles"); }
  }
  // Schedule order: (LHS group,) member-major, m-block, n-block -- the n-blocks of one X row panel are adjacent, so the
  // CTAs that take them side by side fetch the panel from HBM once (re-reads hit L2), and a member's W stays
  // hot in L2 while its tiles are in flight.  (Interleaving tensor-bound with HBM-bound members was measured:
  // no gain on configs[2], the kernel is bound by L2->SM operand traffic there.)
  // batch_linear_lhs: members that share ONE input X (same pointer, stride, M, K) form an LHS group
  // whose schedule is m-block-major ACROSS its members -- all n-blocks of all members that read a given X row
  // panel are adjacent, so the panel is fetched from HBM once for the whole group (weights logically concatenated).
  std::vector<TileEntry> flat;
  flat.reserve((size_t)tiles);
  auto push_tiles = [&](int32_t i, int mb) {
    const opt_linear_member& m = members[i];
    const MemberTiling& tl = tiling[i];
    for (int nb = 0; nb < tl.nbn; ++nb) {
      TileEntry e;
      e.member = i; e.m0 = mb * tile_m; e.n0 = nb * tl.bn; e.idesc = tl.idesc;
      e.bn_nkb = (uint32_t)tl.bn | ((uint32_t)tl.nkb << 16);
      e.misc = (uint32_t)tl.klast | ((uint32_t)m.act << 8) | ((uint32_t)std::min(tl.bn, m.N - e.n0) << 16) | tl.flags;
      e.bias = m.bias ? static_cast<const char*>(m.bias) + (size_t)e.n0 * 2 : nullptr;
      flat.push_back(e);
    }
  };
  {
    std::map<std::tuple<const void*, int64_t, int32_t, int32_t>, std::vector<int32_t>> lhs;
    std::vector<std::tuple<const void*, int64_t, int32_t, int32_t>> first_seen;
    for (int32_t i = 0; i < n; ++i) {
      const auto key = std::make_tuple(members[i].x, members[i].ldx, members[i].M, members[i].K);
      if (lhs.find(key) == lhs.end()) first_seen.push_back(key);
      lhs[key].push_back(i);
    }
    const bool no_lhs = opts.no_lhs_order != 0;
    if (no_lhs) { first_seen.clear(); for (int32_t i = 0; i < n; ++i) { const int nmb = (members[i].M + tile_m - 1) / tile_m; for (int mb = 0; mb < nmb; ++mb) push_tiles(i, mb); } }
    for (const auto& key : first_seen) {
      const std::vector<int32_t>& grp = lhs[key];
      const int nmb = (std::get<2>(key) + tile_m - 1) / tile_m;
      for (int mb = 0; mb < nmb; ++mb)
        for (int32_t i : grp) push_tiles(i, mb);
    }
  }
  // Chunks of 4 tiles (one 128-byte line, one atomic); the last ~3 waves go one tile per chunk so that the
  // tail of the persistent loop is balanced at tile granularity.
  TileEntry pad_entry;
  memset(&pad_entry, 0, sizeof pad_entry);
  pad_entry.member = -1;
  const size_t tail_waves = 3;
  const int n_sched = num_sms / ncta;                         // persistent CTAs (or CTA pairs)
  const size_t tail = std::min(flat.size(), tail_waves * n_sched);
  const size_t body = flat.size() - tail;
  std::vector<TileEntry> chunked;
  // chunk c = tiles c, c+nC, c+2nC, c+3nC of the schedule order: CTAs that run side by side work on
  // neighbouring tiles (one X panel, fetched from HBM once), and one CTA's consecutive tiles come from
  // different members (an HBM-bound tile's epilogue overlaps a tensor-bound tile's MMAs)
  const size_t nC = (body + kTilesPerChunk - 1) / kTilesPerChunk;
  for (size_t c = 0; c < nC; ++c)
    for (int g = 0; g < kTilesPerChunk; ++g) {
      const size_t k = (size_t)g * nC + c;
      chunked.push_back(k < body ? flat[k] : pad_entry);
    }
  for (size_t k = body; k < flat.size(); ++k) {
    chunked.push_back(flat[k]);
    for (int g = 1; g < kTilesPerChunk; ++g) chunked.push_back(pad_entry);
  }
  const int64_t n_chunks = (int64_t)(chunked.size() / kTilesPerChunk);

  const int stage_bytes = kABytes + max_bn / ncta * kBK * 2;
  const int nstages = std::min(kMaxStages, (kSmemMax - kSmemFixed) / stage_bytes);
  const int smem_bytes = nstages * stage_bytes + kSmemFixed;
  p->kind = kPlanLinearBf16;
  p->off0 = 0;
  p->off1 = align_up(tab.size() * sizeof(GemmMember));
  p->off2 = p->off1 + align_up(chunked.size() * sizeof(TileEntry));
  const size_t total = p->off2 + 256;                         // two int32 scheduler counters, zero-initialised
  std::vector<char> blob(total, 0);
  memcpy(blob.data(), tab.data(), tab.size() * sizeof(GemmMember));
  memcpy(blob.data() + p->off1, chunked.data(), chunked.size() * sizeof(TileEntry));
  if (opt_status st = upload_tables(p, blob.data(), total)) { delete p; return st; }
  cudaError_t e = ncta == 2
      ? cudaFuncSetAttribute(grouped_gemm_sm100_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMax)
      : cudaFuncSetAttribute(grouped_gemm_sm100_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMax);
  if (e != cudaSuccess) {
    cudaFree(p->dev_tables); delete p;
    return fail(OPT_ERR_CUDA, "cudaFuncSetAttribute(max dynamic smem %d) failed: %s", kSmemMax, cudaGetErrorString(e));
  }
  p->grid = dim3((unsigned)(std::min<int64_t>(n_chunks, n_sched) * ncta)); p->block = dim3(kGemmThreads); p->smem = smem_bytes;
  p->ncta = ncta;
  p->total_tiles = (int32_t)tiles;
  p->n_chunks = (int32_t)n_chunks; p->nstages = nstages; p->stage_bytes = stage_bytes;
  *plan = p;
  return OPT_OK;
}
