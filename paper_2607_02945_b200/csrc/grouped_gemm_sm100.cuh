// grouped_gemm_sm100_kernel -- the bf16 grouped Linear (+bias +activation, optional FP8 copy of the output) of
// liboptimus_b200: N independent  Y_i = act_i(X_i W_i^T + b_i)  in ONE launch (batch_linear / batch_linear_post_grad /
// batch_linear_lhs with the epilogue fused: PAPER.md:292, :148 group fusion).  Included by linear.cu (planner + launch).
//
// Persistent, one CTA per SM; by default the CTAs work as PAIRS (cluster of 2, tcgen05 cta_group::2) on 256 x BN
// tiles -- each CTA stages its 128 rows of X and half of the W tile, the leader issues the MMAs for both, so W crosses
// L2->SM once per pair.  Warp-specialised:
//   warp 0      TMA producer: cp.async.bulk.tensor 2-D loads of a 128x64 X tile and this CTA's part of the BNx64 W
//               tile (128-byte swizzle) into a shared-memory ring (4..8 stages, sized per plan) guarded by full/empty
//               mbarriers.  The W tile of a COMPOSITE tile is assembled from 64-row (or 32-row) boxes of several members' W.
//   warp 1      TMEM allocator + MMA issuer (leader CTA only): one elected lane issues tcgen05.mma.kind::f16
//               (M=128 or 256 per pair, N=BN, K=16) four times per stage into a TMEM accumulator; tcgen05.commit
//               releases the stage / publishes the accumulator.
//   warp 2      device-side tile scheduler (one per pair): one atomicAdd per chunk of 4 tiles (four 128-byte lines of
//               the plan's tile table), the next chunk id fetched one ahead; per tile it copies the entry head, the four
//               64-column chunk descriptors and the bias slices into a 4-deep shared-memory queue of BOTH CTAs,
//               prefetches the member's tensor maps; the last scheduler to finish re-arms the counters.
//   warps 3..10 epilogue, two warps per TMEM lane quadrant taking alternate 64-column chunks: tcgen05.ld (32 lanes x
//               32 columns x2), + bias (from the queue slot: no global load in the epilogue), activation (ReLU folded
//               into cvt.rn.relu.bf16x2), RNE to bf16, swizzled st.shared, TMA store (64x32 boxes) into the chunk's
//               member output or its slot of a concatenated output; then, if the member wants it, the FP8 (E4M3) codes
//               of the ROUNDED bf16 values x scale8 through the same staging buffer and a second TMA store.
// TMEM holds two accumulator stages (2 x 256 columns) so the epilogue of tile t overlaps the MMAs of tile t+1.
// Deterministic: the scheduler only decides WHICH CTA computes a tile, never how (no split-K, no atomics on data).
#pragma once
#include "sm100_ptx.h"

namespace optb {

constexpr int kBM = 128;           // tile rows per CTA (UMMA M, cta_group::1; a pair covers 256)
constexpr int kBK = 64;            // K per stage = one 128-byte swizzle row of bf16
constexpr int kMaxBN = 256;        // widest tile (UMMA N)
constexpr int kMaxStages = 8;      // smem ring depth is chosen per plan (stage = A tile + widest W tile of the group)
constexpr int kAccStages = 2;
constexpr int kTmemCols = 512;     // 2 accumulator stages x 256 fp32 columns
constexpr int kEpiWarps = 8;       // two per TMEM lane quadrant, alternating 64-column chunks
constexpr int kFirstEpiWarp = 3;   // warp 0 TMA, warp 1 MMA, warp 2 tile scheduler, warps 3..10 epilogue
constexpr int kGemmThreads = 32 * (kFirstEpiWarp + kEpiWarps);
constexpr int kABytes = kBM * kBK * 2;          // 16 KB
constexpr int kEpiBufBytes = 32 * 128;          // one warp's 32 rows x 64 bf16 staging tile (reused for 32 x 64 fp8 codes)
constexpr int kQDepth = 4;                      // tile queue: scheduler warp -> TMA / MMA / epilogue warps
constexpr int kQBiasBytes = kMaxBN * 2;         // the tile's bias slices, bf16, chunk c at 128 c
constexpr int kQHeadOff = kQBiasBytes;          // 32-byte entry head
constexpr int kQDescOff = kQBiasBytes + 32;     // four 16-byte chunk descriptors
constexpr int kQSlotBytes = kQBiasBytes + 96;
constexpr int kTilesPerChunk = 4;               // tiles fetched per atomic
constexpr int kSmemMax = 227 * 1024;
constexpr int kSmemFixed = kEpiWarps * kEpiBufBytes + kQDepth * kQSlotBytes + 256;   // staging + queue + barriers
// TileEntry::misc
constexpr uint32_t kMiscComposite = 1u << 26;                // the W tile is assembled from boxes of several members' W
constexpr uint32_t kTransX = 1u << 28, kTransW = 1u << 29;   // operand stored transposed
// chunk descriptor flags
constexpr uint32_t kChunkHasY = 1u << 8, kChunkHasY8 = 1u << 9;

struct alignas(128) GemmMember {
  CUtensorMap tmA;       // X [M,K]   box {64, 128}   load
  CUtensorMap tmB;       // W [N,K]   box {64, BN}    load
  CUtensorMap tmY;       // Y [M,N]   box {64, 32}    store (bf16)
  CUtensorMap tmB2;      // W [N,K]   box {64, BN/2}  load (CTA-pair kernel: each CTA holds half of the W tile)
  CUtensorMap tmB64;     // W [N,K]   box {64, 64}    load (composite tiles: one 64-column chunk of the tile)
  CUtensorMap tmB32;     // W [N,K]   box {64, 32}    load (composite tiles with an odd chunk count, CTA pair: half a chunk)
  CUtensorMap tmY8;      // Y8 [M,N]  box {64, 32}    store (uint8, 64-byte swizzle)
};
static_assert(sizeof(GemmMember) == 896, "GemmMember must keep tensor maps 128-byte aligned");

// One 64-column chunk of an output tile: whose columns they are and what the epilogue does with them.
struct alignas(16) ChunkDesc {
  int32_t member;        // member that owns the chunk (its tmY / tmY8 / tmB64 / tmB32)
  int32_t n0;            // first output column of the chunk inside that member
  uint32_t act_flags;    // opt_act | kChunkHasY | kChunkHasY8
  float scale8;          // FP8 scale of that member
};

// One output tile, everything the warp roles need (built by the planner, one 128-byte line; the scheduler warp copies
// head + chunk descriptors + the bias slices into shared memory).  member < 0: padding entry of a chunk (skipped).
struct alignas(128) TileEntry {
  int32_t member, m0, n0;  // member of the X tile (and of the W tile unless composite); first row / column
  uint32_t idesc;          // tcgen05 instruction descriptor (M=128 or 256, N=bn, bf16 x bf16 -> fp32)
  uint32_t bn_nkb;         // tile width | K blocks << 16
  uint32_t misc;           // K=16 steps in the last K block | valid columns (min(bn, N-n0)) << 16 | kMisc* / kTrans*
  uint32_t pad0, pad1;
  ChunkDesc chunk[4];      // chunk c = accumulator columns [64c, 64c+64)
  const void* cbias[4];    // bias slice of each chunk (bf16) or NULL
};
static_assert(sizeof(TileEntry) == 128, "TileEntry is one 128-byte line = eight 16-byte pieces");

// Pipeline trace build (-DOPTB_GEMM_TRACE, paper_2607_02945_b200/build.py build(trace=True) -> a SEPARATE
// liboptimus_b200_trace.so; the product library has none of this): every warp role adds up the clock64() cycles it
// spends blocked on each barrier and writes one record per CTA at the end of the launch.  bench.py --side gemm_trace
// reads the records (profiles/r02_gemm_trace.md).
#ifdef OPTB_GEMM_TRACE
__device__ unsigned long long* g_gemm_trace = nullptr;     // [gridDim.x][16] or NULL
#define TR_DECL(name) long long name = 0
#define TR_NOW(name) name = clock64()
#define TR_WAIT(acc, stmt) do { const long long t0__ = clock64(); stmt; acc += clock64() - t0__; } while (0)
#define TR_ADD(acc, val) acc += (val)
#define TR_STORE(slot, val) do { if (g_gemm_trace) g_gemm_trace[(size_t)blockIdx.x * 16 + (slot)] = (unsigned long long)(val); } while (0)
#else
#define TR_DECL(name)
#define TR_NOW(name) do { } while (0)
#define TR_WAIT(acc, stmt) do { stmt; } while (0)
#define TR_ADD(acc, val) do { } while (0)
#define TR_STORE(slot, val) do { } while (0)
#endif

// Kernel-wide shared-memory map (dynamic, 1024-byte aligned base):
//   [0, nstages*stage_bytes)   operand ring: per stage a 128x64 X tile then the CTA's W tile (128B swizzle)
//   + 8 x 4 KB                 epilogue staging tiles (one per epilogue warp)
//   + kQDepth x 608 B          tile queue slots: 512 B bias slices (bf16) + 32 B entry head + 4 x 16 B chunk descriptors
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
  auto arrive_leader = [&](uint32_t bar) { if (NCTA == 2) mbar_arrive_cluster(mapa(bar, 0)); else mbar_arrive(bar); };

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
    // Dynamic: one atomic per CHUNK of 4 tiles (four 128-byte table lines: lane 8g+j holds 16-byte piece j of tile
    // g); the next chunk id is fetched while this chunk is published.
    // CTA pair: the leader's scheduler serves both CTAs (remote shared-memory stores + remote arrive).
    if (rank == 0) {
      const int n_sched = NCTA == 2 ? (int)num_clusters_x() : (int)gridDim.x;
      int qs = 0; uint32_t qph = 0;
      // queue slot `qs` of both CTAs: local st.shared + arrive; peer: st.async pieces counted on ITS qfull
      auto publish = [&](int qs_, uint32_t off, uint4 v) {
        sts128(q_slot(qs_) + off, v);
        if (NCTA == 2) st_async128(mapa(q_slot(qs_) + off, 1), v, mapa(qfull_bar(qs_), 1));
      };
      auto signal_full = [&](int qs_, uint32_t peer_bytes) {
        mbar_arrive(qfull_bar(qs_));
        if (NCTA == 2) mbar_expect_tx_cluster(mapa(qfull_bar(qs_), 1), peer_bytes);
      };
      auto load_lines = [&](int c) {
        uint4 v = make_uint4(0xFFFFFFFFu, 0, 0, 0);
        if (c < n_chunks) v = __ldg(chunks + (size_t)c * (8 * kTilesPerChunk) + lane);
        return v;
      };
      auto next_id = [&]() { int v = 0; if (lane == 0) v = atomicAdd(counters, 1) + n_sched; return v; };   // lane 0 only, not broadcast yet
      // bias slices of the 4 tiles of a chunk (this lane: columns [8 lane, 8 lane + 8) of each tile) and tensor-map
      // prefetches for them
      auto stage_tiles = [&](const uint4& e, uint4 (&bias_v)[kTilesPerChunk]) {
        const int cc = lane >> 3;                              // this lane's 64-column chunk
#pragma unroll
        for (int g = 0; g < kTilesPerChunk; ++g) {
          const int member = (int)__shfl_sync(0xffffffffu, e.x, 8 * g);
          const uint32_t misc = __shfl_sync(0xffffffffu, e.y, 8 * g + 1);
          const int src = 8 * g + 6 + (cc >> 1);               // cbias[cc]: piece 6 holds chunks 0,1; piece 7 chunks 2,3
          const uint32_t lo_a = __shfl_sync(0xffffffffu, e.x, src), hi_a = __shfl_sync(0xffffffffu, e.y, src);
          const uint32_t lo_b = __shfl_sync(0xffffffffu, e.z, src), hi_b = __shfl_sync(0xffffffffu, e.w, src);
          const uint64_t bptr = (cc & 1) ? (((uint64_t)hi_b << 32) | lo_b) : (((uint64_t)hi_a << 32) | lo_a);
          const uint4* bp = reinterpret_cast<const uint4*>(bptr) + (lane & 7);
          bias_v[g] = make_uint4(0, 0, 0, 0);
          if (member < 0) continue;                            // warp-uniform
          const int nvalid = (int)((misc >> 16) & 0x1FFu);
          if (bptr != 0 && 8 * lane + 8 <= nvalid) {
            bias_v[g] = __ldg(bp);
          } else if (bptr != 0 && 8 * lane < nvalid) {         // ragged N: the last piece element by element
            const unsigned short* be = reinterpret_cast<const unsigned short*>(bp);
            uint32_t w[4] = {0, 0, 0, 0};
            for (int t = 0; t < nvalid - 8 * lane; ++t) w[t >> 1] |= (uint32_t)__ldg(be + t) << (16 * (t & 1));
            bias_v[g] = make_uint4(w[0], w[1], w[2], w[3]);
          }
          const GemmMember* m = members + member;
          if (lane < 4)   // warm the descriptor cache for the member's tensor maps (tmA, tmB, tmY, tmB2)
            asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<const char*>(m) + 128 * lane) : "memory");
        }
      };
      // Look-ahead is ONE chunk id only: a scheduler that reserved chunks further ahead would hoard work the idle
      // pairs could take at the end of the launch (measured: the slowest pair +4 %).  The 4-deep tile queue hides
      // the two dependent global latencies (table lines, then bias slices) of a chunk behind the tiles in flight.
      int c = NCTA == 2 ? (int)cluster_id_x() : (int)blockIdx.x;
      int nextraw = 0;
      while (c < n_chunks) {
        nextraw = next_id();
        const uint4 e0 = load_lines(c);
        uint4 b0[kTilesPerChunk];
        stage_tiles(e0, b0);
#pragma unroll
        for (int g = 0; g < kTilesPerChunk; ++g) {
          if ((int)__shfl_sync(0xffffffffu, e0.x, 8 * g) < 0) continue;       // warp-uniform
          mbar_wait(qempty_bar(qs), qph ^ 1);
          publish(qs, 16 * lane, b0[g]);
          if ((lane >> 3) == g && (lane & 7) < 6) publish(qs, kQHeadOff + 16 * (lane & 7), e0);
          __syncwarp();
          if (lane == 0) signal_full(qs, kQSlotBytes);
          if (++qs == kQDepth) { qs = 0; qph ^= 1; }
        }
        c = __shfl_sync(0xffffffffu, nextraw, 0);
      }
      const int c2raw = nextraw;
      // end marker, then the last scheduler to get here re-arms the counters for the next launch of this plan
      mbar_wait(qempty_bar(qs), qph ^ 1);
      if (lane == 0) {
        publish(qs, kQHeadOff, make_uint4(0xFFFFFFFFu, 0, 0, 0));
        signal_full(qs, 16);
        __threadfence();
        // (c2raw < 0 is never true: the data dependency makes this scheduler's last id fetch return first)
        if (atomicAdd(counters + 1, 1 + (c2raw < 0)) == n_sched - 1) {
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
      TR_DECL(tr_q); TR_DECL(tr_empty); TR_DECL(tr_t0);
      TR_NOW(tr_t0);
      for (;;) {
        TR_WAIT(tr_q, mbar_wait(qfull_bar(qs), qph));
        const uint4 e0 = lds128(q_slot(qs) + kQHeadOff);
        const uint4 e1 = lds128(q_slot(qs) + kQHeadOff + 16);
        const int bn = (int)(e1.x & 0xFFFFu), nkb = (int)(e1.x >> 16);
        const bool composite = (e1.y & kMiscComposite) != 0;
        // composite tile: this CTA's part of the W tile is assembled from boxes of the chunks' members -- whole
        // 64-row chunks when the CTA's share is whole chunks, else 32-row half chunks (odd chunk count, CTA pair);
        // everything the k-loop needs (tensor map, first W row, byte offset step) goes to registers here
        const int nch = bn >> 6;
        const bool half_boxes = NCTA == 2 && (nch & 1);
        const int nbox = !composite ? 0 : half_boxes ? nch : nch / NCTA;
        const uint32_t box_bytes = half_boxes ? 4096u : 8192u;
        const CUtensorMap* box_tm[4] = {nullptr, nullptr, nullptr, nullptr};
        int box_row[4] = {0, 0, 0, 0};
        if (composite && (int)e0.x >= 0) {
          const uint4 d0 = lds128(q_slot(qs) + kQDescOff), d1 = lds128(q_slot(qs) + kQDescOff + 16);
          const uint4 d2 = lds128(q_slot(qs) + kQDescOff + 32), d3 = lds128(q_slot(qs) + kQDescOff + 48);
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const int u = (int)rank * nbox + j;                       // box index inside the tile
            const int ch = half_boxes ? (u >> 1) : u;
            const int mem = ch == 0 ? (int)d0.x : ch == 1 ? (int)d1.x : ch == 2 ? (int)d2.x : (int)d3.x;
            const int row = ch == 0 ? (int)d0.y : ch == 1 ? (int)d1.y : ch == 2 ? (int)d2.y : (int)d3.y;
            box_tm[j] = half_boxes ? &members[mem].tmB32 : &members[mem].tmB64;
            box_row[j] = row + (half_boxes ? 32 * (u & 1) : 0);
          }
        }
        arrive_leader(qempty_bar(qs));
        if (++qs == kQDepth) { qs = 0; qph ^= 1; }
        if ((int)e0.x < 0) break;
        const GemmMember* m = members + (int)e0.x;
        const int m0 = (int)e0.y + (int)rank * kBM;              // this CTA's 128 rows of the (pair) tile
        const int n0 = (int)e0.z + (int)rank * (bn / NCTA);      // this CTA's rows of the W tile
        const uint32_t b_bytes = (uint32_t)(bn / NCTA) * (kBK * 2);
        const CUtensorMap* tmB = NCTA == 2 ? &m->tmB2 : &m->tmB;
        for (int kb = 0; kb < nkb; ++kb) {
          TR_WAIT(tr_empty, mbar_wait(empty_bar(stage), phase ^ 1));
          const uint32_t sa = sbase + stage * stage_bytes;
          if (NCTA == 2) {
            // the leader's barrier counts the bytes of both CTAs
            if (rank == 0) mbar_expect_tx(full_bar(stage), 2 * (kABytes + b_bytes));
            const uint32_t lb = mapa(full_bar(stage), 0);
            if (e1.y & kTransX) {                    // stored [K, M]: two 64x64 boxes (contraction rows, M contiguous)
              tma_load_2d_pair(sa, &m->tmA, lb, m0, kb * kBK);
              tma_load_2d_pair(sa + 8192, &m->tmA, lb, m0 + 64, kb * kBK);
            } else {
              tma_load_2d_pair(sa, &m->tmA, lb, kb * kBK, m0);
            }
            if (e1.y & kTransW) {                    // stored [K, N]: this CTA's BN/2 columns = BN/128 boxes of 64
              for (int j = 0; j < bn / 128; ++j) tma_load_2d_pair(sa + kABytes + j * 8192, &m->tmB, lb, n0 + 64 * j, kb * kBK);
            } else if (composite) {
#pragma unroll
              for (int j = 0; j < 4; ++j)
                if (j < nbox) tma_load_2d_pair(sa + kABytes + j * box_bytes, box_tm[j], lb, kb * kBK, box_row[j]);
            } else {
              tma_load_2d_pair(sa + kABytes, tmB, lb, kb * kBK, n0);
            }
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
            } else if (composite) {
#pragma unroll
              for (int j = 0; j < 4; ++j)
                if (j < nbox) tma_load_2d(sa + kABytes + j * box_bytes, box_tm[j], full_bar(stage), kb * kBK, box_row[j]);
            } else {
              tma_load_2d(sa + kABytes, tmB, full_bar(stage), kb * kBK, n0);
            }
          }
          if (++stage == nstages) { stage = 0; phase ^= 1; }
        }
      }
      TR_STORE(0, clock64() - tr_t0); TR_STORE(1, tr_q); TR_STORE(2, tr_empty);
    }
  } else if (warp == 1) {
    // ------------------------------------------- MMA issuer (leader only) ----
    if (lane == 0 && rank == 0) {
      int stage = 0; uint32_t phase = 0;
      int as = 0; uint32_t aphase = 0;
      int qs = 0; uint32_t qph = 0;
      // K-major shared-memory descriptors of the current ring stage, advanced with the stage (no rebuild per k-block)
      const uint64_t adesc_ring0 = umma_desc_sw128(sbase), desc_stage_step = (uint64_t)(stage_bytes >> 4);
      uint64_t adesc_ring = adesc_ring0, bdesc_ring = adesc_ring0 + (kABytes >> 4);
      TR_DECL(tr_q); TR_DECL(tr_full); TR_DECL(tr_tempty); TR_DECL(tr_t0); TR_DECL(tr_tiles); TR_DECL(tr_kb);
      TR_NOW(tr_t0);
      // the next tile's header is taken from the queue BEFORE the last k-block of the current tile is issued, while
      // the tensor pipe still has work: the queue wait + two shared-memory loads are off the tile-to-tile path
      uint4 e0, e1;
      auto next_header = [&]() {
        TR_WAIT(tr_q, mbar_wait(qfull_bar(qs), qph));
        e0 = lds128(q_slot(qs) + kQHeadOff);
        e1 = lds128(q_slot(qs) + kQHeadOff + 16);
        arrive_leader(qempty_bar(qs));
        if (++qs == kQDepth) { qs = 0; qph ^= 1; }
      };
      next_header();
      for (;;) {
        if ((int)e0.x < 0) break;
        const uint32_t idesc = e0.w;
        const int nkb = (int)(e1.x >> 16), klast = (int)(e1.y & 0xFFu);
        const bool tx = (e1.y & kTransX) != 0, tw = (e1.y & kTransW) != 0;
        TR_ADD(tr_tiles, 1); TR_ADD(tr_kb, nkb * (int)(e1.x & 0xFFFFu));     // k-blocks weighted by tile width = tensor work
        TR_WAIT(tr_tempty, mbar_wait(tempty_bar(as), aphase ^ 1));   // the epilogues (of both CTAs) have drained this accumulator stage
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + as * kMaxBN;
        // the issue loop sits on the critical path between "stage landed" and "tensor pipe busy": everything that does
        // not change inside a tile is hoisted, and the common K-major case keeps compile-time descriptor steps
        if (!tx && !tw) {
          for (int kb = 0; kb < nkb; ++kb) {
            if (kb + 1 == nkb) next_header();    // (e0 / e1 of THIS tile are not used below this point)
            TR_WAIT(tr_full, mbar_wait(full_bar(stage), phase));
            tc_fence_after();
            // per K=16 step: +32 bytes inside the 128-byte swizzle row (+2 encoded)
            if (kb + 1 < nkb) {                  // a whole k-block: four steps, straight-line
              if (NCTA == 2) {
                tc_mma_bf16_pair(d_tmem, adesc_ring, bdesc_ring, idesc, (uint32_t)kb);
                tc_mma_bf16_pair(d_tmem, adesc_ring + 2, bdesc_ring + 2, idesc, 1u);
                tc_mma_bf16_pair(d_tmem, adesc_ring + 4, bdesc_ring + 4, idesc, 1u);
                tc_mma_bf16_pair(d_tmem, adesc_ring + 6, bdesc_ring + 6, idesc, 1u);
              } else {
                tc_mma_bf16(d_tmem, adesc_ring, bdesc_ring, idesc, (uint32_t)kb);
                tc_mma_bf16(d_tmem, adesc_ring + 2, bdesc_ring + 2, idesc, 1u);
                tc_mma_bf16(d_tmem, adesc_ring + 4, bdesc_ring + 4, idesc, 1u);
                tc_mma_bf16(d_tmem, adesc_ring + 6, bdesc_ring + 6, idesc, 1u);
              }
            } else {
              for (int k = 0; k < klast; ++k) {
                if (NCTA == 2) tc_mma_bf16_pair(d_tmem, adesc_ring + 2 * k, bdesc_ring + 2 * k, idesc, (kb | k) != 0);
                else tc_mma_bf16(d_tmem, adesc_ring + 2 * k, bdesc_ring + 2 * k, idesc, (kb | k) != 0);
              }
            }
            // frees the smem stage (in both CTAs) when these MMAs retire
            if (NCTA == 2) tc_commit_pair(empty_bar(stage)); else tc_commit(empty_bar(stage));
            adesc_ring += desc_stage_step; bdesc_ring += desc_stage_step;
            if (++stage == nstages) { stage = 0; phase ^= 1; adesc_ring = adesc_ring0; bdesc_ring = adesc_ring0 + (kABytes >> 4); }
          }
        } else {
          // an operand stored transposed: MN-major descriptors, a K=16 step is two groups of 8 contraction rows (+128)
          const uint64_t astep = tx ? 128 : 2, bstep = tw ? 128 : 2;
          for (int kb = 0; kb < nkb; ++kb) {
            if (kb + 1 == nkb) next_header();
            TR_WAIT(tr_full, mbar_wait(full_bar(stage), phase));
            tc_fence_after();
            const uint32_t sa = sbase + stage * stage_bytes;
            const uint64_t adesc = tx ? umma_desc_sw128_mn(sa) : umma_desc_sw128(sa);
            const uint64_t bdesc = tw ? umma_desc_sw128_mn(sa + kABytes) : umma_desc_sw128(sa + kABytes);
            const int ksteps = kb + 1 < nkb ? kBK / 16 : klast;
            for (int k = 0; k < ksteps; ++k) {
              if (NCTA == 2) tc_mma_bf16_pair(d_tmem, adesc + astep * k, bdesc + bstep * k, idesc, (kb | k) != 0);
              else tc_mma_bf16(d_tmem, adesc + astep * k, bdesc + bstep * k, idesc, (kb | k) != 0);
            }
            if (NCTA == 2) tc_commit_pair(empty_bar(stage)); else tc_commit(empty_bar(stage));
            adesc_ring += desc_stage_step; bdesc_ring += desc_stage_step;
            if (++stage == nstages) { stage = 0; phase ^= 1; adesc_ring = adesc_ring0; bdesc_ring = adesc_ring0 + (kABytes >> 4); }
          }
        }
        if (NCTA == 2) tc_commit_pair(tfull_bar(as)); else tc_commit(tfull_bar(as));   // accumulator complete
        if (++as == kAccStages) { as = 0; aphase ^= 1; }
      }
      TR_STORE(3, clock64() - tr_t0); TR_STORE(4, tr_q); TR_STORE(5, tr_full); TR_STORE(6, tr_tempty);
      TR_STORE(7, tr_tiles); TR_STORE(8, tr_kb);
    }
  } else {
    // ----------------------------------------------------------- epilogue ----
    const int ew = warp - kFirstEpiWarp;
    const int quad = warp & 3;               // TMEM lane quadrant this warp may read
    const int half = ew >> 2;                // 0: even 64-column chunks, 1: odd ones
    const uint32_t sbuf = epi_base + (uint32_t)ew * kEpiBufBytes;
    const uint32_t srow = sbuf + lane * 128;
    const uint32_t srow8 = sbuf + lane * 64;  // FP8 codes: 64 bytes per row, 64-byte swizzle
    int as = 0; uint32_t aphase = 0;
    int qs = 0; uint32_t qph = 0;
    TR_DECL(tr_q); TR_DECL(tr_tfull); TR_DECL(tr_store); TR_DECL(tr_t0);
    TR_NOW(tr_t0);
    for (;;) {
      TR_WAIT(tr_q, mbar_wait(qfull_bar(qs), qph));
      const uint32_t slot = q_slot(qs);
      const uint4 e0 = lds128(slot + kQHeadOff);
      const uint4 e1 = lds128(slot + kQHeadOff + 16);
      if ((int)e0.x < 0) break;
      const int m0 = (int)e0.y + (int)rank * kBM;
      const int bn = (int)(e1.x & 0xFFFFu);
      TR_WAIT(tr_tfull, mbar_wait(tfull_bar(as), aphase));
      tc_fence_after();
      const uint32_t t_row = tmem_base + ((uint32_t)(quad * 32) << 16) + as * kMaxBN;
      const int nchunks = (bn + 63) >> 6;
      bool released = false;
      for (int c = half; c < nchunks; c += 2) {
        uint32_t v[64];
        tc_ld_32x32(t_row + c * 64, *reinterpret_cast<uint32_t(*)[32]>(&v[0]));
        tc_ld_32x32(t_row + c * 64 + 32, *reinterpret_cast<uint32_t(*)[32]>(&v[32]));
        const uint4 cd = lds128(slot + kQDescOff + 16 * c);      // this chunk: member, first column, act | flags, FP8 scale
        tc_wait_ld();
        if (c + 2 >= nchunks) {              // this warp's part of the accumulator is in registers
          tc_fence_before();
          __syncwarp();
          if (lane == 0) arrive_leader(tempty_bar(as));
          released = true;
        }
        const GemmMember* m = members + (int)cd.x;
        const int act = (int)(cd.z & 0xFFu);
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
        TR_WAIT(tr_store, if (lane == 0) tma_store_wait_read<0>());
        __syncwarp();
        if (cd.z & kChunkHasY) {
#pragma unroll
          for (int j = 0; j < 8; ++j)            // 16-byte pieces at their 128B-swizzled position
            sts128(srow + ((j ^ (lane & 7)) << 4), make_uint4(p[4 * j], p[4 * j + 1], p[4 * j + 2], p[4 * j + 3]));
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) {
            tma_store_2d(&m->tmY, sbuf, (int)cd.y, m0 + quad * 32);
            tma_store_commit();
          }
        }
        if (cd.z & kChunkHasY8) {
          // FP8 copy (activation quantisation fused into the producer of the saved tensor): the
          // E4M3 codes of the ROUNDED bf16 values x scale8 -- what OPT_PW_QUANT_E4M3 would compute from the stored Y
          const float sc = __uint_as_float(cd.w);
          uint32_t q[16];
#pragma unroll
          for (int j = 0; j < 16; ++j) q[j] = quant4_e4m3(p[2 * j], p[2 * j + 1], sc);
          if (cd.z & kChunkHasY) {               // the bf16 store still reads the staging buffer
            if (lane == 0) tma_store_wait_read<0>();
            __syncwarp();
          }
#pragma unroll
          for (int j = 0; j < 4; ++j)            // 16-byte pieces at their 64B-swizzled position
            sts128(srow8 + ((j ^ ((lane >> 1) & 3)) << 4), make_uint4(q[4 * j], q[4 * j + 1], q[4 * j + 2], q[4 * j + 3]));
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) {
            tma_store_2d(&m->tmY8, sbuf, (int)cd.y, m0 + quad * 32);
            tma_store_commit();
          }
        }
      }
      if (!released) {                       // no chunk for this warp in a narrow tile: still hand the stage back
        tc_fence_before();
        __syncwarp();
        if (lane == 0) arrive_leader(tempty_bar(as));
      }
      __syncwarp();                          // every lane has read the slot's bias and chunk descriptors
      if (lane == 0) arrive_leader(qempty_bar(qs));
      if (++qs == kQDepth) { qs = 0; qph ^= 1; }
      if (++as == kAccStages) { as = 0; aphase ^= 1; }
    }
    if (lane == 0) tma_store_wait_all();
    if (ew == 0 && lane == 0) { TR_STORE(9, clock64() - tr_t0); TR_STORE(10, tr_q); TR_STORE(11, tr_tfull); TR_STORE(12, tr_store); }
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

}  // namespace optb
