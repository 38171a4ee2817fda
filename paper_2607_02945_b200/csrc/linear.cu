// Grouped Linear (+bias +activation): N independent  Y_i = act_i(X_i W_i^T + b_i)
// in ONE launch -- batch_linear / batch_linear_post_grad / batch_linear_lhs with the epilogue
// fused (PAPER.md:292, :148 group fusion; include/optimus_b200.h).  This file: the host planner
// (validation, tile table, tensor maps), the launchers, and the fp32 kernel.
//
//   grouped_gemm_sm100_kernel  bf16 in/out, fp32 accumulate: grouped_gemm_sm100.cuh (tcgen05 / TMEM / TMA, CTA pairs,
//       device-side tile scheduler, fused epilogue incl. the optional FP8 copy of the output).
//   grouped_gemm_f32_kernel    plain fp32 FFMA (no TF32) 32x32 tiles for fp32 groups (configs[0]); prefix-sum tile
//       walk, accurate tanhf/expf epilogue.
//   huge-M / tiny-K-and-N groups go to the streaming row kernel of linear_skinny.cu.
#include <algorithm>
#include <map>
#include <set>
#include <tuple>
#include <cstdlib>

#include "grouped_gemm_sm100.cuh"

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
// (the kernel lives in grouped_gemm_sm100.cuh)
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

#ifdef OPTB_GEMM_TRACE
// trace build only: where the grouped GEMM writes its per-CTA wait-cycle records ([grid][16] uint64), or NULL
extern "C" int opt_trace_set_gemm_buffer(void* device_buffer) {
  unsigned long long* p = static_cast<unsigned long long*>(device_buffer);
  return (int)cudaMemcpyToSymbol(g_gemm_trace, &p, sizeof p);
}
#endif

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
#ifndef OPTB_GEMM_TRACE
  for (int32_t r : opts.reserved) if (r != 0) return fail(OPT_ERR_INVALID_ARG, "options.reserved must be zero");
#endif
  if (n < 1 || n > 65535) return fail(OPT_ERR_INVALID_ARG, "n = %d outside [1, 65535]", n);
  if (io != OPT_F32 && io != OPT_BF16) return fail(OPT_ERR_INVALID_ARG, "bad io dtype %d", (int)io);
  const int esz = elem_size(io), V = vec_elems(io);
  std::vector<Region> regions;
  int64_t flops = 0, bytes = 0;
  std::set<std::tuple<const void*, int64_t, int32_t, int32_t>> seen_x;
  // huge-M / tiny-K-and-N groups (decompose_mm_pass) stream through the SIMT row kernel (linear_skinny.cu)
  bool skinny = io == OPT_BF16 && !opts.no_skinny;
  for (int32_t i = 0; skinny && i < n; ++i) skinny = skinny_linear_member(members[i]) && !members[i].y8;
  for (int32_t i = 0; i < n; ++i) {
    const opt_linear_member& m = members[i];
    if (!m.x || !m.w || (!m.y && !m.y8)) return fail(OPT_ERR_INVALID_ARG, "member %d: NULL pointer", i);
    if (m.M < 1 || m.N < 1 || m.K < 1) return fail(OPT_ERR_INVALID_ARG, "member %d: M=%d N=%d K=%d must be >= 1", i, m.M, m.N, m.K);
    if (m.act < OPT_ACT_NONE || m.act > OPT_ACT_SIGMOID) return fail(OPT_ERR_INVALID_ARG, "member %d: bad activation %d", i, m.act);
    if (m.layout & ~(OPT_LAYOUT_X_TRANSPOSED | OPT_LAYOUT_W_TRANSPOSED)) return fail(OPT_ERR_INVALID_ARG, "member %d: bad layout flags %d", i, m.layout);
    const bool tx = m.layout & OPT_LAYOUT_X_TRANSPOSED, tw = m.layout & OPT_LAYOUT_W_TRANSPOSED;
    if ((tx || tw) && io != OPT_BF16) return fail(OPT_ERR_UNSUPPORTED, "member %d: transposed operands are implemented for bf16 groups only", i);
    // stored shapes: x [M,K] or (transposed) [K,M]; w [N,K] or (transposed) [K,N]
    const int32_t x_rows = tx ? m.K : m.M, x_cols = tx ? m.M : m.K, w_rows = tw ? m.K : m.N, w_cols = tw ? m.N : m.K;
    if ((x_rows > 1 && m.ldx < x_cols) || (m.y && m.M > 1 && m.ldy < m.N) || (w_rows > 1 && m.ldw < w_cols))
      return fail(OPT_ERR_INVALID_ARG, "member %d: row stride smaller than the row", i);
    if (!aligned16(m.x) || !aligned16(m.w) || !aligned16(m.y) || !aligned16(m.bias))
      return fail(OPT_ERR_ALIGNMENT, "member %d: pointers must be 16-byte aligned", i);
    if (m.y8) {      // FP8 copy of the output (activation quantisation fused into the epilogue)
      if (io != OPT_BF16 || m.layout) return fail(OPT_ERR_UNSUPPORTED, "member %d: the FP8 output is implemented for bf16 groups with layout 0", i);
      if (!(m.scale8 > 0.f) || !(m.scale8 < INFINITY)) return fail(OPT_ERR_INVALID_ARG, "member %d: scale8 must be a positive finite number", i);
      if (m.M > 1 && m.ldy8 < m.N) return fail(OPT_ERR_INVALID_ARG, "member %d: ldy8 smaller than the row", i);
      if (!aligned16(m.y8) || m.ldy8 % 16 || m.N % 16)
        return fail(OPT_ERR_ALIGNMENT, "member %d: y8 needs a 16-byte aligned base, ldy8 %% 16 == 0 and N %% 16 == 0", i);
    }
    // bf16: K and N need NOT be multiples of 8 -- TMA zero-fills the K / N tails of the operand tiles and clips the
    // store, which is what pad_aten_mm_pass achieves by padding; only bases and row strides must be
    // 16-byte aligned.  fp32 (SIMT path): multiples of 4.
    if (io == OPT_F32 && (m.K % V || m.N % V))
      return fail(OPT_ERR_ALIGNMENT, "member %d: K=%d and N=%d must be multiples of %d", i, m.K, m.N, V);
    if (skinny) {      // rows are read and written as 4-byte words
      if (m.ldx % 2 || m.ldw % 2 || m.ldy % 2)
        return fail(OPT_ERR_ALIGNMENT, "member %d: row strides must be even (4-byte words)", i);
    } else if (m.ldx % V || m.ldw % V || (m.y && m.ldy % V)) {
      return fail(OPT_ERR_ALIGNMENT, "member %d: row strides must be multiples of %d elements", i, V);
    }
    regions.push_back({(uintptr_t)m.x, m.ldx * esz, (int64_t)x_cols * esz, x_rows, false, i});
    regions.push_back({(uintptr_t)m.w, m.ldw * esz, (int64_t)w_cols * esz, w_rows, false, i});
    if (m.bias) regions.push_back({(uintptr_t)m.bias, 0, (int64_t)m.N * esz, 1, false, i});
    if (m.y) regions.push_back({(uintptr_t)m.y, m.ldy * esz, (int64_t)m.N * esz, m.M, true, i});
    if (m.y8) regions.push_back({(uintptr_t)m.y8, m.ldy8, (int64_t)m.N, m.M, true, i});
    flops += 2ll * m.M * m.N * m.K;
    // an input shared by several members (batch_linear_lhs) is read once
    const bool first_use_of_x = seen_x.insert(std::make_tuple(m.x, m.ldx, m.M, tx ? -m.K : m.K)).second;
    bytes += ((first_use_of_x ? (int64_t)m.M * m.K : 0) + (int64_t)m.N * m.K + (m.bias ? m.N : 0) + (m.y ? (int64_t)m.M * m.N : 0)) * esz +
             (m.y8 ? (int64_t)m.M * m.N : 0);
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
  // (transposed operands run through both: a CTA of a pair stages its own 128 rows of X^T and its own half of the
  // W^T tile as rows of 64 x 64 boxes, so a transposed-W tile of a pair is a multiple of 128 columns wide)
  const int ncta = opts.cta_pair == 1 ? 1 : 2;
  const int tile_m = kBM * ncta;
  struct MemberTiling { int bn, nbn, nkb, klast; uint32_t flags, cflags; };
  std::vector<MemberTiling> tiling(n);
  // tcgen05 instruction descriptor, kind::f16: D fp32 (bits 4-5 = 1), A bf16 (bits 7-9 = 1), B bf16
  // (bits 10-12 = 1), A / B MN-major (bits 15 / 16), N>>3 at bits 17-22, M>>4 at bits 24-28.
  auto make_idesc = [&](int bn, bool tx, bool tw) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)tx << 15) | ((uint32_t)tw << 16) | ((uint32_t)(bn >> 3) << 17) |
           ((uint32_t)(tile_m >> 4) << 24);
  };
  int max_bn = 16;
  for (int32_t i = 0; i < n; ++i) {
    const opt_linear_member& m = members[i];
    GemmMember& t = tab[i];
    const bool tx = m.layout & OPT_LAYOUT_X_TRANSPOSED, tw = m.layout & OPT_LAYOUT_W_TRANSPOSED;
    int bn = choose_bn(m.N);
    if (tw) bn = std::min(kMaxBN, (bn + 64 * ncta - 1) / (64 * ncta) * (64 * ncta));   // MN-major W tiles are rows of 64x64 boxes per CTA
    opt_status st;
    // K-major operand: box {64 k, rows};  transposed operand (stored [K, out]): box {64 out, 64 k}
    st = tx ? encode_2d(enc, &t.tmA, m.x, m.K, m.M, m.ldx, 64, kBK, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, "X^T", i)
            : encode_2d(enc, &t.tmA, m.x, m.M, m.K, m.ldx, kBK, kBM, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, "X", i);
    if (!st) st = tw ? encode_2d(enc, &t.tmB, m.w, m.K, m.N, m.ldw, 64, kBK, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, "W^T", i)
                     : encode_2d(enc, &t.tmB, m.w, m.N, m.K, m.ldw, kBK, bn, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, "W", i);
    if (!st && m.y) st = encode_2d(enc, &t.tmY, m.y, m.M, m.N, m.ldy, 64, 32, CU_TENSOR_MAP_L2_PROMOTION_NONE, "Y", i);
    if (!st && !tw) st = encode_2d(enc, &t.tmB2, m.w, m.N, m.K, m.ldw, kBK, bn / 2, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, "W/2", i);
    if (!st && !tw) st = encode_2d(enc, &t.tmB64, m.w, m.N, m.K, m.ldw, kBK, 64, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, "W/64", i);
    if (!st && !tw) st = encode_2d(enc, &t.tmB32, m.w, m.N, m.K, m.ldw, kBK, 32, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, "W/32", i);
    if (!st && m.y8) st = encode_2d_u8(enc, &t.tmY8, m.y8, m.M, m.N, m.ldy8, 64, 32, "Y8", i);
    if (st) {
      delete p;
      return st;
    }
    MemberTiling& tl = tiling[i];
    tl.bn = bn; tl.nbn = (m.N + bn - 1) / bn; tl.nkb = (m.K + kBK - 1) / kBK;
    tl.klast = (m.K - (tl.nkb - 1) * kBK + 15) / 16;
    tl.flags = (tx ? kTransX : 0u) | (tw ? kTransW : 0u);
    tl.cflags = (uint32_t)m.act | (m.y ? kChunkHasY : 0u) | (m.y8 ? kChunkHasY8 : 0u);
    max_bn = std::max(max_bn, bn);
  }
  // Schedule order: (LHS group,) member-major, m-block, n-block -- the n-blocks of one X row panel are adjacent, so the
  // CTAs that take them side by side fetch the panel from HBM once (re-reads hit L2), and a member's W stays
  // hot in L2 while its tiles are in flight.  (Interleaving tensor-bound with HBM-bound members was measured:
  // no gain on configs[2], the kernel is bound by L2->SM operand traffic there.)
  // batch_linear_lhs: members that share ONE input X (same pointer, stride, M, K) form an LHS group.
  //   * If every member of the group has N % 64 == 0 the weights are LOGICALLY CONCATENATED: the group is tiled as
  //     one [M, sum N] problem in 64-column chunks, a tile (up to 4 chunks = 256 columns) may span several members
  //     (COMPOSITE tile: its W tile is assembled from 64-row boxes of the members' W, each chunk keeps its own
  //     bias / activation / output) -- eight N=64 members cost two 256-wide tiles per X panel instead of eight 64-wide.
  //   * Otherwise the group's schedule is m-block-major ACROSS its members (all n-blocks of all members that read a
  //     given X row panel are adjacent): the panel is fetched from HBM once for the whole group.
  std::vector<TileEntry> flat;
  auto chunk_of = [&](int32_t i, int n0c) {
    const opt_linear_member& m = members[i];
    ChunkDesc d;
    d.member = i; d.n0 = n0c; d.act_flags = tiling[i].cflags; d.scale8 = m.y8 ? m.scale8 : 0.f;
    return d;
  };
  auto bias_of = [&](int32_t i, int n0c) -> const void* {
    return members[i].bias ? static_cast<const char*>(members[i].bias) + (size_t)n0c * 2 : nullptr;
  };
  auto push_tiles = [&](int32_t i, int mb) {
    const opt_linear_member& m = members[i];
    const MemberTiling& tl = tiling[i];
    for (int nb = 0; nb < tl.nbn; ++nb) {
      TileEntry e;
      memset(&e, 0, sizeof e);
      e.member = i; e.m0 = mb * tile_m; e.n0 = nb * tl.bn;
      e.idesc = make_idesc(tl.bn, tl.flags & kTransX, tl.flags & kTransW);
      e.bn_nkb = (uint32_t)tl.bn | ((uint32_t)tl.nkb << 16);
      e.misc = (uint32_t)tl.klast | ((uint32_t)std::min(tl.bn, m.N - e.n0) << 16) | tl.flags;
      for (int c = 0; c * 64 < tl.bn; ++c) { e.chunk[c] = chunk_of(i, e.n0 + 64 * c); e.cbias[c] = bias_of(i, e.n0 + 64 * c); }
      flat.push_back(e);
    }
  };
  {
    std::map<std::tuple<const void*, int64_t, int32_t, int32_t>, std::vector<int32_t>> lhs;
    std::vector<std::tuple<const void*, int64_t, int32_t, int32_t>> first_seen;
    for (int32_t i = 0; i < n; ++i) {
      const auto key = std::make_tuple(members[i].x, members[i].ldx, members[i].M, members[i].layout ? -members[i].K : members[i].K);
      if (lhs.find(key) == lhs.end()) first_seen.push_back(key);
      lhs[key].push_back(i);
    }
    const bool no_lhs = opts.no_lhs_order != 0;
    if (no_lhs) { first_seen.clear(); for (int32_t i = 0; i < n; ++i) { const int nmb = (members[i].M + tile_m - 1) / tile_m; for (int mb = 0; mb < nmb; ++mb) push_tiles(i, mb); } }
    for (const auto& key : first_seen) {
      const std::vector<int32_t>& grp = lhs[key];
      const int nmb = (std::get<2>(key) + tile_m - 1) / tile_m;
      bool concat = grp.size() >= 2;
      for (int32_t i : grp) concat = concat && members[i].layout == 0 && members[i].N % 64 == 0;
      if (!concat) {
        for (int mb = 0; mb < nmb; ++mb)
          for (int32_t i : grp) push_tiles(i, mb);
        continue;
      }
      // logically concatenated weights: the group's 64-column chunks, cut into tiles of 4 chunks (the last: what is left)
      std::vector<std::pair<int32_t, int>> vchunks;
      for (int32_t i : grp)
        for (int n0c = 0; n0c < members[i].N; n0c += 64) vchunks.push_back({i, n0c});
      std::vector<std::pair<size_t, int>> vtiles;     // (first chunk, number of chunks)
      for (size_t c = 0; c < vchunks.size();) {
        const size_t left = vchunks.size() - c;
        const int take = (int)std::min<size_t>(4, left);
        vtiles.push_back({c, take});
        c += take;
      }
      const MemberTiling& tl0 = tiling[grp[0]];         // K is shared by the group
      for (int mb = 0; mb < nmb; ++mb)
        for (const auto& vt : vtiles) {
          TileEntry e;
          memset(&e, 0, sizeof e);
          const int bn = 64 * vt.second;
          e.member = grp[0]; e.m0 = mb * tile_m; e.n0 = (int32_t)(64 * vt.first);
          e.idesc = make_idesc(bn, false, false);
          e.bn_nkb = (uint32_t)bn | ((uint32_t)tl0.nkb << 16);
          e.misc = (uint32_t)tl0.klast | ((uint32_t)bn << 16) | kMiscComposite;
          for (int c = 0; c < vt.second; ++c) {
            const auto& vc = vchunks[vt.first + c];
            e.chunk[c] = chunk_of(vc.first, vc.second);
            e.cbias[c] = bias_of(vc.first, vc.second);
          }
          max_bn = std::max(max_bn, bn);
          flat.push_back(e);
        }
    }
  }
  tiles = (int64_t)flat.size();
  if (tiles > INT32_MAX / 2) { delete p; return fail(OPT_ERR_UNSUPPORTED, "too many tiles"); }
  // Chunks of 4 tiles (four 128-byte lines, one atomic); the last waves go one tile per chunk so that the tail of the
  // persistent loop is balanced at tile granularity.  How many: a 4-tile chunk of long tiles taken just before the tail
  // keeps its CTA busy for several tile times, and the tail has to hold that much work per CTA to level it -- with
  // configs[2]'s tiles (8.8 k-blocks on average, up to 16) 3 waves left the CTA pairs finishing 10 % apart (trace:
  // 365 k .. 406 k cycles) and 16 waves are 4 % faster (263 -> 252 us; 24: the same, 40: slower again); short tiles
  // (configs[4]'s groups: 2 - 5 k-blocks, HBM-bound) do not need it and would outrun a scheduler that serves one tile
  // per atomic (C4b: 594 us with 3 - 6 waves, 601 with 16).  Hence twice the average k-block count, in [3, 16].
  TileEntry pad_entry;
  memset(&pad_entry, 0, sizeof pad_entry);
  pad_entry.member = -1;
  uint64_t sum_nkb = 0;
  for (const TileEntry& e : flat) sum_nkb += e.bn_nkb >> 16;
  const size_t tail_waves = std::min<size_t>(16, std::max<size_t>(3, (size_t)((2 * sum_nkb + flat.size() / 2) / std::max<size_t>(1, flat.size()))));
  const int n_sched = num_sms / ncta;                         // persistent CTAs (or CTA pairs)
  const size_t tail = std::min(flat.size(), tail_waves * n_sched);
  const size_t body = flat.size() - tail;
  // the tail goes longest tile first (cost = K blocks x width), so that the last tiles handed out are the cheap ones
  std::stable_sort(flat.begin() + body, flat.end(), [](const TileEntry& a, const TileEntry& b) {
    return (uint64_t)(a.bn_nkb >> 16) * (a.bn_nkb & 0xFFFFu) > (uint64_t)(b.bn_nkb >> 16) * (b.bn_nkb & 0xFFFFu);
  });
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
  int nstages = std::min(kMaxStages, (kSmemMax - kSmemFixed) / stage_bytes);
#ifdef OPTB_GEMM_TRACE
  if (opts.reserved[0] > 0) nstages = std::min(nstages, (int)opts.reserved[0]);     // trace build: ring-depth sensitivity
#endif
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
