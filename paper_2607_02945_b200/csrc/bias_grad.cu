// batched_bias_grad: the bias gradients of N independent Linear layers in ONE launch (
// batch_linear_post_grad operates on post-grad graphs, and the headline metric is TRAINING
// throughput):
//
//   db[n] = sum over m of dZ[m, n]            dZ:[M,N] bf16, db:[N] fp32 or bf16
//
// and, when a member names the stored forward output y of a ReLU epilogue, the mask of that ReLU fused in front
// (vertical fusion inside the backward): dZ = dY where y > 0 else 0 is formed in registers from dY and
// y, written once (dz_out, optional) and summed in the same pass -- 3 M N instead of 4 M N elements of HBM traffic.
//
// Design (HBM-bound: dZ read once, nothing else of size moves):
//   * a work item is (member, row part, 256-column tile); a 16-byte vector column of the tile is owned by one lane,
//     the L = 2^k lanes that cover the tile walk a row together (coalesced 16 L-byte segments), the 256/L row
//     groups of the block stride over the part's rows, four rows of loads in flight per thread;
//   * fp32 accumulators in registers (packed f32x2 adds); at the end of the part the row groups are summed through
//     shared memory in group order and the part's partial goes to a plan-owned workspace; the LAST block of a
//     member (atomic ticket, re-armed by that block) adds the parts in part order and writes db: one launch,
//     no atomics on data, bitwise reproducible from run to run.
#include <algorithm>
#include <cstring>

#include "common.h"

namespace optb {

struct BgMember {
  const char* dz; char* db;
  const char* y; char* dzo;        // fused ReLU mask: stored forward output, masked gradient out (either may be NULL)
  int64_t ldz16, ldy16, lddzo16;   // row strides in 16-byte vectors
  float* ws;                       // [nparts][N] fp32 partial sums (plan workspace)
  int32_t* ticket;                 // blocks of this member that have finished
  int32_t rows, nvec, nparts, nblocks;
  int32_t l_log2;                  // lanes per row of a column tile
  int32_t act;                     // fused derivative: 0 / 1 ReLU mask, 2 tanh, 3 sigmoid
};
struct BgBlock { int32_t member, row0, nrows, part, vec0; };

constexpr int kBgThreads = 256;
constexpr int kBgTileVec = 32;       // 32 vectors = 256 bf16 columns per tile
constexpr int kBgMinBlocks = 6;
constexpr int kBgBlockBytes = 131072;
constexpr int kBgInflight = 4;       // rows of loads in flight per thread

// torch threshold_backward on a bf16 pair: keep the gradient unless y <= 0 (a NaN y keeps it); the zero written is +0
__device__ __forceinline__ uint32_t bg_mask2(uint32_t g, uint32_t y) {
  const uint32_t m = (bf16_lo(y) <= 0.f ? 0u : 0x0000FFFFu) | (bf16_hi(y) <= 0.f ? 0u : 0xFFFF0000u);
  return g & m;
}
__device__ __forceinline__ int4 bg_mask(int4 g, const int4& y) {
  g.x = (int)bg_mask2((uint32_t)g.x, (uint32_t)y.x); g.y = (int)bg_mask2((uint32_t)g.y, (uint32_t)y.y);
  g.z = (int)bg_mask2((uint32_t)g.z, (uint32_t)y.z); g.w = (int)bg_mask2((uint32_t)g.w, (uint32_t)y.w);
  return g;
}

// derivative of the epilogue from its stored output, applied to a 16-byte vector of gradients: act 0 / 1 the ReLU mask
// (bit-exact select), 2 tanh dy (1 - y^2), 3 sigmoid dy (1 - y) y -- fp32, one rounding to bf16, the same arithmetic as
// OPT_PW_TANH_BWD / OPT_PW_SIGMOID_BWD of the pointwise kernel (bitwise equal results)
__device__ __forceinline__ float bg_dact(float g, float y, int act) { return act == 2 ? g * fmaf(-y, y, 1.f) : g * ((1.f - y) * y); }
__device__ __forceinline__ int4 bg_deriv(int4 g, const int4& y, int act) {
  if (act <= 1) return bg_mask(g, y);
  uint32_t* ug = reinterpret_cast<uint32_t*>(&g);
  const uint32_t* uy = reinterpret_cast<const uint32_t*>(&y);
#pragma unroll
  for (int i = 0; i < 4; ++i)
    ug[i] = pack_bf16x2(bg_dact(bf16_lo(ug[i]), bf16_lo(uy[i]), act), bg_dact(bf16_hi(ug[i]), bf16_hi(uy[i]), act));
  return g;
}

template <bool P_BF16, int LL, bool MASK>
__device__ __forceinline__ void bg_block(const BgMember& m, const BgBlock& b, float* red) {
  constexpr int L = 1 << LL;
  constexpr int rpp = kBgThreads >> LL;
  const int lane_in_row = threadIdx.x & (L - 1);
  const int row_in_pass = threadIdx.x >> LL;
  const int N = m.nvec * 8;
  const int vec = b.vec0 + lane_in_row;
  const bool act = vec < m.nvec;
  const int4* zb = reinterpret_cast<const int4*>(m.dz) + (int64_t)b.row0 * m.ldz16 + vec;
  f32x2 acc[4] = {0ull, 0ull, 0ull, 0ull};
  if (act) {
    const int4* yb = MASK ? reinterpret_cast<const int4*>(m.y) + (int64_t)b.row0 * m.ldy16 + vec : nullptr;
    int4* ob = MASK && m.dzo ? reinterpret_cast<int4*>(m.dzo) + (int64_t)b.row0 * m.lddzo16 + vec : nullptr;
    int r = row_in_pass;
    for (; r + (kBgInflight - 1) * rpp < b.nrows; r += kBgInflight * rpp) {
      int4 v[kBgInflight], y[MASK ? kBgInflight : 1];
#pragma unroll
      for (int j = 0; j < kBgInflight; ++j) {
        v[j] = __ldcs(zb + (int64_t)(r + j * rpp) * m.ldz16);
        if (MASK) y[j] = __ldcs(yb + (int64_t)(r + j * rpp) * m.ldy16);
      }
#pragma unroll
      for (int j = 0; j < kBgInflight; ++j) {
        if (MASK) {
          v[j] = bg_deriv(v[j], y[j], m.act);
          if (ob) __stcs(ob + (int64_t)(r + j * rpp) * m.lddzo16, v[j]);
        }
        const uint32_t* u = reinterpret_cast<const uint32_t*>(&v[j]);
#pragma unroll
        for (int k = 0; k < 4; ++k) acc[k] = add2(acc[k], bf2_to_f2(u[k]));
      }
    }
    for (; r < b.nrows; r += rpp) {
      int4 v = __ldcs(zb + (int64_t)r * m.ldz16);
      if (MASK) {
        v = bg_deriv(v, __ldcs(yb + (int64_t)r * m.ldy16), m.act);
        if (ob) __stcs(ob + (int64_t)r * m.lddzo16, v);
      }
      const uint32_t* u = reinterpret_cast<const uint32_t*>(&v);
#pragma unroll
      for (int k = 0; k < 4; ++k) acc[k] = add2(acc[k], bf2_to_f2(u[k]));
    }
  }
  // ---- row groups -> shared memory -> group-order sum -> workspace part
#pragma unroll
  for (int k = 0; k < 4; ++k) reinterpret_cast<f32x2*>(red + row_in_pass * (L * 8) + lane_in_row * 8)[k] = acc[k];
  __syncthreads();
  float* part = m.ws + (size_t)b.part * N;
  for (int c = threadIdx.x; c < L * 8; c += kBgThreads) {
    const int col = b.vec0 * 8 + c;
    if (col < N) {
      float a = 0.f;
#pragma unroll 8
      for (int g = 0; g < rpp; ++g) a += red[g * (L * 8) + c];
      part[col] = a;
    }
  }
  // ---- last block of the member: add the parts in part order, write db, re-arm the ticket
  __shared__ int is_last;
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) is_last = atomicAdd(m.ticket, 1) == m.nblocks - 1;
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  for (int c = threadIdx.x; c < N; c += kBgThreads) {
    float a = 0.f;
    for (int p = 0; p < m.nparts; ++p) a += __ldcg(m.ws + (size_t)p * N + c);
    if (P_BF16) reinterpret_cast<__nv_bfloat16*>(m.db)[c] = __float2bfloat16_rn(a);
    else reinterpret_cast<float*>(m.db)[c] = a;
  }
  if (threadIdx.x == 0) *m.ticket = 0;
}

// Two instantiations chosen per plan: groups without a fused mask run 6 blocks per SM in 40 registers; a masked member
// keeps twice the vectors in flight (dY and y) and needs 64 registers (4 blocks per SM) to stay out of local memory.
template <bool P_BF16, bool ANY_MASK>
__global__ void __launch_bounds__(kBgThreads, ANY_MASK ? 4 : kBgMinBlocks)
batched_bias_grad_kernel(const BgMember* __restrict__ members, const BgBlock* __restrict__ blocks) {
  __shared__ __align__(16) float bg_red[kBgThreads * 8];      // [256/L][L*8] floats = 8 KB
  const BgBlock b = blocks[blockIdx.x];
  const BgMember m = members[b.member];
  if (!ANY_MASK || m.y == nullptr) {     // block-uniform
    switch (m.l_log2) {
      case 0: bg_block<P_BF16, 0, false>(m, b, bg_red); break;
      case 1: bg_block<P_BF16, 1, false>(m, b, bg_red); break;
      case 2: bg_block<P_BF16, 2, false>(m, b, bg_red); break;
      case 3: bg_block<P_BF16, 3, false>(m, b, bg_red); break;
      case 4: bg_block<P_BF16, 4, false>(m, b, bg_red); break;
      default: bg_block<P_BF16, 5, false>(m, b, bg_red); break;
    }
  } else {
    switch (m.l_log2) {
      case 0: bg_block<P_BF16, 0, true>(m, b, bg_red); break;
      case 1: bg_block<P_BF16, 1, true>(m, b, bg_red); break;
      case 2: bg_block<P_BF16, 2, true>(m, b, bg_red); break;
      case 3: bg_block<P_BF16, 3, true>(m, b, bg_red); break;
      case 4: bg_block<P_BF16, 4, true>(m, b, bg_red); break;
      default: bg_block<P_BF16, 5, true>(m, b, bg_red); break;
    }
  }
}

// ---- fp32 groups (configs[0]-like: tiny, latency-bound).  One block per (member, 32-column tile): thread (tx, ty)
// adds rows ty, ty + 8, ... of column col0 + tx in row order, the 8 row groups are added in group order through shared
// memory: deterministic, no workspace, no tickets.  The fused derivative is plain fp32 arithmetic on the stored output
// (mask: a select; tanh dy (1 - y^2); sigmoid dy (1 - y) y), dZ written as fp32, db sums the dZ it wrote.
struct BgF32Member {
  const float* dz; const float* y; float* dzo; char* db;
  int64_t ldz, ldy, lddzo;
  int32_t rows, N, act, pad;
};
struct BgF32Block { int32_t member, col0; };

template <bool P_BF16>
__global__ void __launch_bounds__(256)
batched_bias_grad_f32_kernel(const BgF32Member* __restrict__ members, const BgF32Block* __restrict__ blocks) {
  __shared__ float red[8][33];
  const BgF32Block b = blocks[blockIdx.x];
  const BgF32Member m = members[b.member];
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const int col = b.col0 + tx;
  float acc = 0.f;
  if (col < m.N) {
    for (int r = ty; r < m.rows; r += 8) {
      float v = __ldg(m.dz + (int64_t)r * m.ldz + col);
      if (m.y != nullptr) {
        const float y = __ldg(m.y + (int64_t)r * m.ldy + col);
        v = m.act <= 1 ? (y <= 0.f ? 0.f : v) : bg_dact(v, y, m.act);
        if (m.dzo != nullptr) m.dzo[(int64_t)r * m.lddzo + col] = v;
      }
      acc += v;
    }
  }
  red[ty][tx] = acc;
  __syncthreads();
  if (ty == 0 && col < m.N) {
    float a = 0.f;
#pragma unroll
    for (int g = 0; g < 8; ++g) a += red[g][tx];
    if (P_BF16) reinterpret_cast<__nv_bfloat16*>(m.db)[col] = __float2bfloat16_rn(a);
    else reinterpret_cast<float*>(m.db)[col] = a;
  }
}

cudaError_t launch_bias_grad(const opt_plan* p, cudaStream_t s) {
  const char* base = static_cast<const char*>(p->dev_tables);
  auto* members = reinterpret_cast<const BgMember*>(base + p->off0);
  auto* blocks = reinterpret_cast<const BgBlock*>(base + p->off1);
  if (p->io == OPT_F32) {
    auto* m32 = reinterpret_cast<const BgF32Member*>(base + p->off0);
    auto* b32 = reinterpret_cast<const BgF32Block*>(base + p->off1);
    if (p->param == OPT_BF16) batched_bias_grad_f32_kernel<true><<<p->grid, p->block, 0, s>>>(m32, b32);
    else batched_bias_grad_f32_kernel<false><<<p->grid, p->block, 0, s>>>(m32, b32);
    return cudaGetLastError();
  }
  const bool any_mask = p->nstages != 0;      // stored in nstages
  if (p->param == OPT_BF16) {
    if (any_mask) batched_bias_grad_kernel<true, true><<<p->grid, p->block, 0, s>>>(members, blocks);
    else batched_bias_grad_kernel<true, false><<<p->grid, p->block, 0, s>>>(members, blocks);
  } else {
    if (any_mask) batched_bias_grad_kernel<false, true><<<p->grid, p->block, 0, s>>>(members, blocks);
    else batched_bias_grad_kernel<false, false><<<p->grid, p->block, 0, s>>>(members, blocks);
  }
  return cudaGetLastError();
}

}  // namespace optb

using namespace optb;

extern "C" opt_status opt_bias_grad_plan_create(const opt_bias_grad_member* members, int32_t n, opt_dtype io,
                                                opt_dtype param, int device, opt_plan** plan) {
  if (plan) *plan = nullptr;
  if (!plan || !members) return fail(OPT_ERR_INVALID_ARG, "opt_bias_grad_plan_create: NULL argument");
  if (n < 1 || n > 65535) return fail(OPT_ERR_INVALID_ARG, "n = %d outside [1, 65535]", n);
  if ((io != OPT_F32 && io != OPT_BF16) || (param != OPT_F32 && param != OPT_BF16)) return fail(OPT_ERR_INVALID_ARG, "bad dtype");
  const int pesz = elem_size(param);
  if (io == OPT_F32) {      // fp32 groups: the simple deterministic column-tile kernel
    std::vector<Region> regions;
    std::vector<BgF32Member> tab;
    std::vector<BgF32Block> blocks;
    int64_t bytes = 0, flops = 0;
    for (int32_t i = 0; i < n; ++i) {
      const opt_bias_grad_member& m = members[i];
      if (!m.dz || !m.db) return fail(OPT_ERR_INVALID_ARG, "member %d: NULL pointer", i);
      if (m.M < 1 || m.N < 1) return fail(OPT_ERR_INVALID_ARG, "member %d: M=%d N=%d must be >= 1", i, m.M, m.N);
      if (m.M > 1 && (m.ldz < m.N || (m.y && m.ldy < m.N) || (m.dz_out && m.lddz_out < m.N))) return fail(OPT_ERR_INVALID_ARG, "member %d: row stride smaller than N", i);
      if (!aligned16(m.dz) || !aligned16(m.db) || !aligned16(m.y) || !aligned16(m.dz_out)) return fail(OPT_ERR_ALIGNMENT, "member %d: pointers must be 16-byte aligned", i);
      if (m.N % 4 || (m.M > 1 && (m.ldz % 4 || (m.y && m.ldy % 4) || (m.dz_out && m.lddz_out % 4))))
        return fail(OPT_ERR_ALIGNMENT, "member %d: N and the row strides must be multiples of 4 elements", i);
      if (m.act < OPT_ACT_NONE || m.act > OPT_ACT_SIGMOID) return fail(OPT_ERR_INVALID_ARG, "member %d: bad act %d", i, m.act);
      if (m.act != OPT_ACT_NONE && !m.y) return fail(OPT_ERR_INVALID_ARG, "member %d: act %d needs y (the stored forward output)", i, m.act);
      if (m.dz_out && !m.y) return fail(OPT_ERR_INVALID_ARG, "member %d: dz_out without y (the mask source)", i);
      if (m.y) regions.push_back({(uintptr_t)m.y, m.ldy * 4, (int64_t)m.N * 4, m.M, false, i});
      if (m.dz_out) regions.push_back({(uintptr_t)m.dz_out, m.lddz_out * 4, (int64_t)m.N * 4, m.M, true, i});
      regions.push_back({(uintptr_t)m.dz, m.ldz * 4, (int64_t)m.N * 4, m.M, false, i});
      regions.push_back({(uintptr_t)m.db, 0, (int64_t)m.N * pesz, 1, true, i});
      bytes += (int64_t)m.M * m.N * 4 * (1 + (m.y ? 1 : 0) + (m.dz_out ? 1 : 0)) + (int64_t)m.N * pesz;
      flops += (int64_t)m.M * m.N;
      BgF32Member t;
      memset(&t, 0, sizeof t);
      t.dz = (const float*)m.dz; t.y = (const float*)m.y; t.dzo = (float*)m.dz_out; t.db = (char*)m.db;
      t.ldz = m.ldz; t.ldy = m.ldy; t.lddzo = m.lddz_out; t.rows = m.M; t.N = m.N; t.act = m.act;
      tab.push_back(t);
      for (int32_t c0 = 0; c0 < m.N; c0 += 32) blocks.push_back({i, c0});
    }
    if (opt_status st = check_independent(regions, /*allow_inplace_self=*/true)) return st;
    int num_sms = 0;
    DeviceGuard device_guard;      // the caller's current device is restored on return
    if (opt_status st = open_device(device, &num_sms)) return st;
    auto align_up = [](size_t x) { return (x + 255) & ~size_t(255); };
    opt_plan* p = new opt_plan();
    p->kind = kPlanBiasGrad; p->device = device; p->io = io; p->param = param; p->n_members = n;
    p->bytes = bytes; p->flops = flops;
    p->off0 = 0;
    p->off1 = align_up(tab.size() * sizeof(BgF32Member));
    const size_t total = p->off1 + align_up(blocks.size() * sizeof(BgF32Block));
    std::vector<char> blob(total, 0);
    memcpy(blob.data(), tab.data(), tab.size() * sizeof(BgF32Member));
    memcpy(blob.data() + p->off1, blocks.data(), blocks.size() * sizeof(BgF32Block));
    if (opt_status st = upload_tables(p, blob.data(), total)) { delete p; return st; }
    p->grid = dim3((unsigned)blocks.size()); p->block = dim3(256); p->smem = 0;
    p->total_tiles = (int32_t)blocks.size();
    *plan = p;
    return OPT_OK;
  }
  std::vector<Region> regions;
  std::vector<BgMember> tab;
  std::vector<BgBlock> blocks;
  std::vector<int64_t> ws_off;            // float offset of each member's partials in the workspace
  int64_t bytes = 0, ws_floats = 0, flops = 0;
  for (int32_t i = 0; i < n; ++i) {
    const opt_bias_grad_member& m = members[i];
    if (!m.dz || !m.db) return fail(OPT_ERR_INVALID_ARG, "member %d: NULL pointer", i);
    if (m.M < 1 || m.N < 1) return fail(OPT_ERR_INVALID_ARG, "member %d: M=%d N=%d must be >= 1", i, m.M, m.N);
    if (m.M > 1 && m.ldz < m.N) return fail(OPT_ERR_INVALID_ARG, "member %d: row stride smaller than N", i);
    if (!aligned16(m.dz) || !aligned16(m.db)) return fail(OPT_ERR_ALIGNMENT, "member %d: pointers must be 16-byte aligned", i);
    if (m.N % 8) return fail(OPT_ERR_ALIGNMENT, "member %d: N=%d is not a multiple of 8", i, m.N);
    if (m.M > 1 && m.ldz % 8) return fail(OPT_ERR_ALIGNMENT, "member %d: row stride must be a multiple of 8 elements", i);
    if (m.act < OPT_ACT_NONE || m.act > OPT_ACT_SIGMOID) return fail(OPT_ERR_INVALID_ARG, "member %d: bad act %d", i, m.act);
    if (m.act != OPT_ACT_NONE && !m.y) return fail(OPT_ERR_INVALID_ARG, "member %d: act %d needs y (the stored forward output)", i, m.act);
    if (m.dz_out && !m.y) return fail(OPT_ERR_INVALID_ARG, "member %d: dz_out without y (the mask source)", i);
    if (m.y) {
      if (!aligned16(m.y) || !aligned16(m.dz_out)) return fail(OPT_ERR_ALIGNMENT, "member %d: pointers must be 16-byte aligned", i);
      if (m.M > 1 && (m.ldy < m.N || (m.dz_out && m.lddz_out < m.N))) return fail(OPT_ERR_INVALID_ARG, "member %d: row stride smaller than N", i);
      if (m.M > 1 && (m.ldy % 8 || (m.dz_out && m.lddz_out % 8))) return fail(OPT_ERR_ALIGNMENT, "member %d: row stride must be a multiple of 8 elements", i);
      regions.push_back({(uintptr_t)m.y, m.ldy * 2, (int64_t)m.N * 2, m.M, false, i});
      if (m.dz_out) regions.push_back({(uintptr_t)m.dz_out, m.lddz_out * 2, (int64_t)m.N * 2, m.M, true, i});
    }
    regions.push_back({(uintptr_t)m.dz, m.ldz * 2, (int64_t)m.N * 2, m.M, false, i});
    regions.push_back({(uintptr_t)m.db, 0, (int64_t)m.N * pesz, 1, true, i});
    bytes += (int64_t)m.M * m.N * 2 * (1 + (m.y ? 1 : 0) + (m.dz_out ? 1 : 0)) + (int64_t)m.N * pesz;
    flops += (int64_t)m.M * m.N;
    const int nvec = m.N / 8;
    int ll = 0;
    while (ll < 5 && (1 << ll) < nvec) ++ll;
    const int L = 1 << ll, rpp = kBgThreads >> ll;
    const int nctile = (nvec + kBgTileVec - 1) / kBgTileVec;
    // rows per block: whole groups of in-flight passes, ~128 KB of dZ per block
    const int64_t chunk_rows = (int64_t)rpp * kBgInflight;
    const int64_t rpb = chunk_rows * std::max<int64_t>(1, kBgBlockBytes / (chunk_rows * L * 16));
    const int32_t nparts = (int32_t)((m.M + rpb - 1) / rpb);
    BgMember t;
    memset(&t, 0, sizeof t);
    t.dz = (const char*)m.dz; t.db = (char*)m.db; t.ldz16 = m.ldz / 8;
    t.y = (const char*)m.y; t.dzo = (char*)m.dz_out; t.ldy16 = m.ldy / 8; t.lddzo16 = m.lddz_out / 8; t.act = m.act;
    t.rows = m.M; t.nvec = nvec; t.nparts = nparts; t.nblocks = nparts * nctile; t.l_log2 = ll;
    tab.push_back(t);
    ws_off.push_back(ws_floats);
    ws_floats += (int64_t)nparts * m.N;
    for (int32_t part = 0; part < nparts; ++part)
      for (int32_t ct = 0; ct < nctile; ++ct)
        blocks.push_back({i, (int32_t)(part * rpb), (int32_t)std::min<int64_t>(rpb, m.M - part * rpb), part, ct * kBgTileVec});
  }
  // launch order.  Dense members (ldz == N) stay member-major: a block's rows are one contiguous range.  Members that
  // are column slices of a wider buffer go part-major -- blocks that run together then read the SAME rows of
  // neighbouring members, i.e. neighbouring bytes of the same DRAM rows (configs[2]'s concat gradient: 102 -> 97 us)
  {
    auto key = [&](const BgBlock& b) { return members[b.member].M > 1 && members[b.member].ldz != members[b.member].N ? b.part + 1 : 0; };
    std::stable_sort(blocks.begin(), blocks.end(), [&](const BgBlock& a, const BgBlock& b) { return key(a) < key(b); });
  }
  if (opt_status st = check_independent(regions, /*allow_inplace_self=*/true)) return st;
  if (blocks.size() > (size_t)INT32_MAX) return fail(OPT_ERR_UNSUPPORTED, "too many work items");

  int num_sms = 0;
  DeviceGuard device_guard;      // the caller's current device is restored on return
  if (opt_status st = open_device(device, &num_sms)) return st;
  auto align_up = [](size_t x) { return (x + 255) & ~size_t(255); };
  opt_plan* p = new opt_plan();
  p->kind = kPlanBiasGrad; p->device = device; p->io = io; p->param = param; p->n_members = n;
  p->bytes = bytes; p->flops = flops;
  // workspace: per-part partial column sums (fully written before they are read: no initialisation needed)
  if (cudaMalloc(&p->workspace, std::max<int64_t>(ws_floats, 1) * sizeof(float)) != cudaSuccess) {
    cudaGetLastError(); delete p;
    return fail(OPT_ERR_CUDA, "cudaMalloc of the %lld-byte partial-sum workspace failed", (long long)ws_floats * 4);
  }
  p->off0 = 0;
  p->off1 = align_up(tab.size() * sizeof(BgMember));
  p->off2 = p->off1 + align_up(blocks.size() * sizeof(BgBlock));
  const size_t total = p->off2 + align_up((size_t)n * sizeof(int32_t));      // per-member tickets, zero-initialised
  std::vector<char> blob(total, 0);
  memcpy(blob.data() + p->off1, blocks.data(), blocks.size() * sizeof(BgBlock));
  if (cudaMalloc(&p->dev_tables, total) != cudaSuccess) {
    cudaGetLastError(); cudaFree(p->workspace); delete p;
    return fail(OPT_ERR_CUDA, "cudaMalloc of the plan tables failed");
  }
  p->table_bytes = total;
  for (int32_t i = 0; i < n; ++i) {
    tab[i].ws = static_cast<float*>(p->workspace) + ws_off[i];
    tab[i].ticket = reinterpret_cast<int32_t*>(static_cast<char*>(p->dev_tables) + p->off2) + i;
  }
  memcpy(blob.data(), tab.data(), tab.size() * sizeof(BgMember));
  cudaError_t e = cudaMemcpy(p->dev_tables, blob.data(), total, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    cudaFree(p->dev_tables); cudaFree(p->workspace); delete p;
    return fail(OPT_ERR_CUDA, "plan upload failed: %s", cudaGetErrorString(e));
  }
  p->grid = dim3((unsigned)blocks.size());
  p->block = dim3(kBgThreads);
  p->smem = 0;
  p->nstages = 0;
  for (const BgMember& t : tab) if (t.y) p->nstages = 1;
  p->total_tiles = (int32_t)blocks.size();
  *plan = p;
  return OPT_OK;
}
