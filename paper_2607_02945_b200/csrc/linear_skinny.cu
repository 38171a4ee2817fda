// Grouped Linear for SKINNY members: huge M, tiny K and N (decompose_mm_pass: "decomposing the
// multiplication into pointwise operations followed by reductions along the K dimension ... particularly effective
// when the matrix multiplication involves a very large M dimension and a small K dimension"; the paper's shapes are
// [18583840, 8] x [8, 8] and [25247936, 4] x [4, 2]).  SURVEY.md 8(f) rank 4.
//
// Such a member is a streaming problem -- (K + N) * 2 bytes per row, 2 K N flops per row -- and a 128 x N x 64 tcgen05
// tile would spend its time on zero-filled operands (measured: 3.8x slower).  The right tensor-core shape for it is
// the warp-level mma.sync m16n8k8 / m16n8k16: a warp multiplies 16 rows at a time, and the fragment layouts make
// every global access a 4-byte word per lane with the lanes of a row group contiguous (thread (g, t) of the warp
// owns x[row g][2t..2t+1] and y[row g][2t..2t+1]): no shared memory, ~1 instruction per row per warp, 64 registers.  W ([N,K], a few hundred bytes) and the
// bias live in registers as B / C fragments; tails (K = 4 < 8, N < 8) are zero fragments and masked stores.
// One launch for the whole group; a block walks 4096 consecutive rows of one member in chunks of 512.  Measured on
// the paper's group (1.83 GB): occupancy beats per-thread unrolling and register double-buffering (16 loads in flight
// per lane at 2 blocks / SM: 500 us; 8 loads at 4 - 6 blocks / SM: 328 us = 85 % of the HBM copy peak).  fp32 accumulation, one
// rounding: the semantics of opt_linear_member.
//
// Routing (opt_linear_plan_create): a bf16 group takes this path when EVERY member has K in {4, 8, 16},
// N in {2, 4, 8, 16}, K * N <= 128 and untransposed operands.  Row strides then only need to be even (4-byte words),
// which admits the paper's dense [M, 4] and [M, 2] tensors.
#include <algorithm>
#include <type_traits>

#include "common.h"

namespace optb {

constexpr int kSkThreads = 256;
constexpr int kSkMinBlocks = 4;    // occupancy is what hides the latency here: 4 x 256 threads per SM at <= 64 registers
constexpr int kSkUnroll = 4;                   // 16-row MMA groups per warp and chunk: 8 warps x 4 x 16 = 512 rows
constexpr int kSkChunkRows = (kSkThreads / 32) * kSkUnroll * 16;
constexpr int kSkChunks = 8;                           // chunks a block walks (4096 rows)
constexpr int kSkRowsPerBlock = kSkChunkRows * kSkChunks;

struct alignas(16) SkMember {
  const uint16_t* x; const uint16_t* w; const uint16_t* bias; uint16_t* y;
  int64_t ldx, ldw, ldy;
  int32_t M, N, K, act;        // the shape the kernel walks (packed members: M / 2 rows of 2 K, 2 N)
  int32_t pack, n_real;        // pack = 2: a dense [M,4] x [4,N] member seen as [M/2, 8] x [8, 2N] with W block-diagonal
  int32_t pad[2];
};
static_assert(sizeof(SkMember) == 96, "SkMember layout");

__device__ __forceinline__ void mma_16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void mma_1688(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t b0) {
  asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a0), "r"(a1), "r"(b0));
}

template <int K, int N>
__device__ __forceinline__ void sk_rows(const SkMember& m, int row0) {
  constexpr int NF = N == 16 ? 2 : 1;                  // n8 fragments
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int g = lane >> 2, t = lane & 3;               // fragment coordinates: row group / column pair
  const bool kin = 2 * t < K;                          // K = 4: only t < 2 holds real k
  // B fragments (W[n][k], k pairs contiguous) and C = bias, once per warp
  uint32_t b[NF][K == 16 ? 2 : 1];
  float bias[NF][2];
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    const int n = 8 * f + g;
    const bool nin = n < N;
    const int c0 = 8 * f + 2 * t;
    if (K == 8 && m.pack == 2) {
      // two data rows per MMA row: k 0..3 belong to the first, k 4..7 to the second; output columns [0, n_real) come
      // from the first, [n_real, 2 n_real) from the second -> B is W twice on the diagonal, zero elsewhere
      const int half = n >= m.n_real, nr = n - half * m.n_real;
      b[f][0] = (nin && (t >> 1) == half) ? __ldg(reinterpret_cast<const uint32_t*>(m.w + (int64_t)nr * m.ldw + 2 * (t & 1))) : 0u;
      const int cr = c0 % m.n_real;                    // n_real is even: the pair stays inside one copy
      bias[f][0] = (m.bias && c0 < N) ? __uint_as_float((uint32_t)__ldg(m.bias + cr) << 16) : 0.f;
      bias[f][1] = (m.bias && c0 + 1 < N) ? __uint_as_float((uint32_t)__ldg(m.bias + cr + 1) << 16) : 0.f;
      continue;
    }
    b[f][0] = (nin && kin) ? __ldg(reinterpret_cast<const uint32_t*>(m.w + (int64_t)n * m.ldw + 2 * t)) : 0u;
    if (K == 16) b[f][1] = nin ? __ldg(reinterpret_cast<const uint32_t*>(m.w + (int64_t)n * m.ldw + 2 * t + 8)) : 0u;
    bias[f][0] = (m.bias && c0 < N) ? __uint_as_float((uint32_t)__ldg(m.bias + c0) << 16) : 0.f;
    bias[f][1] = (m.bias && c0 + 1 < N) ? __uint_as_float((uint32_t)__ldg(m.bias + c0 + 1) << 16) : 0.f;
  }
  // one chunk = kSkUnroll 16-row groups per warp.  FULL: every row of the chunk exists (no row predicates);
  // NOACT: no activation (both block-uniform).  Row pointers advance by a constant stride of 8 rows.
  auto chunk = [&](int base, auto full_tag, auto noact_tag) {
    constexpr bool FULL = decltype(full_tag)::value, NOACT = decltype(noact_tag)::value;
    constexpr int AR = K == 16 ? 4 : 2;
    const int64_t sx8 = 4 * m.ldx, sy8 = 4 * m.ldy;            // 8 rows, in 4-byte words
    const uint32_t* px = reinterpret_cast<const uint32_t*>(m.x + (int64_t)(base + g) * m.ldx) + t;
    uint32_t* py = reinterpret_cast<uint32_t*>(m.y + (int64_t)(base + g) * m.ldy) + t;
    uint32_t a[kSkUnroll][AR];
#pragma unroll
    for (int u = 0; u < kSkUnroll; ++u) {                      // all loads first: independent, streaming
      const int rlo = base + u * 16 + g, rhi = rlo + 8;
      const uint32_t* plo = px + (2 * u) * sx8;
      const uint32_t* phi = plo + sx8;
      const bool vlo = FULL || rlo < m.M, vhi = FULL || rhi < m.M;
      a[u][0] = (vlo && kin) ? __ldcs(plo) : 0u;
      a[u][1] = (vhi && kin) ? __ldcs(phi) : 0u;
      if (K == 16) {
        a[u][AR - 2] = vlo ? __ldcs(plo + 4) : 0u;
        a[u][AR - 1] = vhi ? __ldcs(phi + 4) : 0u;
      }
    }
#pragma unroll
    for (int u = 0; u < kSkUnroll; ++u) {
      const int rlo = base + u * 16 + g, rhi = rlo + 8;
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        float c[4] = {bias[f][0], bias[f][1], bias[f][0], bias[f][1]};
        if (K == 16) {
          const uint32_t aa[4] = {a[u][0], a[u][1], a[u][AR - 2], a[u][AR - 1]};
          mma_16816(c, aa, b[f][0], b[f][K == 16 ? 1 : 0]);
        } else {
          mma_1688(c, a[u][0], a[u][1], b[f][0]);
        }
        if (8 * f + 2 * t < N) {                       // N is even: a column pair is valid or not as a whole
          const uint32_t lo = NOACT ? pack_bf16x2(c[0], c[1]) : pack_bf16x2(act_f32<true>(c[0], m.act), act_f32<true>(c[1], m.act));
          const uint32_t hi = NOACT ? pack_bf16x2(c[2], c[3]) : pack_bf16x2(act_f32<true>(c[2], m.act), act_f32<true>(c[3], m.act));
          if (FULL || rlo < m.M) __stcs(py + (2 * u) * sy8 + 4 * f, lo);
          if (FULL || rhi < m.M) __stcs(py + (2 * u + 1) * sy8 + 4 * f, hi);
        }
      }
    }
  };
  using T = std::true_type;
  using F = std::false_type;
  const int wofs = warp * (kSkUnroll * 16);
  for (int ch = 0, start = row0; ch < kSkChunks && start < m.M; ++ch, start += kSkChunkRows) {
    const bool full = start + kSkChunkRows <= m.M;
    if (m.act == OPT_ACT_NONE) { if (full) chunk(start + wofs, T{}, T{}); else chunk(start + wofs, F{}, T{}); }
    else { if (full) chunk(start + wofs, T{}, F{}); else chunk(start + wofs, F{}, F{}); }
  }
}

__global__ void __launch_bounds__(kSkThreads, kSkMinBlocks)
grouped_skinny_linear_kernel(const SkMember* __restrict__ members, const int2* __restrict__ blocks) {
  const int2 b = __ldg(blocks + blockIdx.x);
  const SkMember m = members[b.x];
#define SK_CASE(KK, NN) case (KK) * 32 + (NN): sk_rows<KK, NN>(m, b.y); break;
  switch (m.K * 32 + m.N) {
    SK_CASE(4, 2) SK_CASE(4, 4) SK_CASE(4, 8) SK_CASE(4, 16)
    SK_CASE(8, 2) SK_CASE(8, 4) SK_CASE(8, 8) SK_CASE(8, 16)
    SK_CASE(16, 2) SK_CASE(16, 4) SK_CASE(16, 8)
    default: break;
  }
#undef SK_CASE
}

bool skinny_linear_member(const opt_linear_member& m) {
  const bool k_ok = m.K == 4 || m.K == 8 || m.K == 16, n_ok = m.N == 2 || m.N == 4 || m.N == 8 || m.N == 16;
  return m.layout == 0 && k_ok && n_ok && m.K * m.N <= 128;
}

// members validated by opt_linear_plan_create (skinny rules); fills the plan's tables
opt_status plan_skinny_linear(const opt_linear_member* members, int32_t n, opt_plan* p) {
  auto align_up = [](size_t x) { return (x + 255) & ~size_t(255); };
  std::vector<SkMember> tab;
  std::vector<int2> blocks;
  auto add = [&](const SkMember& t) {
    tab.push_back(t);
    for (int64_t r0 = 0; r0 < t.M; r0 += kSkRowsPerBlock) blocks.push_back(make_int2((int)tab.size() - 1, (int)r0));
  };
  for (int32_t i = 0; i < n; ++i) {
    const opt_linear_member& m = members[i];
    SkMember t;
    memset(&t, 0, sizeof t);
    t.x = static_cast<const uint16_t*>(m.x); t.w = static_cast<const uint16_t*>(m.w);
    t.bias = static_cast<const uint16_t*>(m.bias); t.y = static_cast<uint16_t*>(m.y);
    t.ldx = m.ldx; t.ldw = m.ldw; t.ldy = m.ldy; t.M = m.M; t.N = m.N; t.K = m.K; t.act = m.act;
    t.pack = 1; t.n_real = m.N;
    if (m.K == 4 && m.N <= 4 && m.ldx == 4 && m.ldy == m.N && m.M >= 2) {
      // dense [M,4] x [4,N]: two data rows per MMA row (twice the bytes per access); an odd last row goes unpacked
      SkMember v = t;
      v.M = m.M / 2; v.K = 8; v.N = 2 * m.N; v.ldx = 8; v.ldy = 2 * m.N; v.pack = 2;
      add(v);
      if (m.M & 1) {
        t.x += (int64_t)(m.M - 1) * m.ldx; t.y += (int64_t)(m.M - 1) * m.ldy; t.M = 1;
        add(t);
      }
    } else {
      add(t);
    }
    if (blocks.size() > (size_t)INT32_MAX) return fail(OPT_ERR_UNSUPPORTED, "too many blocks");
  }
  p->kind = kPlanLinearSkinny;
  p->off0 = 0;
  p->off1 = align_up(tab.size() * sizeof(SkMember));
  const size_t total = p->off1 + align_up(blocks.size() * sizeof(int2));
  std::vector<char> blob(total, 0);
  memcpy(blob.data(), tab.data(), tab.size() * sizeof(SkMember));
  memcpy(blob.data() + p->off1, blocks.data(), blocks.size() * sizeof(int2));
  if (opt_status st = upload_tables(p, blob.data(), total)) return st;
  p->grid = dim3((unsigned)blocks.size()); p->block = dim3(kSkThreads); p->smem = 0;
  p->total_tiles = (int32_t)blocks.size();
  return OPT_OK;
}

cudaError_t launch_linear_skinny(const opt_plan* p, cudaStream_t s) {
  char* base = static_cast<char*>(p->dev_tables);
  grouped_skinny_linear_kernel<<<p->grid, p->block, 0, s>>>(reinterpret_cast<const SkMember*>(base + p->off0),
                                                            reinterpret_cast<const int2*>(base + p->off1));
  return cudaGetLastError();
}

}  // namespace optb
