// batched_layernorm: N independent LayerNorms (different D_i, rows_i, strides,
// gamma/beta) in one launch -- batch_layernorm.
//
//   mu = mean(x_r); v = mean((x_r - mu)^2); y_r = (x_r - mu) * rsqrt(v + eps) * gamma + beta
//
// Design (HBM-bound):
//   * a row is owned by L = 2^k lanes of one warp (L chosen per member so that
//     L * VPL 16-byte vectors cover D with the least waste): D=32 packs 16 rows
//     into a warp, D>=256 uses the whole warp.  Each lane keeps VPL vectors of
//     the row in registers: x is read from HBM exactly once.
//   * fp32 statistics, two passes over the registers (mean, then centred sum of
//     squares), width-L shuffle-xor reductions.
//   * the next rows' vectors are prefetched before the current rows' math; a
//     thread works on RU rows at a time (RU x VPL ~ 4 vectors) so that enough
//     bytes are in flight per SM.
//   * bf16 path: the kernel is close to ISSUE-bound (ncu: sm throughput 66-81 %
//     for the first version), so the arithmetic runs on packed fp32 pairs
//     (add/mul/fma.rn.f32x2) and gamma/beta are staged once per block as fp32 in
//     shared memory (a block never leaves its member).
//   * a per-block table (member, first row, row count) maps blocks to members.
#include <algorithm>

#include "common.h"

namespace optb {

struct LnMember {
  const char* x;
  char* y;
  const char* gamma;
  const char* beta;
  int64_t ldx16, ldy16;    // row stride in 16-byte vectors
  int32_t rows, nvec;      // nvec = D / elements-per-vector
  float eps, inv_D;
  int32_t l_log2, vpl;     // lanes per row (log2), vectors per lane
};
struct LnBlock { int32_t member, row0, nrows; };

constexpr int kLnThreads = 256;
constexpr int kLnMaxVpl = 8;

template <bool BF16>
struct LnVec {
  static constexpr int E = BF16 ? 8 : 4;
  static __device__ __forceinline__ void unpack(const int4& v, float (&f)[E]) {
    if (BF16) {
      const uint32_t* u = reinterpret_cast<const uint32_t*>(&v);
#pragma unroll
      for (int i = 0; i < 4; ++i) { f[2 * i] = bf16_lo(u[i]); f[2 * i + 1] = bf16_hi(u[i]); }
    } else {
      const float* p = reinterpret_cast<const float*>(&v);
#pragma unroll
      for (int i = 0; i < 4; ++i) f[i] = p[i];
    }
  }
  static __device__ __forceinline__ int4 pack(const float (&f)[E]) {
    int4 v;
    if (BF16) {
      uint32_t* u = reinterpret_cast<uint32_t*>(&v);
#pragma unroll
      for (int i = 0; i < 4; ++i) u[i] = pack_bf16x2(f[2 * i], f[2 * i + 1]);
    } else {
      float* p = reinterpret_cast<float*>(&v);
#pragma unroll
      for (int i = 0; i < 4; ++i) p[i] = f[i];
    }
    return v;
  }
};

// gamma/beta vector j of a member (parameters may be bf16 or fp32, independent of io)
template <bool IO_BF16, bool P_BF16>
__device__ __forceinline__ void ln_load_param(const char* base, int vec, float dflt, float (&out)[IO_BF16 ? 8 : 4]) {
  constexpr int E = IO_BF16 ? 8 : 4;
  if (base == nullptr) {
#pragma unroll
    for (int i = 0; i < E; ++i) out[i] = dflt;
    return;
  }
  if (P_BF16) {                       // E bf16 values = E*2 bytes
    if (E == 8) {
      int4 v = __ldg(reinterpret_cast<const int4*>(base) + vec);
      const uint32_t* u = reinterpret_cast<const uint32_t*>(&v);
#pragma unroll
      for (int i = 0; i < 4; ++i) { out[2 * i] = bf16_lo(u[i]); out[2 * i + 1] = bf16_hi(u[i]); }
    } else {
      int2 v = __ldg(reinterpret_cast<const int2*>(base) + vec);
      const uint32_t* u = reinterpret_cast<const uint32_t*>(&v);
#pragma unroll
      for (int i = 0; i < 2; ++i) { out[2 * i] = bf16_lo(u[i]); out[2 * i + 1] = bf16_hi(u[i]); }
    }
  } else {                            // E fp32 values
#pragma unroll
    for (int i = 0; i < E / 4; ++i) {
      float4 v = __ldg(reinterpret_cast<const float4*>(base) + vec * (E / 4) + i);
      out[4 * i] = v.x; out[4 * i + 1] = v.y; out[4 * i + 2] = v.z; out[4 * i + 3] = v.w;
    }
  }
}

template <bool IO_BF16, bool P_BF16, int VPL>
__device__ __forceinline__ void ln_block(const LnMember& m, int row0, int nrows) {
  using VT = LnVec<IO_BF16>;
  constexpr int E = VT::E;
  const int L = 1 << m.l_log2;
  const int lane_in_row = threadIdx.x & (L - 1);
  const int row_in_pass = threadIdx.x >> m.l_log2;
  const int rows_per_pass = kLnThreads >> m.l_log2;
  const int npass = (nrows + rows_per_pass - 1) / rows_per_pass;
  const int4* xb = reinterpret_cast<const int4*>(m.x);
  int4* yb = reinterpret_cast<int4*>(m.y);

  bool act[VPL];
#pragma unroll
  for (int i = 0; i < VPL; ++i) act[i] = lane_in_row + i * L < m.nvec;

  constexpr bool kPrefetch = VPL <= 3;            // wider rows already keep >= 4 loads in flight per lane
  int4 cur[VPL], nxt[kPrefetch ? VPL : 1];
  auto load_row = [&](int pass, int4 (&dst)[VPL]) {
    const int r = pass * rows_per_pass + row_in_pass;
    const bool ok = pass < npass && r < nrows;
    const int4* p = xb + (int64_t)(row0 + r) * m.ldx16 + lane_in_row;
#pragma unroll
    for (int i = 0; i < VPL; ++i) dst[i] = (ok && act[i]) ? __ldcs(p + i * L) : make_int4(0, 0, 0, 0);
  };
  load_row(0, cur);
  for (int pass = 0; pass < npass; ++pass) {
    if (kPrefetch) load_row(pass + 1, *reinterpret_cast<int4(*)[VPL]>(&nxt[0]));   // next row in flight during this row's math
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < VPL; ++i) {
      float f[E];
      VT::unpack(cur[i], f);
#pragma unroll
      for (int e = 0; e < E; ++e) s += f[e];       // inactive vectors are zeros
    }
    for (int o = L >> 1; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    const float mu = s * m.inv_D;
    float q = 0.f;
#pragma unroll
    for (int i = 0; i < VPL; ++i) {
      if (act[i]) {
        float f[E];
        VT::unpack(cur[i], f);
#pragma unroll
        for (int e = 0; e < E; ++e) { const float d = f[e] - mu; q = fmaf(d, d, q); }
      }
    }
    for (int o = L >> 1; o > 0; o >>= 1) q += __shfl_xor_sync(0xffffffffu, q, o);
    const float rstd = rsqrtf(q * m.inv_D + m.eps);
    const int r = pass * rows_per_pass + row_in_pass;
    if (r < nrows) {
      int4* yp = yb + (int64_t)(row0 + r) * m.ldy16 + lane_in_row;
#pragma unroll
      for (int i = 0; i < VPL; ++i) {
        if (act[i]) {
          float f[E], g[E], b[E];
          VT::unpack(cur[i], f);
          ln_load_param<IO_BF16, P_BF16>(m.gamma, lane_in_row + i * L, 1.f, g);   // L1-resident
          ln_load_param<IO_BF16, P_BF16>(m.beta, lane_in_row + i * L, 0.f, b);
#pragma unroll
          for (int e = 0; e < E; ++e) f[e] = fmaf((f[e] - mu) * rstd, g[e], b[e]);
          __stcs(yp + i * L, VT::pack(f));
        }
      }
    }
    if (kPrefetch) {
#pragma unroll
      for (int i = 0; i < VPL; ++i) cur[i] = nxt[kPrefetch ? i : 0];
    } else {
      load_row(pass + 1, cur);
    }
  }
}

// ---- packed fp32 pairs (sm_100 add/mul/fma.rn.f32x2) -------------------------
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ float sum2(f32x2 v) { float lo, hi; asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); return lo + hi; }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ f32x2 bf2_to_f2(uint32_t u) { return pk2(bf16_lo(u), bf16_hi(u)); }
__device__ __forceinline__ uint32_t f2_to_bf2(f32x2 v) {
  float lo, hi;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
  return pack_bf16x2(lo, hi);
}

constexpr int kLnMaxD = 2048;        // gamma/beta staging: 2 x 8 KB of shared memory

// bf16 in/out.  sg/sb: the member's gamma/beta as fp32 in shared memory.
template <int VPL, int RU>
__device__ __forceinline__ void ln_rows_bf16(const LnMember& m, int row0, int nrows, const float* sg, const float* sb) {
  const int L = 1 << m.l_log2;
  const int lane_in_row = threadIdx.x & (L - 1);
  const int row_in_pass = threadIdx.x >> m.l_log2;
  const int rpp = kLnThreads >> m.l_log2;              // rows per pass of the block
  const int niter = (nrows + rpp * RU - 1) / (rpp * RU);
  const int4* xb = reinterpret_cast<const int4*>(m.x);
  int4* yb = reinterpret_cast<int4*>(m.y);

  bool act[VPL];
#pragma unroll
  for (int i = 0; i < VPL; ++i) act[i] = lane_in_row + i * L < m.nvec;

  int4 nxt[RU][VPL];
  auto load = [&](int it, int4 (&dst)[RU][VPL]) {
#pragma unroll
    for (int u = 0; u < RU; ++u) {
      const int r = (it * RU + u) * rpp + row_in_pass;
      const int4* p = xb + (int64_t)(row0 + r) * m.ldx16 + lane_in_row;
#pragma unroll
      for (int i = 0; i < VPL; ++i) dst[u][i] = (r < nrows && act[i]) ? __ldcs(p + i * L) : make_int4(0, 0, 0, 0);
    }
  };
  load(0, nxt);
  for (int it = 0; it < niter; ++it) {
    f32x2 x[RU][VPL][4];
    float s[RU], q[RU];
#pragma unroll
    for (int u = 0; u < RU; ++u) {
      f32x2 acc = 0ull;
#pragma unroll
      for (int i = 0; i < VPL; ++i) {
        const uint32_t* w = reinterpret_cast<const uint32_t*>(&nxt[u][i]);
#pragma unroll
        for (int k = 0; k < 4; ++k) { x[u][i][k] = bf2_to_f2(w[k]); acc = add2(acc, x[u][i][k]); }   // inactive vectors are zeros
      }
      s[u] = sum2(acc);
    }
    load(it + 1, nxt);                                  // next rows in flight during this iteration's math
    for (int o = L >> 1; o > 0; o >>= 1) {
#pragma unroll
      for (int u = 0; u < RU; ++u) s[u] += __shfl_xor_sync(0xffffffffu, s[u], o);
    }
#pragma unroll
    for (int u = 0; u < RU; ++u) {
      const float nmu = -s[u] * m.inv_D;
      const f32x2 nmu2 = pk2(nmu, nmu);
      f32x2 acc = 0ull;
#pragma unroll
      for (int i = 0; i < VPL; ++i) {
        if (act[i]) {
#pragma unroll
          for (int k = 0; k < 4; ++k) { x[u][i][k] = add2(x[u][i][k], nmu2); acc = fma2(x[u][i][k], x[u][i][k], acc); }
        }
      }
      q[u] = sum2(acc);
    }
    for (int o = L >> 1; o > 0; o >>= 1) {
#pragma unroll
      for (int u = 0; u < RU; ++u) q[u] += __shfl_xor_sync(0xffffffffu, q[u], o);
    }
#pragma unroll
    for (int u = 0; u < RU; ++u) {
      const float rstd = rsqrtf(q[u] * m.inv_D + m.eps);
      const f32x2 rstd2 = pk2(rstd, rstd);
      const int r = (it * RU + u) * rpp + row_in_pass;
      if (r < nrows) {
        int4* yp = yb + (int64_t)(row0 + r) * m.ldy16 + lane_in_row;
#pragma unroll
        for (int i = 0; i < VPL; ++i) {
          if (act[i]) {
            const int vec = lane_in_row + i * L;
            const ulonglong2 g0 = *reinterpret_cast<const ulonglong2*>(sg + vec * 8);
            const ulonglong2 g1 = *reinterpret_cast<const ulonglong2*>(sg + vec * 8 + 4);
            const ulonglong2 b0 = *reinterpret_cast<const ulonglong2*>(sb + vec * 8);
            const ulonglong2 b1 = *reinterpret_cast<const ulonglong2*>(sb + vec * 8 + 4);
            int4 o;
            o.x = (int)f2_to_bf2(fma2(mul2(x[u][i][0], rstd2), g0.x, b0.x));
            o.y = (int)f2_to_bf2(fma2(mul2(x[u][i][1], rstd2), g0.y, b0.y));
            o.z = (int)f2_to_bf2(fma2(mul2(x[u][i][2], rstd2), g1.x, b1.x));
            o.w = (int)f2_to_bf2(fma2(mul2(x[u][i][3], rstd2), g1.y, b1.y));
            __stcs(yp + i * L, o);
          }
        }
      }
    }
  }
}

template <bool P_BF16>
__global__ void __launch_bounds__(kLnThreads, 3)
batched_layernorm_bf16_kernel(const LnMember* __restrict__ members, const LnBlock* __restrict__ blocks) {
  __shared__ __align__(16) float sg[kLnMaxD];
  __shared__ __align__(16) float sb[kLnMaxD];
  const LnBlock b = blocks[blockIdx.x];
  const LnMember m = members[b.member];
  for (int v = threadIdx.x; v < m.nvec; v += kLnThreads) {     // gamma/beta -> fp32, once per block
    float g[8], bt[8];
    ln_load_param<true, P_BF16>(m.gamma, v, 1.f, g);
    ln_load_param<true, P_BF16>(m.beta, v, 0.f, bt);
#pragma unroll
    for (int e = 0; e < 8; ++e) { sg[v * 8 + e] = g[e]; sb[v * 8 + e] = bt[e]; }
  }
  __syncthreads();
  switch (m.vpl) {   // block-uniform; RU rows at a time so that RU x VPL ~ 4 vectors are in flight per thread
    case 1: ln_rows_bf16<1, 4>(m, b.row0, b.nrows, sg, sb); break;
    case 2: ln_rows_bf16<2, 2>(m, b.row0, b.nrows, sg, sb); break;
    case 3: ln_rows_bf16<3, 1>(m, b.row0, b.nrows, sg, sb); break;
    case 4: ln_rows_bf16<4, 1>(m, b.row0, b.nrows, sg, sb); break;
    // D > 1024: the unpacked row would not fit the register budget; the generic path re-unpacks per pass
    case 5: ln_block<true, P_BF16, 5>(m, b.row0, b.nrows); break;
    case 6: ln_block<true, P_BF16, 6>(m, b.row0, b.nrows); break;
    case 7: ln_block<true, P_BF16, 7>(m, b.row0, b.nrows); break;
    default: ln_block<true, P_BF16, 8>(m, b.row0, b.nrows); break;
  }
}

template <bool IO_BF16, bool P_BF16>
__global__ void __launch_bounds__(kLnThreads, 4)
batched_layernorm_kernel(const LnMember* __restrict__ members, const LnBlock* __restrict__ blocks) {
  const LnBlock b = blocks[blockIdx.x];
  const LnMember m = members[b.member];
  switch (m.vpl) {   // block-uniform
    case 1: ln_block<IO_BF16, P_BF16, 1>(m, b.row0, b.nrows); break;
    case 2: ln_block<IO_BF16, P_BF16, 2>(m, b.row0, b.nrows); break;
    case 3: ln_block<IO_BF16, P_BF16, 3>(m, b.row0, b.nrows); break;
    case 4: ln_block<IO_BF16, P_BF16, 4>(m, b.row0, b.nrows); break;
    case 5: ln_block<IO_BF16, P_BF16, 5>(m, b.row0, b.nrows); break;
    case 6: ln_block<IO_BF16, P_BF16, 6>(m, b.row0, b.nrows); break;
    case 7: ln_block<IO_BF16, P_BF16, 7>(m, b.row0, b.nrows); break;
    default: ln_block<IO_BF16, P_BF16, 8>(m, b.row0, b.nrows); break;
  }
}

cudaError_t launch_layernorm(const opt_plan* p, cudaStream_t s) {
  const char* base = static_cast<const char*>(p->dev_tables);
  auto* members = reinterpret_cast<const LnMember*>(base + p->off0);
  auto* blocks = reinterpret_cast<const LnBlock*>(base + p->off1);
  const bool io_bf16 = p->io == OPT_BF16, p_bf16 = p->param == OPT_BF16;
  if (io_bf16 && p_bf16) batched_layernorm_bf16_kernel<true><<<p->grid, p->block, 0, s>>>(members, blocks);
  else if (io_bf16) batched_layernorm_bf16_kernel<false><<<p->grid, p->block, 0, s>>>(members, blocks);
  else if (p_bf16) batched_layernorm_kernel<false, true><<<p->grid, p->block, 0, s>>>(members, blocks);
  else batched_layernorm_kernel<false, false><<<p->grid, p->block, 0, s>>>(members, blocks);
  return cudaGetLastError();
}

}  // namespace optb

using namespace optb;

extern "C" opt_status opt_layernorm_plan_create(const opt_layernorm_member* members, int32_t n, opt_dtype io,
                                                opt_dtype param, int device, opt_plan** plan) {
  if (plan) *plan = nullptr;
  if (!plan || !members) return fail(OPT_ERR_INVALID_ARG, "opt_layernorm_plan_create: NULL argument");
  if (n < 1 || n > 65535) return fail(OPT_ERR_INVALID_ARG, "n = %d outside [1, 65535]", n);
  if ((io != OPT_F32 && io != OPT_BF16) || (param != OPT_F32 && param != OPT_BF16))
    return fail(OPT_ERR_INVALID_ARG, "bad dtype");
  const int esz = elem_size(io), V = vec_elems(io), pesz = elem_size(param);
  std::vector<Region> regions;
  std::vector<LnMember> tab;
  std::vector<LnBlock> blocks;
  int64_t bytes = 0;
  for (int32_t i = 0; i < n; ++i) {
    const opt_layernorm_member& m = members[i];
    if (!m.x || !m.y) return fail(OPT_ERR_INVALID_ARG, "member %d: NULL pointer", i);
    if (m.rows < 1 || m.D < 1) return fail(OPT_ERR_INVALID_ARG, "member %d: rows=%d D=%d must be >= 1", i, m.rows, m.D);
    if (!(m.eps >= 0.f)) return fail(OPT_ERR_INVALID_ARG, "member %d: eps must be >= 0", i);
    if (m.rows > 1 && (m.ldx < m.D || m.ldy < m.D)) return fail(OPT_ERR_INVALID_ARG, "member %d: row stride smaller than D", i);
    if (!aligned16(m.x) || !aligned16(m.y) || !aligned16(m.gamma) || !aligned16(m.beta))
      return fail(OPT_ERR_ALIGNMENT, "member %d: pointers must be 16-byte aligned", i);
    if (m.D % V) return fail(OPT_ERR_ALIGNMENT, "member %d: D=%d is not a multiple of %d", i, m.D, V);
    if (m.rows > 1 && (m.ldx % V || m.ldy % V))
      return fail(OPT_ERR_ALIGNMENT, "member %d: row strides must be multiples of %d elements", i, V);
    const int nvec = m.D / V;
    if (nvec > 32 * kLnMaxVpl)
      return fail(OPT_ERR_UNSUPPORTED, "member %d: D=%d exceeds the register-resident limit %d", i, m.D, 32 * kLnMaxVpl * V);
    regions.push_back({(uintptr_t)m.x, m.ldx * esz, (int64_t)m.D * esz, m.rows, false, i});
    regions.push_back({(uintptr_t)m.y, m.ldy * esz, (int64_t)m.D * esz, m.rows, true, i});
    if (m.gamma) regions.push_back({(uintptr_t)m.gamma, 0, (int64_t)m.D * pesz, 1, false, i});
    if (m.beta) regions.push_back({(uintptr_t)m.beta, 0, (int64_t)m.D * pesz, 1, false, i});
    bytes += 2ll * m.rows * m.D * esz + (m.gamma ? (int64_t)m.D * pesz : 0) + (m.beta ? (int64_t)m.D * pesz : 0);

    // lanes per row: least waste, then 2..4 vectors per lane, then wider
    int best_l = -1, best_vpl = 0;
    long best_score = 1l << 60;
    for (int ll = 5; ll >= 0; --ll) {
      const int L = 1 << ll, vpl = (nvec + L - 1) / L;
      if (vpl > kLnMaxVpl) continue;
      if (L > 1 && L / 2 >= nvec) continue;                 // half the lanes would be idle
      const long waste = (long)L * vpl - nvec;
      const long score = waste * 1000 / nvec * 16 + (vpl < 2 ? 8 : vpl > 4 ? 4 : 0) + (5 - ll);
      if (score < best_score) { best_score = score; best_l = ll; best_vpl = vpl; }
    }
    LnMember t;
    t.x = (const char*)m.x; t.y = (char*)m.y; t.gamma = (const char*)m.gamma; t.beta = (const char*)m.beta;
    t.ldx16 = m.ldx / V; t.ldy16 = m.ldy / V; t.rows = m.rows; t.nvec = nvec;
    t.eps = m.eps; t.inv_D = 1.0f / (float)m.D; t.l_log2 = best_l; t.vpl = best_vpl;
    tab.push_back(t);
    // rows per block: whole passes, ~64 KB of input per block
    const int rpp = kLnThreads >> best_l;
    int64_t passes = std::max<int64_t>(1, 65536 / ((int64_t)rpp * m.D * esz));
    const int64_t rpb = rpp * passes;
    for (int64_t r0 = 0; r0 < m.rows; r0 += rpb)
      blocks.push_back({i, (int32_t)r0, (int32_t)std::min<int64_t>(rpb, m.rows - r0)});
  }
  if (opt_status st = check_independent(regions, /*allow_inplace_self=*/false)) return st;
  if (blocks.size() > (size_t)INT32_MAX) return fail(OPT_ERR_UNSUPPORTED, "too many work items");

  int num_sms = 0;
  if (opt_status st = open_device(device, &num_sms)) return st;
  auto align_up = [](size_t x) { return (x + 255) & ~size_t(255); };
  opt_plan* p = new opt_plan();
  p->kind = kPlanLayerNorm; p->device = device; p->io = io; p->param = param; p->n_members = n;
  p->off0 = 0;
  p->off1 = align_up(tab.size() * sizeof(LnMember));
  const size_t total = p->off1 + align_up(blocks.size() * sizeof(LnBlock));
  std::vector<char> blob(total, 0);
  memcpy(blob.data(), tab.data(), tab.size() * sizeof(LnMember));
  memcpy(blob.data() + p->off1, blocks.data(), blocks.size() * sizeof(LnBlock));
  if (opt_status st = upload_tables(p, blob.data(), total)) { delete p; return st; }
  p->grid = dim3((unsigned)blocks.size());
  p->block = dim3(kLnThreads);
  p->total_tiles = (int32_t)blocks.size();
  p->bytes = bytes; p->flops = 0;
  *plan = p;
  return OPT_OK;
}
