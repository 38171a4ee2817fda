// batched_layernorm: N independent LayerNorms (different D_i, rows_i, strides,
// gamma/beta) in one launch -- batch_layernorm.
//
//   mu = mean(x_r); v = mean((x_r - mu)^2); y_r = (x_r - mu) * rsqrt(v + eps) * gamma + beta
//
// Two kernels (HBM-bound):
//   batched_layernorm_staged_kernel   bf16 activations (configs[1], configs[4] group 1).  Persistent CTAs, three
//       per SM: ONE producer warp + 8 consumer warps around a shared-memory ring (<= 4 stages, 72 KB per CTA).  A
//       work item is a tile of whole rows of one member (~16 KB); the producer takes items from a dynamic scheduler
//       (one atomicAdd per chunk of 8 items, software-pipelined three chunks deep) and streams each tile plus the
//       member's gamma and beta into a stage with cp.async.bulk, counted on the stage's mbarrier; a 64-byte header
//       tells the consumers what the stage holds.  Consumers never issue a global load: a row is owned by L = 2^k
//       lanes (L per member for the least lane waste: D=32 packs 8 rows into a warp, D>=256 uses the whole warp),
//       each lane reads its 16-byte vectors from shared memory, fp32 two-pass statistics (mean, then centred sum
//       of squares) on packed f32x2 arithmetic with width-L shuffle-xor reductions, affine, one RNE, coalesced
//       16-byte st.global.cs -- and, when the member asks for it, the FP8 (E4M3) copy of the rounded output
//       (8-byte stores; activation quantisation fused into the producer of the saved tensor).
//       Rows wider than 1024 elements stay in shared memory and are re-read per pass.
//   batched_layernorm_kernel          fp32 activations: register-resident rows, one block per (member, row range)
//       from a block table, the next rows' vectors prefetched before the current rows' math.
#include <algorithm>
#include <cstdlib>

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

// ======================================================= bf16 staged path =====
// Persistent CTAs (3 per SM), 8 consumer warps + 1 producer warp.  The producer takes work items (a
// tile of ~16 KB of whole rows of one member) from a dynamic scheduler -- one atomic per chunk of 8
// items -- and streams each tile plus the member's gamma/beta into a 4-stage shared-memory ring with
// cp.async.bulk (one copy per tile when the rows are contiguous, one per row otherwise), counted on
// the stage's mbarrier.  Consumers never issue a global load: they read their 16-byte vectors of the
// row from shared memory, do the fp32 two-pass statistics with width-L shuffles on packed f32x2
// arithmetic, and store y with 16-byte coalesced st.global.cs.  Bytes in flight are set by the ring
// (3 x 4 x 16 KB per SM), not by registers.
struct LnsMember {           // 64 bytes
  const char* x; char* y; const char* gamma; const char* beta;
  int64_t ldx16, ldy16;      // row strides in 16-byte vectors
  int32_t nvec;              // D / 8
  float eps, inv_D;
  uint8_t l_log2, vpl, contiguous, pad;     // one 32-bit word: l_log2 | vpl << 8 | contiguous << 16
};
static_assert(sizeof(LnsMember) == 64, "LnsMember is one 64-byte record");
struct LnsItem { int32_t member, row0, nrows, pad; };   // member < 0: padding entry of a chunk

constexpr int kLnsConsumers = 256;
constexpr int kLnsThreads = kLnsConsumers + 32;
constexpr int kLnsItemsPerChunk = 8;
constexpr int kLnsMaxStages = 4;
constexpr int kLnsHdrBytes = 64;
constexpr int kLnsSmemBudget = 72 * 1024;      // per CTA: 3 CTAs per SM

__device__ __forceinline__ uint32_t lns_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void lns_mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done = 0;
  for (uint32_t spin = 0; !done; ++spin) {
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    if (spin > (1u << 26)) __trap();      // a protocol bug becomes a CUDA error, not a hang
  }
}
__device__ __forceinline__ void lns_bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ uint4 lns_lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
  return v;
}

// gamma / beta vector `vec` (8 elements) of the staged parameters as four f32x2
template <bool P_BF16>
__device__ __forceinline__ void lns_param(uint32_t base, bool present, int vec, float dflt, f32x2 (&out)[4]) {
  if (!present) {
#pragma unroll
    for (int k = 0; k < 4; ++k) out[k] = pk2(dflt, dflt);
  } else if (P_BF16) {
    const uint4 v = lns_lds128(base + vec * 16);
    out[0] = bf2_to_f2(v.x); out[1] = bf2_to_f2(v.y); out[2] = bf2_to_f2(v.z); out[3] = bf2_to_f2(v.w);
  } else {
    const uint4 a = lns_lds128(base + vec * 32), b = lns_lds128(base + vec * 32 + 16);
    out[0] = pk2(__uint_as_float(a.x), __uint_as_float(a.y)); out[1] = pk2(__uint_as_float(a.z), __uint_as_float(a.w));
    out[2] = pk2(__uint_as_float(b.x), __uint_as_float(b.y)); out[3] = pk2(__uint_as_float(b.z), __uint_as_float(b.w));
  }
}

struct LnsHdr {               // what the consumers need of a staged item (written by the producer)
  int32_t member, row0, nrows, nvec;
  char* y; int64_t ldy16;
  float eps, inv_D; uint32_t shape;       // l_log2 | vpl << 8 | has_gamma << 16 | has_beta << 17
  uint32_t pad;
  char* y8; int32_t ldy8_8; float scale8;  // FP8 copy of the output (Q8 kernel): base, row stride in 8-byte vectors, scale
};
static_assert(sizeof(LnsHdr) == kLnsHdrBytes, "LnsHdr is the 64-byte stage header");

// FAST: every lane's vectors exist (D = 8 L VPL), the tile is whole passes, gamma and beta are present --
// the common case, compiled without any predicate or branch in the loop body.
template <bool P_BF16, int VPL, int RU, bool FAST, bool Q8>
__device__ __forceinline__ void lns_tile(const LnsHdr& h, uint32_t tile, uint32_t sgamma, uint32_t sbeta) {
  const int l_log2 = h.shape & 0xFF;
  const bool has_g = FAST || ((h.shape >> 16) & 1), has_b = FAST || ((h.shape >> 17) & 1);
  const int L = 1 << l_log2;
  const int lane_in_row = threadIdx.x & (L - 1);
  const int row_in_pass = threadIdx.x >> l_log2;
  const int rpp = kLnsConsumers >> l_log2;
  const int niter = (h.nrows + rpp * RU - 1) / (rpp * RU);
  const uint32_t row_bytes = (uint32_t)h.nvec * 16u;
  int4* yb = reinterpret_cast<int4*>(h.y);
  bool act[VPL];
#pragma unroll
  for (int i = 0; i < VPL; ++i) act[i] = FAST || lane_in_row + i * L < h.nvec;

  // this thread's first vector of the tile; rows advance by rpp per unrolled row, columns by L per vector
  uint32_t xaddr = tile + (uint32_t)row_in_pass * row_bytes + (uint32_t)lane_in_row * 16u;
  const uint32_t row_step = (uint32_t)rpp * row_bytes;
  int4* yrow = yb + (int64_t)(h.row0 + row_in_pass) * h.ldy16 + lane_in_row;
  const int64_t y_step = (int64_t)rpp * h.ldy16;
  // FP8 copy of the rounded output (activation quantisation fused into the LayerNorm)
  int2* y8row = Q8 ? reinterpret_cast<int2*>(h.y8) + (int64_t)(h.row0 + row_in_pass) * h.ldy8_8 + lane_in_row : nullptr;
  const int64_t y8_step = Q8 ? (int64_t)rpp * h.ldy8_8 : 0;
  const bool wr_y = !Q8 || h.y != nullptr, wr_y8 = Q8 && h.y8 != nullptr;
  int rbase = row_in_pass;
  for (int it = 0; it < niter; ++it, xaddr += RU * row_step, yrow += RU * y_step, y8row += RU * y8_step, rbase += RU * rpp) {
    f32x2 x[RU][VPL][4];
    float s[RU], q[RU];
#pragma unroll
    for (int u = 0; u < RU; ++u) {
      const bool rok = FAST || rbase + u * rpp < h.nrows;
      f32x2 acc = 0ull;
#pragma unroll
      for (int i = 0; i < VPL; ++i) {
        uint4 v = make_uint4(0, 0, 0, 0);
        if (rok && act[i]) v = lns_lds128(xaddr + u * row_step + (uint32_t)(i * L) * 16u);
        x[u][i][0] = bf2_to_f2(v.x); x[u][i][1] = bf2_to_f2(v.y); x[u][i][2] = bf2_to_f2(v.z); x[u][i][3] = bf2_to_f2(v.w);
#pragma unroll
        for (int k = 0; k < 4; ++k) acc = add2(acc, x[u][i][k]);      // inactive vectors are zeros
      }
      s[u] = sum2(acc);
    }
    for (int o = L >> 1; o > 0; o >>= 1) {
#pragma unroll
      for (int u = 0; u < RU; ++u) s[u] += __shfl_xor_sync(0xffffffffu, s[u], o);
    }
#pragma unroll
    for (int u = 0; u < RU; ++u) {
      const float nmu = -s[u] * h.inv_D;
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
    for (int i = 0; i < VPL; ++i) {
      if (!act[i]) continue;
      const int vec = lane_in_row + i * L;
      f32x2 g[4], b[4];
      lns_param<P_BF16>(sgamma, has_g, vec, 1.f, g);
      lns_param<P_BF16>(sbeta, has_b, vec, 0.f, b);
#pragma unroll
      for (int u = 0; u < RU; ++u) {
        if (!FAST && rbase + u * rpp >= h.nrows) continue;
        const float rstd = rsqrtf(q[u] * h.inv_D + h.eps);
        const f32x2 rstd2 = pk2(rstd, rstd);
        int4 o;
        o.x = (int)f2_to_bf2(fma2(mul2(x[u][i][0], rstd2), g[0], b[0]));
        o.y = (int)f2_to_bf2(fma2(mul2(x[u][i][1], rstd2), g[1], b[1]));
        o.z = (int)f2_to_bf2(fma2(mul2(x[u][i][2], rstd2), g[2], b[2]));
        o.w = (int)f2_to_bf2(fma2(mul2(x[u][i][3], rstd2), g[3], b[3]));
        if (wr_y) __stcs(yrow + u * y_step + i * L, o);
        if (wr_y8) __stcs(y8row + u * y8_step + i * L, make_int2((int)quant4_e4m3((uint32_t)o.x, (uint32_t)o.y, h.scale8),
                                                                 (int)quant4_e4m3((uint32_t)o.z, (uint32_t)o.w, h.scale8)));
      }
    }
  }
}

// rows wider than 4 vectors per lane (D > 1024): the row stays in shared memory and is re-read per pass
template <bool P_BF16, bool Q8>
__device__ __forceinline__ void lns_tile_wide(const LnsHdr& h, uint32_t tile, uint32_t sgamma, uint32_t sbeta) {
  const bool has_g = (h.shape >> 16) & 1, has_b = (h.shape >> 17) & 1;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t row_bytes = (uint32_t)h.nvec * 16u;
  int4* yb = reinterpret_cast<int4*>(h.y);
  for (int r = warp; r < h.nrows; r += kLnsConsumers / 32) {
    const uint32_t row = tile + (uint32_t)r * row_bytes;
    f32x2 acc = 0ull;
    for (int v = lane; v < h.nvec; v += 32) {
      const uint4 w = lns_lds128(row + v * 16);
      acc = add2(add2(acc, bf2_to_f2(w.x)), add2(bf2_to_f2(w.y), add2(bf2_to_f2(w.z), bf2_to_f2(w.w))));
    }
    float s = sum2(acc);
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    const float nmu = -s * h.inv_D;
    const f32x2 nmu2 = pk2(nmu, nmu);
    acc = 0ull;
    for (int v = lane; v < h.nvec; v += 32) {
      const uint4 w = lns_lds128(row + v * 16);
      const uint32_t ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
      for (int k = 0; k < 4; ++k) { const f32x2 d = add2(bf2_to_f2(ww[k]), nmu2); acc = fma2(d, d, acc); }
    }
    float q = sum2(acc);
    for (int o = 16; o > 0; o >>= 1) q += __shfl_xor_sync(0xffffffffu, q, o);
    const float rstd = rsqrtf(q * h.inv_D + h.eps);
    const f32x2 rstd2 = pk2(rstd, rstd);
    for (int v = lane; v < h.nvec; v += 32) {
      const uint4 w = lns_lds128(row + v * 16);
      const uint32_t ww[4] = {w.x, w.y, w.z, w.w};
      f32x2 g[4], b[4];
      lns_param<P_BF16>(sgamma, has_g, v, 1.f, g);
      lns_param<P_BF16>(sbeta, has_b, v, 0.f, b);
      uint32_t o[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) o[k] = f2_to_bf2(fma2(mul2(add2(bf2_to_f2(ww[k]), nmu2), rstd2), g[k], b[k]));
      if (!Q8 || h.y != nullptr) __stcs(yb + (int64_t)(h.row0 + r) * h.ldy16 + v, make_int4((int)o[0], (int)o[1], (int)o[2], (int)o[3]));
      if (Q8 && h.y8 != nullptr)
        __stcs(reinterpret_cast<int2*>(h.y8) + (int64_t)(h.row0 + r) * h.ldy8_8 + v,
               make_int2((int)quant4_e4m3(o[0], o[1], h.scale8), (int)quant4_e4m3(o[2], o[3], h.scale8)));
    }
  }
}

// stage layout: [tile_max bytes of rows][gamma: pmax][beta: pmax][64-byte header]
// Q8: some member wants the FP8 (E4M3) copy of its output; `ext` then holds one 16-byte record per member
// {y8 pointer, row stride in 8-byte vectors, scale8} (y8 == NULL: none for that member).
// OCC: CTAs per SM the instantiation is compiled for.  3 (72 registers) for small groups -- a few items per CTA, where
// the launch ramp dominates and more resident CTAs start more loads at once (configs[1]: 33 vs 38 us); 2 (no spills)
// for large groups (configs[4]'s LayerNorm group: 303 vs 314 us) and for the Q8 instantiation, whose extra pointers /
// flags of the FP8 store would spill at 72 registers.  The bytes in flight are set by the ring either way.
template <bool P_BF16, bool Q8, int OCC>
__global__ void __launch_bounds__(kLnsThreads, OCC)
batched_layernorm_staged_kernel(const LnsMember* __restrict__ members, const LnsItem* __restrict__ items, int n_chunks,
                                int* __restrict__ counters, int nstages, int tile_max, int pmax, const uint4* __restrict__ ext) {
  extern __shared__ __align__(128) uint8_t lns_smem[];
  __shared__ __align__(8) uint64_t bars[2 * kLnsMaxStages];
  const uint32_t sbase = lns_smem_u32(lns_smem);
  const uint32_t stage_bytes = (uint32_t)(tile_max + 2 * pmax + kLnsHdrBytes);
  auto full_bar = [&](int s) { return lns_smem_u32(&bars[s]); };
  auto empty_bar = [&](int s) { return lns_smem_u32(&bars[kLnsMaxStages + s]); };
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < nstages; ++s) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(full_bar(s)));
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(empty_bar(s)), "n"(kLnsConsumers / 32));
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp == kLnsConsumers / 32) {
    // --------------------------------------------------------- producer ----
    // Software pipeline over chunks so that no global latency sits between two items: while chunk n is
    // issued, the member records of chunk n+1 (lane 4g+k holds 16-byte piece k of item g's member), the
    // item line of chunk n+2 and the id of chunk n+3 are in flight.
    int s = 0; uint32_t ph = 0;
    auto fetch_id = [&]() { int v = 0; if (lane == 0) v = atomicAdd(counters, 1) + (int)gridDim.x; return v; };
    auto load_line = [&](int cc) {
      int4 v = make_int4(-1, 0, 0, 0);
      if (lane < kLnsItemsPerChunk && cc < n_chunks) v = __ldg(reinterpret_cast<const int4*>(items) + (size_t)cc * kLnsItemsPerChunk + lane);
      return v;
    };
    auto load_members = [&](const int4& line) {
      const int mem = __shfl_sync(0xffffffffu, line.x, lane >> 2);
      uint4 v = make_uint4(0, 0, 0, 0);
      if (mem >= 0) v = __ldg(reinterpret_cast<const uint4*>(members + mem) + (lane & 3));
      return v;
    };
    auto load_ext = [&](const int4& line) {        // lane g < 8: the FP8 record of item g's member
      uint4 v = make_uint4(0, 0, 0, 0);
      if (Q8 && lane < kLnsItemsPerChunk && line.x >= 0) v = __ldg(ext + line.x);
      return v;
    };
    int c0 = blockIdx.x;
    int4 line0 = load_line(c0);
    int c1 = __shfl_sync(0xffffffffu, fetch_id(), 0);
    int4 line1 = load_line(c1);
    int c2 = fetch_id();
    uint4 mv0 = load_members(line0);
    uint4 xv0 = load_ext(line0);
    while (c0 < n_chunks) {
      c2 = __shfl_sync(0xffffffffu, c2, 0);
      const uint4 mv1 = load_members(line1);
      const uint4 xv1 = load_ext(line1);
      const int4 line2 = load_line(c2);
      const int c3 = fetch_id();
#pragma unroll 1
      for (int g = 0; g < kLnsItemsPerChunk; ++g) {
        const int member = __shfl_sync(0xffffffffu, line0.x, g);
        if (member < 0) continue;      // warp-uniform
        const int row0 = __shfl_sync(0xffffffffu, line0.y, g), nrows = __shfl_sync(0xffffffffu, line0.z, g);
        auto piece = [&](uint32_t w, int k) { return __shfl_sync(0xffffffffu, w, 4 * g + k); };
        auto ptr64 = [](uint32_t lo, uint32_t hi) { return ((uint64_t)hi << 32) | lo; };
        LnsMember m;
        m.x = reinterpret_cast<const char*>(ptr64(piece(mv0.x, 0), piece(mv0.y, 0)));
        m.y = reinterpret_cast<char*>(ptr64(piece(mv0.z, 0), piece(mv0.w, 0)));
        m.gamma = reinterpret_cast<const char*>(ptr64(piece(mv0.x, 1), piece(mv0.y, 1)));
        m.beta = reinterpret_cast<const char*>(ptr64(piece(mv0.z, 1), piece(mv0.w, 1)));
        m.ldx16 = (int64_t)ptr64(piece(mv0.x, 2), piece(mv0.y, 2));
        m.ldy16 = (int64_t)ptr64(piece(mv0.z, 2), piece(mv0.w, 2));
        m.nvec = (int)piece(mv0.x, 3); m.eps = __uint_as_float(piece(mv0.y, 3)); m.inv_D = __uint_as_float(piece(mv0.z, 3));
        const uint32_t shp = piece(mv0.w, 3);                    // l_log2 | vpl << 8 | contiguous << 16
        m.l_log2 = (uint8_t)(shp & 0xFF); m.vpl = (uint8_t)((shp >> 8) & 0xFF); m.contiguous = (uint8_t)((shp >> 16) & 0xFF);
        const uint32_t row_bytes = (uint32_t)m.nvec * 16u;
        const uint32_t pbytes = (uint32_t)m.nvec * (P_BF16 ? 16u : 32u);
        uint4 xe = make_uint4(0, 0, 0, 0);
        if (Q8) { xe.x = __shfl_sync(0xffffffffu, xv0.x, g); xe.y = __shfl_sync(0xffffffffu, xv0.y, g);
                  xe.z = __shfl_sync(0xffffffffu, xv0.z, g); xe.w = __shfl_sync(0xffffffffu, xv0.w, g); }
        lns_mbar_wait(empty_bar(s), ph ^ 1);
        const uint32_t stage = sbase + (uint32_t)s * stage_bytes;
        const uint32_t fb = full_bar(s);
        if (lane == 0) {
          const uint32_t ha = stage + (uint32_t)(tile_max + 2 * pmax);
          const uint32_t shape = (uint32_t)m.l_log2 | ((uint32_t)m.vpl << 8) | ((m.gamma != nullptr) << 16) | ((m.beta != nullptr) << 17);
          const uint64_t yp = reinterpret_cast<uint64_t>(m.y);
          asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(ha), "r"(member), "r"(row0), "r"(nrows), "r"(m.nvec) : "memory");
          asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(ha + 16), "r"((uint32_t)yp), "r"((uint32_t)(yp >> 32)),
                       "r"((uint32_t)m.ldy16), "r"((uint32_t)((uint64_t)m.ldy16 >> 32)) : "memory");
          asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(ha + 32), "r"(__float_as_uint(m.eps)), "r"(__float_as_uint(m.inv_D)),
                       "r"(shape), "r"(0) : "memory");
          if (Q8) asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(ha + 48), "r"(xe.x), "r"(xe.y), "r"(xe.z), "r"(xe.w) : "memory");
          const uint32_t tx = (uint32_t)nrows * row_bytes + (m.gamma ? pbytes : 0u) + (m.beta ? pbytes : 0u);
          asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(fb), "r"(tx) : "memory");
          if (m.gamma) lns_bulk_load(stage + tile_max, m.gamma, pbytes, fb);
          if (m.beta) lns_bulk_load(stage + tile_max + pmax, m.beta, pbytes, fb);
          if (m.contiguous) lns_bulk_load(stage, m.x + (int64_t)row0 * m.ldx16 * 16, (uint32_t)nrows * row_bytes, fb);
        }
        if (!m.contiguous)
          for (int r = lane; r < nrows; r += 32)
            lns_bulk_load(stage + (uint32_t)r * row_bytes, m.x + (int64_t)(row0 + r) * m.ldx16 * 16, row_bytes, fb);
        if (++s == nstages) { s = 0; ph ^= 1; }
      }
      c0 = c1; line0 = line1; mv0 = mv1; xv0 = xv1;
      c1 = c2; line1 = line2;
      c2 = c3;
    }
    asm volatile("" ::"r"(c2) : "memory");     // the last id fetch has returned before the counters are re-armed
    // end marker; the last CTA to finish re-arms the scheduler counters for the next launch of the plan
    lns_mbar_wait(empty_bar(s), ph ^ 1);
    if (lane == 0) {
      asm volatile("st.shared.b32 [%0], %1;" ::"r"(sbase + (uint32_t)s * stage_bytes + (uint32_t)(tile_max + 2 * pmax)), "r"(-1) : "memory");
      asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(full_bar(s)) : "memory");
      __threadfence();
      if (atomicAdd(counters + 1, 1) == (int)gridDim.x - 1) { counters[0] = 0; counters[1] = 0; __threadfence(); }
    }
  } else {
    // -------------------------------------------------------- consumers ----
    int s = 0; uint32_t ph = 0;
    for (;;) {
      lns_mbar_wait(full_bar(s), ph);
      const uint32_t ha = sbase + (uint32_t)s * stage_bytes + (uint32_t)(tile_max + 2 * pmax);
      const uint4 h0 = lns_lds128(ha), h1 = lns_lds128(ha + 16), h2 = lns_lds128(ha + 32);
      LnsHdr h;                                   // field by field: stays in registers
      h.member = (int)h0.x; h.row0 = (int)h0.y; h.nrows = (int)h0.z; h.nvec = (int)h0.w;
      h.y = reinterpret_cast<char*>(((uint64_t)h1.y << 32) | h1.x);
      h.ldy16 = (int64_t)(((uint64_t)h1.w << 32) | h1.z);
      h.eps = __uint_as_float(h2.x); h.inv_D = __uint_as_float(h2.y); h.shape = h2.z;
      h.y8 = nullptr; h.ldy8_8 = 0; h.scale8 = 0.f;
      if (h.member < 0) break;
      if (Q8) {
        const uint4 h3 = lns_lds128(ha + 48);
        h.y8 = reinterpret_cast<char*>(((uint64_t)h3.y << 32) | h3.x); h.ldy8_8 = (int32_t)h3.z; h.scale8 = __uint_as_float(h3.w);
      }
      const uint32_t tile = sbase + (uint32_t)s * stage_bytes;
      const uint32_t sg = tile + tile_max, sb = sg + pmax;
      const int vpl = (h.shape >> 8) & 0xFF, ll = h.shape & 0xFF;
      const int ru = vpl == 1 ? 4 : vpl == 2 ? 2 : 1;
      const bool fast = (h.shape >> 16) == 3u && h.nvec == (vpl << ll) && h.nrows % ((kLnsConsumers >> ll) * ru) == 0;
      switch (fast ? vpl : vpl + 8) {   // CTA-uniform
        case 1: lns_tile<P_BF16, 1, 4, true, Q8>(h, tile, sg, sb); break;
        case 2: lns_tile<P_BF16, 2, 2, true, Q8>(h, tile, sg, sb); break;
        case 3: lns_tile<P_BF16, 3, 1, true, Q8>(h, tile, sg, sb); break;
        case 4: lns_tile<P_BF16, 4, 1, true, Q8>(h, tile, sg, sb); break;
        case 9: lns_tile<P_BF16, 1, 4, false, Q8>(h, tile, sg, sb); break;
        case 10: lns_tile<P_BF16, 2, 2, false, Q8>(h, tile, sg, sb); break;
        case 11: lns_tile<P_BF16, 3, 1, false, Q8>(h, tile, sg, sb); break;
        case 12: lns_tile<P_BF16, 4, 1, false, Q8>(h, tile, sg, sb); break;
        default: lns_tile_wide<P_BF16, Q8>(h, tile, sg, sb); break;
      }
      __syncwarp();
      if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(empty_bar(s)) : "memory");
      if (++s == nstages) { s = 0; ph ^= 1; }
    }
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
  char* base = static_cast<char*>(p->dev_tables);
  const bool io_bf16 = p->io == OPT_BF16, p_bf16 = p->param == OPT_BF16;
  if (io_bf16) {
    auto* members = reinterpret_cast<const LnsMember*>(base + p->off0);
    auto* items = reinterpret_cast<const LnsItem*>(base + p->off1);
    int* counters = reinterpret_cast<int*>(base + p->off2);
    const uint4* ext = p->off3 ? reinterpret_cast<const uint4*>(base + p->off3) : nullptr;
#define LNS_LAUNCH(PB, Q, OCC)                                                                                              \
    batched_layernorm_staged_kernel<PB, Q, OCC><<<p->grid, p->block, p->smem, s>>>(members, items, p->n_chunks, counters,  \
                                                                                   p->nstages, p->ln_tile_max, p->ln_pmax, ext)
    if (ext) { if (p_bf16) LNS_LAUNCH(true, true, 2); else LNS_LAUNCH(false, true, 2); }
    else if (p->ncta == 2) { if (p_bf16) LNS_LAUNCH(true, false, 2); else LNS_LAUNCH(false, false, 2); }
    else { if (p_bf16) LNS_LAUNCH(true, false, 3); else LNS_LAUNCH(false, false, 3); }
#undef LNS_LAUNCH
    return cudaGetLastError();
  }
  auto* members = reinterpret_cast<const LnMember*>(base + p->off0);
  auto* blocks = reinterpret_cast<const LnBlock*>(base + p->off1);
  if (p_bf16) batched_layernorm_kernel<false, true><<<p->grid, p->block, 0, s>>>(members, blocks);
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
  std::vector<LnsMember> stab;      // bf16 staged path
  std::vector<LnsItem> sitems;
  int64_t tile_max = 0, pmax = 0;
  int64_t bytes = 0;
  bool any_y8 = false;
  std::vector<uint4> sext;          // bf16 staged path: FP8 record per member {y8 lo, y8 hi, ldy8 / 8, scale8}
  for (int32_t i = 0; i < n; ++i) {
    const opt_layernorm_member& m = members[i];
    if (!m.x || (!m.y && !m.y8)) return fail(OPT_ERR_INVALID_ARG, "member %d: NULL pointer", i);
    if (m.rows < 1 || m.D < 1) return fail(OPT_ERR_INVALID_ARG, "member %d: rows=%d D=%d must be >= 1", i, m.rows, m.D);
    if (!(m.eps >= 0.f)) return fail(OPT_ERR_INVALID_ARG, "member %d: eps must be >= 0", i);
    if (m.rows > 1 && (m.ldx < m.D || (m.y && m.ldy < m.D))) return fail(OPT_ERR_INVALID_ARG, "member %d: row stride smaller than D", i);
    if (!aligned16(m.x) || !aligned16(m.y) || !aligned16(m.gamma) || !aligned16(m.beta))
      return fail(OPT_ERR_ALIGNMENT, "member %d: pointers must be 16-byte aligned", i);
    if (m.D % V) return fail(OPT_ERR_ALIGNMENT, "member %d: D=%d is not a multiple of %d", i, m.D, V);
    if (m.rows > 1 && (m.ldx % V || (m.y && m.ldy % V)))
      return fail(OPT_ERR_ALIGNMENT, "member %d: row strides must be multiples of %d elements", i, V);
    if (m.y8) {      // FP8 copy of the output (activation quantisation fused into the LayerNorm)
      if (io != OPT_BF16) return fail(OPT_ERR_UNSUPPORTED, "member %d: the FP8 output is implemented for bf16 activations", i);
      if (!(m.scale8 > 0.f) || !(m.scale8 < INFINITY)) return fail(OPT_ERR_INVALID_ARG, "member %d: scale8 must be a positive finite number", i);
      if (m.rows > 1 && m.ldy8 < m.D) return fail(OPT_ERR_INVALID_ARG, "member %d: ldy8 smaller than D", i);
      if ((reinterpret_cast<uintptr_t>(m.y8) & 7u) || m.ldy8 % 8)
        return fail(OPT_ERR_ALIGNMENT, "member %d: y8 needs an 8-byte aligned base and ldy8 %% 8 == 0", i);
      any_y8 = true;
    }
    const int nvec = m.D / V;
    if (nvec > 32 * kLnMaxVpl)
      return fail(OPT_ERR_UNSUPPORTED, "member %d: D=%d exceeds the register-resident limit %d", i, m.D, 32 * kLnMaxVpl * V);
    regions.push_back({(uintptr_t)m.x, m.ldx * esz, (int64_t)m.D * esz, m.rows, false, i});
    if (m.y) regions.push_back({(uintptr_t)m.y, m.ldy * esz, (int64_t)m.D * esz, m.rows, true, i});
    if (m.y8) regions.push_back({(uintptr_t)m.y8, m.ldy8, (int64_t)m.D, m.rows, true, i});
    if (m.gamma) regions.push_back({(uintptr_t)m.gamma, 0, (int64_t)m.D * pesz, 1, false, i});
    if (m.beta) regions.push_back({(uintptr_t)m.beta, 0, (int64_t)m.D * pesz, 1, false, i});
    bytes += (int64_t)m.rows * m.D * esz * (m.y ? 2 : 1) + (m.y8 ? (int64_t)m.rows * m.D : 0) + (m.gamma ? (int64_t)m.D * pesz : 0) + (m.beta ? (int64_t)m.D * pesz : 0);

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
    if (io == OPT_BF16) {
      LnsMember t;
      t.x = (const char*)m.x; t.y = (char*)m.y; t.gamma = (const char*)m.gamma; t.beta = (const char*)m.beta;
      t.ldx16 = m.ldx / V; t.ldy16 = m.ldy / V; t.nvec = nvec; t.eps = m.eps; t.inv_D = 1.0f / (float)m.D;
      t.l_log2 = (uint8_t)best_l; t.vpl = (uint8_t)best_vpl; t.contiguous = (m.rows == 1 || m.ldx == m.D); t.pad = 0;
      stab.push_back(t);
      const uint64_t y8p = reinterpret_cast<uint64_t>(m.y8);
      float sc = m.y8 ? m.scale8 : 0.f;
      uint32_t scbits; memcpy(&scbits, &sc, 4);
      sext.push_back(make_uint4((uint32_t)y8p, (uint32_t)(y8p >> 32), (uint32_t)(m.ldy8 / 8), scbits));
      // work items: whole rows, ~16 KB, a multiple of what one pass of the CTA covers
      const int64_t row_bytes = (int64_t)nvec * 16;
      const int rpp = kLnsConsumers >> best_l;
      const int unit = best_vpl > 4 ? kLnsConsumers / 32 : rpp * (best_vpl == 1 ? 4 : best_vpl == 2 ? 2 : 1);
      int64_t R = std::max<int64_t>(1, 16384 / row_bytes);
      if (R >= unit) R = R / unit * unit;
      R = std::min<int64_t>(R, m.rows);
      tile_max = std::max<int64_t>(tile_max, R * row_bytes);
      pmax = std::max<int64_t>(pmax, (int64_t)nvec * (param == OPT_BF16 ? 16 : 32));
      for (int64_t r0 = 0; r0 < m.rows; r0 += R)
        sitems.push_back({i, (int32_t)r0, (int32_t)std::min<int64_t>(R, m.rows - r0), 0});
      continue;
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
  DeviceGuard device_guard;      // the caller's current device is restored on return
  if (opt_status st = open_device(device, &num_sms)) return st;
  auto align_up = [](size_t x) { return (x + 255) & ~size_t(255); };
  opt_plan* p = new opt_plan();
  p->kind = kPlanLayerNorm; p->device = device; p->io = io; p->param = param; p->n_members = n;
  p->bytes = bytes; p->flops = 0;
  if (io == OPT_BF16) {
    // ring shape: stage = row tile + gamma + beta + header; as many stages (<= 4) as fit 72 KB (3 CTAs per SM)
    tile_max = (tile_max + 127) & ~int64_t(127);
    pmax = (pmax + 127) & ~int64_t(127);
    const int64_t stage_bytes = tile_max + 2 * pmax + kLnsHdrBytes;
    const int nstages = (int)std::min<int64_t>(kLnsMaxStages, kLnsSmemBudget / stage_bytes);
    if (nstages < 2) { delete p; return fail(OPT_ERR_UNSUPPORTED, "LayerNorm rows too wide for the shared-memory ring"); }
    // CTAs per SM (see the kernel): 2 for large groups (>= 64 items per CTA) and whenever an FP8 copy is written, else 3
    const int occ = (any_y8 || sitems.size() >= (size_t)64 * 2 * num_sms) ? 2 : 3;
    const int n_cta = num_sms * occ;
    // chunks of 8 consecutive items (one 128-byte table line, one atomic); the last 4 waves one item per chunk
    const LnsItem pad_item = {-1, 0, 0, 0};
    const size_t tail_waves = 4;
    const size_t tail = std::min(sitems.size(), tail_waves * n_cta);
    const size_t body = sitems.size() - tail;
    std::vector<LnsItem> chunked;
    for (size_t k = 0; k < body; k += kLnsItemsPerChunk)
      for (int g = 0; g < kLnsItemsPerChunk; ++g) chunked.push_back(k + g < body ? sitems[k + g] : pad_item);
    for (size_t k = body; k < sitems.size(); ++k) {
      chunked.push_back(sitems[k]);
      for (int g = 1; g < kLnsItemsPerChunk; ++g) chunked.push_back(pad_item);
    }
    const int64_t n_chunks = (int64_t)(chunked.size() / kLnsItemsPerChunk);
    p->off0 = 0;
    p->off1 = align_up(stab.size() * sizeof(LnsMember));
    p->off2 = p->off1 + align_up(chunked.size() * sizeof(LnsItem));
    p->off3 = any_y8 ? p->off2 + 256 : 0;                      // FP8 records (selects the Q8 kernel)
    const size_t total = p->off2 + 256 + (any_y8 ? align_up(sext.size() * sizeof(uint4)) : 0);   // + scheduler counters, zero-initialised
    std::vector<char> blob(total, 0);
    memcpy(blob.data(), stab.data(), stab.size() * sizeof(LnsMember));
    memcpy(blob.data() + p->off1, chunked.data(), chunked.size() * sizeof(LnsItem));
    if (any_y8) memcpy(blob.data() + p->off3, sext.data(), sext.size() * sizeof(uint4));
    if (opt_status st = upload_tables(p, blob.data(), total)) { delete p; return st; }
    const int smem = (int)(nstages * stage_bytes);
    // the attribute belongs to the kernel FUNCTION, not to the plan (the last call wins): always the fixed budget,
    // so that a later, smaller plan never lowers the limit under a live, larger one
    const bool pb = param == OPT_BF16;
    const void* fn = any_y8 ? (pb ? (const void*)batched_layernorm_staged_kernel<true, true, 2> : (const void*)batched_layernorm_staged_kernel<false, true, 2>)
                   : occ == 2 ? (pb ? (const void*)batched_layernorm_staged_kernel<true, false, 2> : (const void*)batched_layernorm_staged_kernel<false, false, 2>)
                              : (pb ? (const void*)batched_layernorm_staged_kernel<true, false, 3> : (const void*)batched_layernorm_staged_kernel<false, false, 3>);
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, kLnsSmemBudget);
    if (e != cudaSuccess) {
      cudaFree(p->dev_tables); delete p;
      return fail(OPT_ERR_CUDA, "cudaFuncSetAttribute(max dynamic smem %d) failed: %s", smem, cudaGetErrorString(e));
    }
    p->grid = dim3((unsigned)std::min<int64_t>(n_chunks, n_cta));
    p->block = dim3(kLnsThreads);
    p->smem = (size_t)smem;
    p->total_tiles = (int32_t)sitems.size();
    p->n_chunks = (int32_t)n_chunks; p->nstages = nstages; p->ln_tile_max = (int32_t)tile_max; p->ln_pmax = (int32_t)pmax;
    p->ncta = occ;                                             // which instantiation launch_layernorm picks
    *plan = p;
    return OPT_OK;
  }
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
