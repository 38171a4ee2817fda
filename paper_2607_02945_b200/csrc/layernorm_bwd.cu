// batched_layernorm_bwd: the backward of N independent LayerNorms in ONE launch (the paper's
// headline metric is TRAINING throughput, and batch_layernorm groups appear in the backward graph too).
//
//   mu, v over the last dim; rstd = 1/sqrt(v + eps); xhat = (x - mu) rstd; g = dy * gamma
//   dx     = rstd * (g - mean(g) - xhat * mean(g xhat))                       per row
//   dgamma = sum_rows dy * xhat ;  dbeta = sum_rows dy                         per column
//
// Design (HBM-bound: x and dy read once, dx written once):
//   * a row is owned by L = 2^k lanes of a warp, each lane keeps its <= 2 16-byte vectors of x and of dy in
//     registers; fp32 statistics (two-pass) and the two row means by width-L shuffles, as in the forward kernel;
//   * every thread accumulates dy*xhat and dy for its own columns over the rows it visits; at the end of the block
//     the row groups are summed through shared memory in a fixed order and the block's partial goes to a plan-owned
//     workspace; the LAST block of a member (atomic ticket, re-armed by that block) adds the partials in part order
//     and writes dgamma / dbeta: one launch, no atomics on data, bitwise reproducible.
#include <algorithm>

#include "common.h"

namespace optb {

struct LnbMember {
  const char* x; const char* dy; const char* gamma; char* dx; char* dgamma; char* dbeta;
  int64_t ldx16, lddy16, lddx16;   // row strides in 16-byte vectors
  float* ws;                       // [nparts][2][D] fp32 partial sums (plan workspace)
  int32_t* ticket;                 // blocks of this member that have finished
  int32_t rows, nvec, nparts;
  float eps, inv_D;
  int32_t l_log2, vpl;
};
struct LnbBlock { int32_t member, row0, nrows, part; };

constexpr int kLnbThreads = 256;
constexpr int kLnbSlotKB = 32;       // thread-private cp.async prefetch slots per block (alias the reduction buffer)
constexpr int kLnbTargetBlocks = 16 * 148;   // blocks a large group should still have (see the planner)
constexpr int kLnbMaxVpl = 2;        // D <= 512: x, dy and the two column accumulators stay in registers

__device__ __forceinline__ void lnb_unpack(const int4& v, float (&f)[8]) {
  const uint32_t* u = reinterpret_cast<const uint32_t*>(&v);
#pragma unroll
  for (int i = 0; i < 4; ++i) { f[2 * i] = bf16_lo(u[i]); f[2 * i + 1] = bf16_hi(u[i]); }
}

template <bool P_BF16>
__device__ __forceinline__ void lnb_store_param(char* base, int col, float v) {
  if (P_BF16) reinterpret_cast<__nv_bfloat16*>(base)[col] = __float2bfloat16_rn(v);
  else reinterpret_cast<float*>(base)[col] = v;
}

// butterfly sum over the L = 2^LL lanes that own a row (unrolled)
template <int LL>
__device__ __forceinline__ float lnb_rowsum(float v) {
#pragma unroll
  for (int o = (1 << LL) >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

template <bool P_BF16, int VPL, int LL>
__device__ __forceinline__ void lnb_block(const LnbMember& m, const LnbBlock& b, float* red) {
  constexpr int L = 1 << LL;
  const int lane_in_row = threadIdx.x & (L - 1);
  const int row_in_pass = threadIdx.x >> LL;
  constexpr int rpp = kLnbThreads >> LL;
  const int D = m.nvec * 8;
  const int4* xb = reinterpret_cast<const int4*>(m.x);
  const int4* dyb = reinterpret_cast<const int4*>(m.dy);
  int4* dxb = reinterpret_cast<int4*>(m.dx);
  bool act[VPL];
  f32x2 gam[VPL][4], acc_g[VPL][4], acc_b[VPL][4];       // packed fp32 pairs (add/mul/fma.rn.f32x2)
#pragma unroll
  for (int i = 0; i < VPL; ++i) {
    const int vec = lane_in_row + i * L;
    act[i] = vec < m.nvec;
#pragma unroll
    for (int k = 0; k < 4; ++k) { gam[i][k] = pk2(1.f, 1.f); acc_g[i][k] = 0ull; acc_b[i][k] = 0ull; }
    if (act[i] && m.gamma != nullptr) {
      if (P_BF16) {
        const int4 v = __ldg(reinterpret_cast<const int4*>(m.gamma) + vec);
        const uint32_t* u = reinterpret_cast<const uint32_t*>(&v);
#pragma unroll
        for (int k = 0; k < 4; ++k) gam[i][k] = bf2_to_f2(u[k]);
      } else {
        const float4 a = __ldg(reinterpret_cast<const float4*>(m.gamma) + 2 * vec), c = __ldg(reinterpret_cast<const float4*>(m.gamma) + 2 * vec + 1);
        gam[i][0] = pk2(a.x, a.y); gam[i][1] = pk2(a.z, a.w); gam[i][2] = pk2(c.x, c.y); gam[i][3] = pk2(c.z, c.w);
      }
    }
  }
  const int npass = (b.nrows + rpp - 1) / rpp;
  // The kernel is bound by loads in flight, not by issue slots, and registers are what it cannot spare (64 x 4 blocks
  // per SM): the vectors of the next kPD passes travel through THREAD-PRIVATE slots of shared memory filled with
  // cp.async (no register is held while a load is in flight).  The slots alias the reduction buffer `red`, which is only
  // used after the row loop (a __syncthreads separates the two uses).
  constexpr int kPD = kLnbSlotKB / (8 * VPL);                           // kLnbSlotKB of slots per block: 4 passes (VPL 1), 2 (VPL 2); 48 KB measured no faster
  const uint32_t slot0 = (uint32_t)__cvta_generic_to_shared(red) + threadIdx.x * 16u;
  auto slot = [&](int pass, int i, int which) {                         // [pass % kPD][i][x | dy][thread]
    return slot0 + (uint32_t)((((pass % kPD) * VPL + i) * 2 + which) * kLnbThreads) * 16u;
  };
  auto fetch = [&](int pass) {
    const int r = pass * rpp + row_in_pass;
#pragma unroll
    for (int i = 0; i < VPL; ++i) {
      if (pass < npass && r < b.nrows && act[i]) {
        const int4* gx = xb + (int64_t)(b.row0 + r) * m.ldx16 + lane_in_row + i * L;
        const int4* gd = dyb + (int64_t)(b.row0 + r) * m.lddy16 + lane_in_row + i * L;
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(slot(pass, i, 0)), "l"(gx) : "memory");
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(slot(pass, i, 1)), "l"(gd) : "memory");
      } else if (pass < npass) {                                        // rows / vectors that do not exist read as zeros
        asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(slot(pass, i, 0)), "r"(0) : "memory");
        asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(slot(pass, i, 1)), "r"(0) : "memory");
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");               // one group per pass, empty ones included
  };
#pragma unroll
  for (int pp = 0; pp < kPD; ++pp) fetch(pp);
  int4 nx[VPL], nd[VPL];
  for (int pass = 0; pass < npass; ++pass) {
    const int r = pass * rpp + row_in_pass;
    const bool ok = r < b.nrows;
    f32x2 x[VPL][4], dy[VPL][4];
    // three row sums that do not depend on the mean go through ONE butterfly: sum x, sum g, sum g x  (g = dy gamma);
    // sum g xhat = rstd (sum g x - mu sum g)
    f32x2 s2 = 0ull, sg2 = 0ull, sgx2 = 0ull;
    asm volatile("cp.async.wait_group %0;" ::"n"(kPD - 1) : "memory");   // this pass's group has landed
#pragma unroll
    for (int i = 0; i < VPL; ++i) {
      asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(nx[i].x), "=r"(nx[i].y), "=r"(nx[i].z), "=r"(nx[i].w) : "r"(slot(pass, i, 0)) : "memory");
      asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(nd[i].x), "=r"(nd[i].y), "=r"(nd[i].z), "=r"(nd[i].w) : "r"(slot(pass, i, 1)) : "memory");
    }
#pragma unroll
    for (int i = 0; i < VPL; ++i) {
      const uint32_t* ux = reinterpret_cast<const uint32_t*>(&nx[i]);
      const uint32_t* ud = reinterpret_cast<const uint32_t*>(&nd[i]);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        x[i][k] = bf2_to_f2(ux[k]);                          // inactive vectors are zeros
        dy[i][k] = bf2_to_f2(ud[k]);
        const f32x2 g = mul2(dy[i][k], gam[i][k]);
        s2 = add2(s2, x[i][k]); sg2 = add2(sg2, g); sgx2 = fma2(g, x[i][k], sgx2);
      }
    }
    fetch(pass + kPD);                       // refill the slot this pass has just read
    const float s = lnb_rowsum<LL>(sum2(s2)), sg = lnb_rowsum<LL>(sum2(sg2));
    float sgx = lnb_rowsum<LL>(sum2(sgx2));
    const float mu = s * m.inv_D;
    const f32x2 nmu2 = pk2(-mu, -mu);
    f32x2 q2 = 0ull;
#pragma unroll
    for (int i = 0; i < VPL; ++i)
      if (act[i]) {
#pragma unroll
        for (int k = 0; k < 4; ++k) { x[i][k] = add2(x[i][k], nmu2); q2 = fma2(x[i][k], x[i][k], q2); }
      }
    const float q = lnb_rowsum<LL>(sum2(q2));
    const float rstd = rsqrtf(q * m.inv_D + m.eps);
    sgx = rstd * (sgx - mu * sg);
    const float mg = sg * m.inv_D, mgx = sgx * m.inv_D;
    const f32x2 rstd2 = pk2(rstd, rstd), nmg2 = pk2(-mg, -mg), nmgx2 = pk2(-mgx, -mgx);
    if (ok) {
#pragma unroll
      for (int i = 0; i < VPL; ++i)
        if (act[i]) {
          uint32_t o[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const f32x2 xh = mul2(x[i][k], rstd2);
            acc_g[i][k] = fma2(dy[i][k], xh, acc_g[i][k]);
            acc_b[i][k] = add2(acc_b[i][k], dy[i][k]);
            // rstd * (dy gamma - mean(g) - xhat mean(g xhat))
            o[k] = f2_to_bf2(mul2(fma2(xh, nmgx2, fma2(dy[i][k], gam[i][k], nmg2)), rstd2));
          }
          __stcs(dxb + (int64_t)(b.row0 + r) * m.lddx16 + lane_in_row + i * L, make_int4((int)o[0], (int)o[1], (int)o[2], (int)o[3]));
        }
    }
  }
  // ---- column sums of the block: row groups -> shared memory -> fixed-order sum -> workspace part
  const bool want = m.dgamma != nullptr || m.dbeta != nullptr;
  if (!want) return;
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncthreads();                          // every thread is done with its prefetch slots: `red` becomes the reduction buffer
  float* red_g = red;                       // [rpp][D]
  float* red_b = red + rpp * D;
#pragma unroll
  for (int i = 0; i < VPL; ++i)
    if (act[i]) {
#pragma unroll
      for (int k = 0; k < 4; ++k) {                          // 8-byte stores: one packed pair each
        reinterpret_cast<f32x2*>(red_g + row_in_pass * D + (lane_in_row + i * L) * 8)[k] = acc_g[i][k];
        reinterpret_cast<f32x2*>(red_b + row_in_pass * D + (lane_in_row + i * L) * 8)[k] = acc_b[i][k];
      }
    }
  __syncthreads();
  float* part = m.ws + (size_t)b.part * 2 * D;
  for (int c = threadIdx.x; c < D; c += kLnbThreads) {
    float a = 0.f, bb = 0.f;
    for (int g = 0; g < rpp; ++g) { a += red_g[g * D + c]; bb += red_b[g * D + c]; }
    part[c] = a;
    part[D + c] = bb;
  }
  // ---- last block of the member: add the parts in part order, write dgamma / dbeta, re-arm the ticket
  __shared__ int is_last;
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) is_last = atomicAdd(m.ticket, 1) == m.nparts - 1;
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  for (int c = threadIdx.x; c < D; c += kLnbThreads) {
    float a = 0.f, bb = 0.f;
    for (int p = 0; p < m.nparts; ++p) {
      a += __ldcg(m.ws + (size_t)p * 2 * D + c);
      bb += __ldcg(m.ws + (size_t)p * 2 * D + D + c);
    }
    if (m.dgamma) lnb_store_param<P_BF16>(m.dgamma, c, a);
    if (m.dbeta) lnb_store_param<P_BF16>(m.dbeta, c, bb);
  }
  if (threadIdx.x == 0) *m.ticket = 0;
}

// Rows wider than 512 elements (up to 2048, the forward kernel's limit): a WARP owns a row, lane l holds vectors
// l, l + 32, ... (<= 8) of x and dy packed in registers, statistics by full-warp butterflies as above; the column sums
// cannot stay in registers (128 per lane), so every warp accumulates into its own [2][D] fp32 strip of shared memory
// (a lane only ever touches its own columns: no conflicts, no synchronisation inside the row loop); gamma is staged
// once per block as fp32.  The block's 8 strips are then added in warp order -> workspace part -> same last-block
// reduction as the narrow path: bitwise reproducible.
constexpr int kLnbWideVpl = 8;
template <bool P_BF16>
__device__ __forceinline__ void lnb_block_wide(const LnbMember& m, const LnbBlock& b, float* smem) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  constexpr int kWarps = kLnbThreads / 32;
  const int D = m.nvec * 8;
  float* sgam = smem;                               // [D]
  float* acc = smem + D + (size_t)warp * 2 * D;     // this warp's [2][D]: dy * xhat, dy
  for (int c = threadIdx.x; c < D; c += kLnbThreads) {
    float g = 1.f;
    if (m.gamma != nullptr) g = P_BF16 ? __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(m.gamma)[c]) : reinterpret_cast<const float*>(m.gamma)[c];
    sgam[c] = g;
  }
  for (int c = lane; c < 2 * D; c += 32) acc[c] = 0.f;
  __syncthreads();
  const int4* xb = reinterpret_cast<const int4*>(m.x);
  const int4* dyb = reinterpret_cast<const int4*>(m.dy);
  int4* dxb = reinterpret_cast<int4*>(m.dx);
  for (int r = warp; r < b.nrows; r += kWarps) {
    int4 xs[kLnbWideVpl], ds[kLnbWideVpl];
#pragma unroll
    for (int i = 0; i < kLnbWideVpl; ++i) {
      xs[i] = ds[i] = make_int4(0, 0, 0, 0);
      if (lane + 32 * i < m.nvec) {
        xs[i] = __ldcs(xb + (int64_t)(b.row0 + r) * m.ldx16 + lane + 32 * i);
        ds[i] = __ldcs(dyb + (int64_t)(b.row0 + r) * m.lddy16 + lane + 32 * i);
      }
    }
    f32x2 s2 = 0ull, sg2 = 0ull, sgx2 = 0ull;
#pragma unroll
    for (int i = 0; i < kLnbWideVpl; ++i) {
      if (lane + 32 * i >= m.nvec) continue;
      const uint32_t* ux = reinterpret_cast<const uint32_t*>(&xs[i]);
      const uint32_t* ud = reinterpret_cast<const uint32_t*>(&ds[i]);
      const float4 g0 = *reinterpret_cast<const float4*>(sgam + (lane + 32 * i) * 8), g1 = *reinterpret_cast<const float4*>(sgam + (lane + 32 * i) * 8 + 4);
      const f32x2 gv[4] = {pk2(g0.x, g0.y), pk2(g0.z, g0.w), pk2(g1.x, g1.y), pk2(g1.z, g1.w)};
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const f32x2 xv = bf2_to_f2(ux[k]), g = mul2(bf2_to_f2(ud[k]), gv[k]);
        s2 = add2(s2, xv); sg2 = add2(sg2, g); sgx2 = fma2(g, xv, sgx2);
      }
    }
    const float s = lnb_rowsum<5>(sum2(s2)), sg = lnb_rowsum<5>(sum2(sg2));
    float sgx = lnb_rowsum<5>(sum2(sgx2));
    const float mu = s * m.inv_D;
    const f32x2 nmu2 = pk2(-mu, -mu);
    f32x2 q2 = 0ull;
#pragma unroll
    for (int i = 0; i < kLnbWideVpl; ++i) {
      if (lane + 32 * i >= m.nvec) continue;
      const uint32_t* ux = reinterpret_cast<const uint32_t*>(&xs[i]);
#pragma unroll
      for (int k = 0; k < 4; ++k) { const f32x2 d = add2(bf2_to_f2(ux[k]), nmu2); q2 = fma2(d, d, q2); }
    }
    const float q = lnb_rowsum<5>(sum2(q2));
    const float rstd = rsqrtf(q * m.inv_D + m.eps);
    sgx = rstd * (sgx - mu * sg);
    const float mg = sg * m.inv_D, mgx = sgx * m.inv_D;
    const f32x2 rstd2 = pk2(rstd, rstd), nmg2 = pk2(-mg, -mg), nmgx2 = pk2(-mgx, -mgx);
#pragma unroll
    for (int i = 0; i < kLnbWideVpl; ++i) {
      if (lane + 32 * i >= m.nvec) continue;
      const int col = (lane + 32 * i) * 8;
      const uint32_t* ux = reinterpret_cast<const uint32_t*>(&xs[i]);
      const uint32_t* ud = reinterpret_cast<const uint32_t*>(&ds[i]);
      const float4 g0 = *reinterpret_cast<const float4*>(sgam + col), g1 = *reinterpret_cast<const float4*>(sgam + col + 4);
      const f32x2 gv[4] = {pk2(g0.x, g0.y), pk2(g0.z, g0.w), pk2(g1.x, g1.y), pk2(g1.z, g1.w)};
      f32x2* ag = reinterpret_cast<f32x2*>(acc + col);
      f32x2* ab = reinterpret_cast<f32x2*>(acc + D + col);
      uint32_t o[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const f32x2 dyv = bf2_to_f2(ud[k]);
        const f32x2 xh = mul2(add2(bf2_to_f2(ux[k]), nmu2), rstd2);
        ag[k] = fma2(dyv, xh, ag[k]);
        ab[k] = add2(ab[k], dyv);
        o[k] = f2_to_bf2(mul2(fma2(xh, nmgx2, fma2(dyv, gv[k], nmg2)), rstd2));
      }
      __stcs(dxb + (int64_t)(b.row0 + r) * m.lddx16 + lane + 32 * i, make_int4((int)o[0], (int)o[1], (int)o[2], (int)o[3]));
    }
  }
  if (m.dgamma == nullptr && m.dbeta == nullptr) return;
  __syncthreads();
  float* part = m.ws + (size_t)b.part * 2 * D;
  for (int c = threadIdx.x; c < 2 * D; c += kLnbThreads) {
    float a = 0.f;
    for (int w = 0; w < kWarps; ++w) a += smem[D + (size_t)w * 2 * D + c];
    part[c] = a;
  }
  __shared__ int is_last_w;
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) is_last_w = atomicAdd(m.ticket, 1) == m.nparts - 1;
  __syncthreads();
  if (!is_last_w) return;
  __threadfence();
  for (int c = threadIdx.x; c < D; c += kLnbThreads) {
    float a = 0.f, bb = 0.f;
    for (int p = 0; p < m.nparts; ++p) {
      a += __ldcg(m.ws + (size_t)p * 2 * D + c);
      bb += __ldcg(m.ws + (size_t)p * 2 * D + D + c);
    }
    if (m.dgamma) lnb_store_param<P_BF16>(m.dgamma, c, a);
    if (m.dbeta) lnb_store_param<P_BF16>(m.dbeta, c, bb);
  }
  if (threadIdx.x == 0) *m.ticket = 0;
}

// Three instantiations: groups whose rows all fit one vector per lane (D <= 256) run 4 blocks per SM in 64
// registers; groups with rows up to 512 keep two vectors per lane and run 2 blocks per SM without spilling; groups
// with a member wider than that run one block per SM (the wide path's shared-memory strips, up to 136 KB).
template <bool P_BF16, int MAXVPL>
__global__ void __launch_bounds__(kLnbThreads, MAXVPL == 1 ? 4 : MAXVPL == 2 ? 2 : 1)
batched_layernorm_bwd_kernel(const LnbMember* __restrict__ members, const LnbBlock* __restrict__ blocks) {
  extern __shared__ __align__(16) float lnb_red[];      // narrow: 2 x rpp x D floats <= 32 KB; wide: (1 + 16) x D floats
  const LnbBlock b = blocks[blockIdx.x];
  const LnbMember m = members[b.member];
  if (MAXVPL > 2 && m.vpl > 2) {
    lnb_block_wide<P_BF16>(m, b, lnb_red);
  } else if (MAXVPL == 1 || m.vpl == 1) {
    switch (m.l_log2) {      // block-uniform
      case 0: lnb_block<P_BF16, 1, 0>(m, b, lnb_red); break;
      case 1: lnb_block<P_BF16, 1, 1>(m, b, lnb_red); break;
      case 2: lnb_block<P_BF16, 1, 2>(m, b, lnb_red); break;
      case 3: lnb_block<P_BF16, 1, 3>(m, b, lnb_red); break;
      case 4: lnb_block<P_BF16, 1, 4>(m, b, lnb_red); break;
      default: lnb_block<P_BF16, 1, 5>(m, b, lnb_red); break;
    }
  } else {
    lnb_block<P_BF16, 2, 5>(m, b, lnb_red);      // two vectors per lane only occur with full-warp rows
  }
}

cudaError_t launch_layernorm_bwd(const opt_plan* p, cudaStream_t s) {
  const char* base = static_cast<const char*>(p->dev_tables);
  auto* members = reinterpret_cast<const LnbMember*>(base + p->off0);
  auto* blocks = reinterpret_cast<const LnbBlock*>(base + p->off1);
  const int mv = p->nstages;      // max vectors per lane over the group (stored in nstages)
  if (p->param == OPT_BF16) {
    if (mv == 1) batched_layernorm_bwd_kernel<true, 1><<<p->grid, p->block, p->smem, s>>>(members, blocks);
    else if (mv == 2) batched_layernorm_bwd_kernel<true, 2><<<p->grid, p->block, p->smem, s>>>(members, blocks);
    else batched_layernorm_bwd_kernel<true, 8><<<p->grid, p->block, p->smem, s>>>(members, blocks);
  } else {
    if (mv == 1) batched_layernorm_bwd_kernel<false, 1><<<p->grid, p->block, p->smem, s>>>(members, blocks);
    else if (mv == 2) batched_layernorm_bwd_kernel<false, 2><<<p->grid, p->block, p->smem, s>>>(members, blocks);
    else batched_layernorm_bwd_kernel<false, 8><<<p->grid, p->block, p->smem, s>>>(members, blocks);
  }
  return cudaGetLastError();
}

}  // namespace optb

using namespace optb;

extern "C" opt_status opt_layernorm_bwd_plan_create(const opt_layernorm_bwd_member* members, int32_t n, opt_dtype io,
                                                    opt_dtype param, int device, opt_plan** plan) {
  if (plan) *plan = nullptr;
  if (!plan || !members) return fail(OPT_ERR_INVALID_ARG, "opt_layernorm_bwd_plan_create: NULL argument");
  if (n < 1 || n > 65535) return fail(OPT_ERR_INVALID_ARG, "n = %d outside [1, 65535]", n);
  if ((io != OPT_F32 && io != OPT_BF16) || (param != OPT_F32 && param != OPT_BF16)) return fail(OPT_ERR_INVALID_ARG, "bad dtype");
  if (io != OPT_BF16) return fail(OPT_ERR_UNSUPPORTED, "LayerNorm backward is implemented for bf16 activations only");
  const int pesz = elem_size(param);
  std::vector<Region> regions;
  std::vector<LnbMember> tab;
  std::vector<LnbBlock> blocks;
  std::vector<int64_t> ws_off;            // float offset of each member's partials in the workspace
  int64_t bytes = 0, ws_floats = 0;
  int max_wide_D = 0;
  // Rows per block of the register path: a block pays a prologue (kPD passes to fill its prefetch slots) and an
  // epilogue (column sums through shared memory, a workspace part, the ticket), so long blocks are cheaper per row --
  // configs[4]'s LayerNorm shapes: 64 KB of x per block 504 us, 128 KB 476 us, 256 KB 473 us -- as long as the group
  // still fills the machine: aim at >= kLnbTargetBlocks blocks (16 per SM of the 148-SM part: four waves of four
  // blocks per SM), between 64 KB and 256 KB of x per block.
  int64_t group_x_bytes = 0;
  for (int32_t i = 0; i < n; ++i)
    if (members[i].rows > 0 && members[i].D > 0) group_x_bytes += (int64_t)members[i].rows * members[i].D * 2;
  const int64_t block_x_bytes = std::min<int64_t>(262144, std::max<int64_t>(65536, group_x_bytes / kLnbTargetBlocks));
  for (int32_t i = 0; i < n; ++i) {
    const opt_layernorm_bwd_member& m = members[i];
    if (!m.x || !m.dy || !m.dx) return fail(OPT_ERR_INVALID_ARG, "member %d: NULL pointer", i);
    if (m.rows < 1 || m.D < 1) return fail(OPT_ERR_INVALID_ARG, "member %d: rows=%d D=%d must be >= 1", i, m.rows, m.D);
    if (!(m.eps >= 0.f)) return fail(OPT_ERR_INVALID_ARG, "member %d: eps must be >= 0", i);
    if (m.rows > 1 && (m.ldx < m.D || m.lddy < m.D || m.lddx < m.D)) return fail(OPT_ERR_INVALID_ARG, "member %d: row stride smaller than D", i);
    if (!aligned16(m.x) || !aligned16(m.dy) || !aligned16(m.dx) || !aligned16(m.gamma) || !aligned16(m.dgamma) || !aligned16(m.dbeta))
      return fail(OPT_ERR_ALIGNMENT, "member %d: pointers must be 16-byte aligned", i);
    if (m.D % 8) return fail(OPT_ERR_ALIGNMENT, "member %d: D=%d is not a multiple of 8", i, m.D);
    if (m.rows > 1 && (m.ldx % 8 || m.lddy % 8 || m.lddx % 8)) return fail(OPT_ERR_ALIGNMENT, "member %d: row strides must be multiples of 8 elements", i);
    const int nvec = m.D / 8;
    if (nvec > 32 * kLnbWideVpl) return fail(OPT_ERR_UNSUPPORTED, "member %d: D=%d exceeds the limit %d", i, m.D, 32 * kLnbWideVpl * 8);
    const bool wide = nvec > 32 * kLnbMaxVpl;           // a warp per row, column sums in shared memory
    regions.push_back({(uintptr_t)m.x, m.ldx * 2, (int64_t)m.D * 2, m.rows, false, i});
    regions.push_back({(uintptr_t)m.dy, m.lddy * 2, (int64_t)m.D * 2, m.rows, false, i});
    regions.push_back({(uintptr_t)m.dx, m.lddx * 2, (int64_t)m.D * 2, m.rows, true, i});
    if (m.gamma) regions.push_back({(uintptr_t)m.gamma, 0, (int64_t)m.D * pesz, 1, false, i});
    if (m.dgamma) regions.push_back({(uintptr_t)m.dgamma, 0, (int64_t)m.D * pesz, 1, true, i});
    if (m.dbeta) regions.push_back({(uintptr_t)m.dbeta, 0, (int64_t)m.D * pesz, 1, true, i});
    bytes += 3ll * m.rows * m.D * 2 + ((m.gamma ? 1 : 0) + (m.dgamma ? 1 : 0) + (m.dbeta ? 1 : 0)) * (int64_t)m.D * pesz;
    // lanes per row
    int ll = 0;
    while (ll < 5 && (1 << ll) < nvec) ++ll;                  // one vector per lane when the row fits a warp
    while (ll < 5 && (nvec + (1 << ll) - 1) / (1 << ll) > kLnbMaxVpl) ++ll;
    const int L = 1 << ll, vpl = (nvec + L - 1) / L, rpp = kLnbThreads >> ll;
    if (wide) max_wide_D = std::max(max_wide_D, m.D);
    // rows per block: whole passes, block_x_bytes of x per block (wide rows: ~512 KB, the block's shared-memory strips
    // are zeroed and reduced once per block)
    const int64_t passes = std::max<int64_t>(1, (wide ? 524288 : block_x_bytes) / ((int64_t)rpp * m.D * 2));
    const int64_t rpb = rpp * passes;
    const int32_t nparts = (int32_t)((m.rows + rpb - 1) / rpb);
    LnbMember t;
    memset(&t, 0, sizeof t);
    t.x = (const char*)m.x; t.dy = (const char*)m.dy; t.gamma = (const char*)m.gamma; t.dx = (char*)m.dx;
    t.dgamma = (char*)m.dgamma; t.dbeta = (char*)m.dbeta;
    t.ldx16 = m.ldx / 8; t.lddy16 = m.lddy / 8; t.lddx16 = m.lddx / 8;
    t.rows = m.rows; t.nvec = nvec; t.nparts = nparts; t.eps = m.eps; t.inv_D = 1.0f / (float)m.D; t.l_log2 = ll; t.vpl = vpl;
    tab.push_back(t);
    ws_off.push_back(ws_floats);
    ws_floats += (int64_t)nparts * 2 * m.D;
    for (int32_t part = 0; part < nparts; ++part)
      blocks.push_back({i, (int32_t)(part * rpb), (int32_t)std::min<int64_t>(rpb, m.rows - part * rpb), part});
  }
  if (opt_status st = check_independent(regions, /*allow_inplace_self=*/false)) return st;
  if (blocks.size() > (size_t)INT32_MAX) return fail(OPT_ERR_UNSUPPORTED, "too many work items");

  int num_sms = 0;
  DeviceGuard device_guard;      // the caller's current device is restored on return
  if (opt_status st = open_device(device, &num_sms)) return st;
  auto align_up = [](size_t x) { return (x + 255) & ~size_t(255); };
  opt_plan* p = new opt_plan();
  p->kind = kPlanLayerNormBwd; p->device = device; p->io = io; p->param = param; p->n_members = n;
  p->bytes = bytes; p->flops = 0;
  // workspace: per-block partial column sums (fully written before they are read: no initialisation needed)
  if (cudaMalloc(&p->workspace, std::max<int64_t>(ws_floats, 1) * sizeof(float)) != cudaSuccess) {
    cudaGetLastError(); delete p;
    return fail(OPT_ERR_CUDA, "cudaMalloc of the %lld-byte partial-sum workspace failed", (long long)ws_floats * 4);
  }
  p->off0 = 0;
  p->off1 = align_up(tab.size() * sizeof(LnbMember));
  p->off2 = p->off1 + align_up(blocks.size() * sizeof(LnbBlock));
  const size_t total = p->off2 + align_up((size_t)n * sizeof(int32_t));      // per-member tickets, zero-initialised
  std::vector<char> blob(total, 0);
  memcpy(blob.data() + p->off1, blocks.data(), blocks.size() * sizeof(LnbBlock));
  if (cudaMalloc(&p->dev_tables, total) != cudaSuccess) {
    cudaGetLastError(); cudaFree(p->workspace); delete p;
    return fail(OPT_ERR_CUDA, "cudaMalloc of the plan tables failed");
  }
  p->table_bytes = total;
  for (int32_t i = 0; i < n; ++i) {
    tab[i].ws = static_cast<float*>(p->workspace) + ws_off[i];
    tab[i].ticket = reinterpret_cast<int32_t*>(static_cast<char*>(p->dev_tables) + p->off2) + i;
  }
  memcpy(blob.data(), tab.data(), tab.size() * sizeof(LnbMember));
  cudaError_t e = cudaMemcpy(p->dev_tables, blob.data(), total, cudaMemcpyHostToDevice);
  int max_vpl = 1;
  for (const LnbMember& t : tab) max_vpl = std::max(max_vpl, t.vpl);
  max_vpl = max_vpl > 2 ? 8 : max_vpl;
  p->nstages = max_vpl;
  const void* fn = param == OPT_BF16 ? (max_vpl == 1 ? (const void*)batched_layernorm_bwd_kernel<true, 1> : max_vpl == 2 ? (const void*)batched_layernorm_bwd_kernel<true, 2> : (const void*)batched_layernorm_bwd_kernel<true, 8>)
                                     : (max_vpl == 1 ? (const void*)batched_layernorm_bwd_kernel<false, 1> : max_vpl == 2 ? (const void*)batched_layernorm_bwd_kernel<false, 2> : (const void*)batched_layernorm_bwd_kernel<false, 8>);
  // (a fixed maximum per instantiation, never a per-plan value: the attribute belongs to the kernel function)
  const int kWideSmemMax = (1 + 2 * (kLnbThreads / 32)) * 32 * kLnbWideVpl * 8 * (int)sizeof(float);      // 139264
  if (e == cudaSuccess) e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, max_vpl > 2 ? kWideSmemMax : kLnbSlotKB * 1024);
  if (e != cudaSuccess) {
    cudaFree(p->dev_tables); cudaFree(p->workspace); delete p;
    return fail(OPT_ERR_CUDA, "plan upload failed: %s", cudaGetErrorString(e));
  }
  p->grid = dim3((unsigned)blocks.size());
  p->block = dim3(kLnbThreads);
  p->smem = std::max<size_t>((size_t)kLnbSlotKB * 1024, (size_t)(1 + 2 * (kLnbThreads / 32)) * max_wide_D * sizeof(float));
  p->total_tiles = (int32_t)blocks.size();
  *plan = p;
  return OPT_OK;
}
