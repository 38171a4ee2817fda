// multi_pointwise_splitcat: one launch for a whole group of pointwise ops
// and/or the gather-scatter copy that remains of a split->f->cat chain.
//
// What it computes (include/optimus_b200.h, opt_chunk; PAPER.md:292 batch_relu /
// batch_sigmoid / batch_aten_tanh / batch_detach; PAPER.md:150 + Listing 2 for
// the split/cat movement):  dst_j[r, 0:w_j] = op_j(src_j[r, 0:w_j]).
//
// Design (HBM-bound):
//   * the planner turns the chunk list into GROUPS of chunks that share
//     (rows, lds, ldd); inside a group the chunks' 16-byte vectors are laid side
//     by side into one VIRTUAL ROW and a per-vector map (src offset, dst offset,
//     op) is built once.  The map is sorted by op first and destination second:
//     warps are op-uniform (no divergence between relu/tanh/sigmoid chunks) and
//     stores walk the destination in order.
//   * a thread owns ONE virtual column and walks rows, 8 independent 16-byte
//     loads in flight (ld.global.cs), then 8 stores (st.global.cs).  No shared
//     memory, no intermediate tensor.
//   * dense tensors are re-tiled to [rows', 256 vectors] so the same path
//     covers the standalone multi-tensor form with a 2 KB map.
//   * STAGED mode, for groups made of many narrow column slices of one source
//     row span (the split->f->cat residue, configs[3]: 64-byte segments): a block
//     owns a tile of whole rows; one thread pulls the rows' source span into
//     shared memory with cp.async.bulk (TMA, full-line coalesced reads), threads
//     gather their vector from shared memory in op-sorted order, apply the op,
//     scatter it to the destination position in a second shared buffer, and the
//     rows leave with cp.async.bulk stores (full-line writes).  All the
//     scatter/gather happens on chip; HBM sees two streaming copies.
#include <algorithm>
#include <cstdlib>
#include <map>
#include <tuple>

#include <cuda_fp8.h>

#include "common.h"

namespace optb {

struct PwGroup {
  const char* src;
  char* dst;
  int64_t lds16, ldd16;   // row stride in 16-byte vectors
  int32_t rows, W;        // rows; vectors per virtual row
  int32_t map_off;        // first map entry of this group
  int32_t tx_log2;        // log2(threads along the virtual row)
  int32_t src_span;       // STAGED mode: vectors of one source row staged in smem (0 = direct mode)
  int32_t dst_span;       // STAGED mode: vectors of one destination row staged for a bulk store (0 = direct stores)
  int32_t tile_rows;      // STAGED mode: rows per block
  int32_t ext_op;         // EXT mode (0 = off): OPT_PW_CLAMP .. OPT_PW_SIGMOID_BWD, one chunk per group, no map
  const char* src2;       // EXT mode: second operand of the binary ops
  int64_t lds2_16;
  float p0, p1, p2;       // EXT mode: scalar parameters
  int32_t pad;
};
struct PwBlock { int32_t group, q0, r0, nrows; };

constexpr int kPwThreads = 256;
constexpr int kPwUnroll = 8;
constexpr int kFlatW = 256;          // vectors per row when a dense tensor is re-tiled
constexpr int kVecPerBlock = 4096;   // ~64 KB read + 64 KB written per block
constexpr int kStageBudget = 100 * 1024;  // STAGED mode: at most this much shared memory per block (3 source rows + 2 destination rows)
constexpr int kStageMaxSpan = 2048;       // STAGED mode: at most 32 KB per staged row
constexpr int kStageMaxAvgChunk = 32;     // STAGED mode only when the average segment is < 512 bytes

template <bool BF16, int OP>
__device__ __forceinline__ int4 pw_apply(int4 v) {
  if (OP == OPT_PW_COPY) return v;
  if (BF16) {
    uint32_t* u = reinterpret_cast<uint32_t*>(&v);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      if (OP == OPT_PW_RELU) {
        __nv_bfloat162 h = *reinterpret_cast<__nv_bfloat162*>(&u[i]);
        h = __hmax2_nan(h, __float2bfloat162_rn(0.f));      // NaN propagates, -0 -> +0
        u[i] = *reinterpret_cast<uint32_t*>(&h);
      } else {
        u[i] = pack_bf16x2(act_f32<true>(bf16_lo(u[i]), OP), act_f32<true>(bf16_hi(u[i]), OP));
      }
    }
  } else {
    float* f = reinterpret_cast<float*>(&v);
#pragma unroll
    for (int i = 0; i < 4; ++i) f[i] = act_f32<false>(f[i], OP);
  }
  return v;
}

template <bool BF16, int OP>
__device__ __forceinline__ void pw_rows(const int4* __restrict__ s, int4* __restrict__ d, int64_t lds, int64_t ldd,
                                        int r, int rend, int ty_step) {
  for (; r + (kPwUnroll - 1) * ty_step < rend; r += kPwUnroll * ty_step) {
    int4 v[kPwUnroll];
#pragma unroll
    for (int i = 0; i < kPwUnroll; ++i) v[i] = __ldcs(s + (int64_t)(r + i * ty_step) * lds);
#pragma unroll
    for (int i = 0; i < kPwUnroll; ++i) __stcs(d + (int64_t)(r + i * ty_step) * ldd, pw_apply<BF16, OP>(v[i]));
  }
  for (; r < rend; r += ty_step) __stcs(d + (int64_t)r * ldd, pw_apply<BF16, OP>(__ldcs(s + (int64_t)r * lds)));
}

// EXT mode: the remaining pointwise patterns of Table 1 -- batch_clamp, batch_nan_to_num
// (scalar parameters) and batch_aten_sub / div / mul (second operand).  fp32 arithmetic, one rounding.
__device__ __forceinline__ float pw_ext_scalar(float x, float y, int op, float p0, float p1, float p2) {
  switch (op) {
    case OPT_PW_CLAMP: return x != x ? x : fminf(fmaxf(x, p0), p1);            // torch.clamp: min(max(x, lo), hi), NaN stays
    case OPT_PW_NAN_TO_NUM: return x != x ? p0 : (fabsf(x) == INFINITY ? (x > 0.f ? p1 : p2) : x);
    case OPT_PW_SUB: return x - y;
    case OPT_PW_DIV: return x / y;                                             // IEEE division (no fast-math)
    case OPT_PW_RELU_BWD: return y <= 0.f ? 0.f : x;                           // gradient where the forward value is > 0
    case OPT_PW_TANH_BWD: return x * fmaf(-y, y, 1.f);                         // y = tanh(z) stored: dz = dy (1 - y^2)
    case OPT_PW_SIGMOID_BWD: return x * ((1.f - y) * y);                       // y = sigmoid(z) stored: dz = dy (1 - y) y
    default: return x * y;                                                     // OPT_PW_MUL
  }
}
template <bool BF16>
__device__ __forceinline__ int4 pw_ext_apply(int4 a, int4 b, int op, float p0, float p1, float p2) {
  if (BF16) {
    uint32_t* ua = reinterpret_cast<uint32_t*>(&a);
    const uint32_t* ub = reinterpret_cast<const uint32_t*>(&b);
#pragma unroll
    for (int i = 0; i < 4; ++i)
      ua[i] = pack_bf16x2(pw_ext_scalar(bf16_lo(ua[i]), bf16_lo(ub[i]), op, p0, p1, p2),
                          pw_ext_scalar(bf16_hi(ua[i]), bf16_hi(ub[i]), op, p0, p1, p2));
  } else {
    float* fa = reinterpret_cast<float*>(&a);
    const float* fb = reinterpret_cast<const float*>(&b);
#pragma unroll
    for (int i = 0; i < 4; ++i) fa[i] = pw_ext_scalar(fa[i], fb[i], op, p0, p1, p2);
  }
  return a;
}
// FP8 E4M3 quantise / dequantise of saved activations (activation_quantization_aten_pass): the
// bf16 side moves 16-byte vectors, the fp8 side the matching 8-byte vectors; p0 is the scale.  Saturating RNE, NaN -> NaN.
__device__ __forceinline__ int2 pw_quant_e4m3(int4 v, float scale) {
  return make_int2((int)quant4_e4m3((uint32_t)v.x, (uint32_t)v.y, scale), (int)quant4_e4m3((uint32_t)v.z, (uint32_t)v.w, scale));
}
__device__ __forceinline__ int4 pw_dequant_e4m3(int2 v, float scale) {
  const uint32_t w[2] = {(uint32_t)v.x, (uint32_t)v.y};
  uint32_t o[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const __half2_raw h = __nv_cvt_fp8x2_to_halfraw2((__nv_fp8x2_storage_t)((w[i >> 1] >> (16 * (i & 1))) & 0xFFFFu), __NV_E4M3);
    const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&h));
    o[i] = pack_bf16x2(f.x * scale, f.y * scale);
  }
  return make_int4((int)o[0], (int)o[1], (int)o[2], (int)o[3]);
}
__device__ __forceinline__ void pw_fp8_rows(const PwGroup& g, int q, int r, int rend, int ty_step) {
  constexpr int U = 4;
  if (g.ext_op == OPT_PW_QUANT_E4M3) {
    const int4* s = reinterpret_cast<const int4*>(g.src) + q;
    int2* d = reinterpret_cast<int2*>(g.dst) + q;
    for (; r + (U - 1) * ty_step < rend; r += U * ty_step) {
      int4 v[U];
#pragma unroll
      for (int i = 0; i < U; ++i) v[i] = __ldcs(s + (int64_t)(r + i * ty_step) * g.lds16);
#pragma unroll
      for (int i = 0; i < U; ++i) __stcs(d + (int64_t)(r + i * ty_step) * g.ldd16, pw_quant_e4m3(v[i], g.p0));
    }
    for (; r < rend; r += ty_step) __stcs(d + (int64_t)r * g.ldd16, pw_quant_e4m3(__ldcs(s + (int64_t)r * g.lds16), g.p0));
  } else {
    const int2* s = reinterpret_cast<const int2*>(g.src) + q;
    int4* d = reinterpret_cast<int4*>(g.dst) + q;
    for (; r + (U - 1) * ty_step < rend; r += U * ty_step) {
      int2 v[U];
#pragma unroll
      for (int i = 0; i < U; ++i) v[i] = __ldcs(s + (int64_t)(r + i * ty_step) * g.lds16);
#pragma unroll
      for (int i = 0; i < U; ++i) __stcs(d + (int64_t)(r + i * ty_step) * g.ldd16, pw_dequant_e4m3(v[i], g.p0));
    }
    for (; r < rend; r += ty_step) __stcs(d + (int64_t)r * g.ldd16, pw_dequant_e4m3(__ldcs(s + (int64_t)r * g.lds16), g.p0));
  }
}

template <bool BF16>
__device__ __forceinline__ void pw_ext_rows(const PwGroup& g, int q, int r, int rend, int ty_step) {
  const int4* s = reinterpret_cast<const int4*>(g.src) + q;
  const int4* s2 = g.src2 ? reinterpret_cast<const int4*>(g.src2) + q : nullptr;
  int4* d = reinterpret_cast<int4*>(g.dst) + q;
  constexpr int U = 4;
  for (; r + (U - 1) * ty_step < rend; r += U * ty_step) {
    int4 v[U], w[U];
#pragma unroll
    for (int i = 0; i < U; ++i) {
      v[i] = __ldcs(s + (int64_t)(r + i * ty_step) * g.lds16);
      w[i] = s2 ? __ldcs(s2 + (int64_t)(r + i * ty_step) * g.lds2_16) : make_int4(0, 0, 0, 0);
    }
#pragma unroll
    for (int i = 0; i < U; ++i)
      __stcs(d + (int64_t)(r + i * ty_step) * g.ldd16, pw_ext_apply<BF16>(v[i], w[i], g.ext_op, g.p0, g.p1, g.p2));
  }
  for (; r < rend; r += ty_step) {
    const int4 v = __ldcs(s + (int64_t)r * g.lds16);
    const int4 w = s2 ? __ldcs(s2 + (int64_t)r * g.lds2_16) : make_int4(0, 0, 0, 0);
    __stcs(d + (int64_t)r * g.ldd16, pw_ext_apply<BF16>(v, w, g.ext_op, g.p0, g.p1, g.p2));
  }
}

__device__ __forceinline__ uint32_t pw_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// STAGED mode: rows [r0, r0+nrows) of group g, software-pipelined inside the block.
//   smem = kPwInStages source rows (ring) + 2 destination rows (double buffer, only when dst_span != 0).
//   Thread 0 keeps kPwInStages-1 row loads (cp.async.bulk) in flight; every thread owns up to 4 virtual
//   columns whose map entries live in registers for the whole block; per row: gather from the staged
//   source row, apply, scatter into the staged destination row, which leaves with one bulk store.
constexpr int kPwInStages = 3;

template <bool BF16>
__device__ __forceinline__ int4 pw_apply_rt(int4 v, int op) {
  switch (op) {   // warp-uniform except at op boundaries of the virtual row
    case OPT_PW_COPY: return v;
    case OPT_PW_RELU: return pw_apply<BF16, OPT_PW_RELU>(v);
    case OPT_PW_TANH: return pw_apply<BF16, OPT_PW_TANH>(v);
    default:          return pw_apply<BF16, OPT_PW_SIGMOID>(v);
  }
}

template <bool BF16>
__device__ __forceinline__ void pw_staged_tile(const PwGroup& g, const int2* __restrict__ vmap, int r0, int nrows) {
  extern __shared__ __align__(128) uint8_t pw_smem[];
  __shared__ __align__(8) uint64_t bar_storage[kPwInStages];
  const uint32_t in_bytes = (uint32_t)g.src_span * 16u, out_bytes = (uint32_t)g.dst_span * 16u;
  const uint32_t sin0 = pw_smem_u32(pw_smem);
  const uint32_t sout0 = sin0 + kPwInStages * in_bytes;
  const bool staged_out = g.dst_span != 0;
  auto bar = [&](int s) { return pw_smem_u32(&bar_storage[s]); };
  auto load_row = [&](int r) {            // thread 0 only
    const int s = r % kPwInStages;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar(s)), "r"(in_bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(sin0 + (uint32_t)s * in_bytes), "l"(g.src + ((int64_t)(r0 + r) * g.lds16) * 16), "r"(in_bytes), "r"(bar(s)) : "memory");
  };
  if (threadIdx.x == 0) {
    for (int s = 0; s < kPwInStages; ++s) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar(s)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    for (int r = 0; r < kPwInStages - 1 && r < nrows; ++r) load_row(r);
  }
  // this thread's map entries (up to 4 virtual columns), fetched while the first rows are in flight
  constexpr int kPre = 4;
  int2 pre[kPre];
#pragma unroll
  for (int k = 0; k < kPre; ++k) {
    const int q = threadIdx.x + k * kPwThreads;
    pre[k] = q < g.W ? __ldg(vmap + g.map_off + q) : make_int2(0, 0);
  }
  __syncthreads();                       // barriers initialised before anyone polls them
  for (int r = 0; r < nrows; ++r) {
    const int s = r % kPwInStages;
    const uint32_t parity = (uint32_t)(r / kPwInStages) & 1u;
    {
      uint32_t done = 0;
      while (!done)
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(bar(s)), "r"(parity) : "memory");
    }
    // the bulk store that last used this row's destination buffer (row r-2) has read it
    if (staged_out && threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
    __syncthreads();                     // + every thread is done with source row r-1: its stage can be refilled
    if (threadIdx.x == 0 && r + kPwInStages - 1 < nrows) load_row(r + kPwInStages - 1);
    const uint32_t sin = sin0 + (uint32_t)s * in_bytes;
    const uint32_t sout = sout0 + (uint32_t)(r & 1) * out_bytes;
    int4* grow = reinterpret_cast<int4*>(g.dst) + (int64_t)(r0 + r) * g.ldd16;
    auto column = [&](const int2 m) {
      int4 v;
      asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(sin + (uint32_t)m.x * 16u) : "memory");
      v = pw_apply_rt<BF16>(v, (int)((uint32_t)m.y >> 30));
      const uint32_t dof = (uint32_t)m.y & 0x3FFFFFFFu;
      if (staged_out)
        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(sout + dof * 16u), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
      else
        __stcs(grow + dof, v);
    };
#pragma unroll
    for (int k = 0; k < kPre; ++k)
      if (threadIdx.x + k * kPwThreads < g.W) column(pre[k]);
    for (int q = threadIdx.x + kPre * kPwThreads; q < g.W; q += kPwThreads) column(__ldg(vmap + g.map_off + q));
    if (staged_out) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // st.shared results -> visible to the bulk-copy engine
      __syncthreads();
      if (threadIdx.x == 0) {
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                     ::"l"(g.dst + ((int64_t)(r0 + r) * g.ldd16) * 16), "r"(sout), "r"(out_bytes) : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
      }
    }
  }
  if (staged_out && threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // smem outlives the stores' reads
}

constexpr int kPwMinBlocks = 6;
template <bool BF16>
__global__ void __launch_bounds__(kPwThreads, kPwMinBlocks)
multi_pointwise_splitcat_kernel(const PwGroup* __restrict__ groups, const int2* __restrict__ vmap,
                                const PwBlock* __restrict__ blocks) {
  const PwBlock b = blocks[blockIdx.x];
  const PwGroup g = groups[b.group];
  if (g.src_span) {                       // block-uniform
    pw_staged_tile<BF16>(g, vmap, b.r0, b.nrows);
    return;
  }
  const int tx = threadIdx.x & ((1 << g.tx_log2) - 1);
  const int ty = threadIdx.x >> g.tx_log2;
  const int ty_step = kPwThreads >> g.tx_log2;
  const int q = b.q0 + tx;
  if (q >= g.W) return;
  if (g.ext_op) {                         // block-uniform: one chunk, no map
    if (g.ext_op == OPT_PW_QUANT_E4M3 || g.ext_op == OPT_PW_DEQUANT_E4M3) pw_fp8_rows(g, q, b.r0 + ty, b.r0 + b.nrows, ty_step);
    else pw_ext_rows<BF16>(g, q, b.r0 + ty, b.r0 + b.nrows, ty_step);
    return;
  }
  const int2 m = __ldg(vmap + g.map_off + q);
  const int op = (int)((uint32_t)m.y >> 30);
  const int4* s = reinterpret_cast<const int4*>(g.src) + m.x;
  int4* d = reinterpret_cast<int4*>(g.dst) + (m.y & 0x3FFFFFFF);
  const int r = b.r0 + ty, rend = b.r0 + b.nrows;
  switch (op) {   // warp-uniform except at the (at most 3) op boundaries of a virtual row
    case OPT_PW_COPY: pw_rows<BF16, OPT_PW_COPY>(s, d, g.lds16, g.ldd16, r, rend, ty_step); break;
    case OPT_PW_RELU: pw_rows<BF16, OPT_PW_RELU>(s, d, g.lds16, g.ldd16, r, rend, ty_step); break;
    case OPT_PW_TANH: pw_rows<BF16, OPT_PW_TANH>(s, d, g.lds16, g.ldd16, r, rend, ty_step); break;
    default:          pw_rows<BF16, OPT_PW_SIGMOID>(s, d, g.lds16, g.ldd16, r, rend, ty_step); break;
  }
}

cudaError_t launch_pointwise(const opt_plan* p, cudaStream_t s) {
  const char* base = static_cast<const char*>(p->dev_tables);
  auto* groups = reinterpret_cast<const PwGroup*>(base + p->off0);
  auto* vmap = reinterpret_cast<const int2*>(base + p->off1);
  auto* blocks = reinterpret_cast<const PwBlock*>(base + p->off2);
  if (p->io == OPT_BF16)
    multi_pointwise_splitcat_kernel<true><<<p->grid, p->block, p->smem, s>>>(groups, vmap, blocks);
  else
    multi_pointwise_splitcat_kernel<false><<<p->grid, p->block, p->smem, s>>>(groups, vmap, blocks);
  return cudaGetLastError();
}

namespace {
struct CChunk {   // canonical chunk, in 16-byte vectors
  const char* src;
  char* dst;
  int64_t lds16, ldd16;
  int32_t rows, wv, op;
  const char* src2 = nullptr;     // EXT ops only
  int64_t lds2_16 = 0;
  float p0 = 0.f, p1 = 0.f, p2 = 0.f;
};
}  // namespace

}  // namespace optb

using namespace optb;

extern "C" opt_status opt_pointwise_plan_create(const opt_chunk* chunks, int32_t n, opt_dtype io, int device,
                                                opt_plan** plan) {
  if (plan) *plan = nullptr;
  if (!plan || !chunks) return fail(OPT_ERR_INVALID_ARG, "opt_pointwise_plan_create: NULL argument");
  if (n < 1 || n > 65535) return fail(OPT_ERR_INVALID_ARG, "n = %d outside [1, 65535]", n);
  if (io != OPT_F32 && io != OPT_BF16) return fail(OPT_ERR_INVALID_ARG, "bad io dtype %d", (int)io);
  const int esz = elem_size(io), V = vec_elems(io);
  std::vector<Region> regions;
  std::vector<CChunk> cc;
  int64_t bytes = 0;
  for (int32_t i = 0; i < n; ++i) {
    const opt_chunk& c = chunks[i];
    if (!c.src || !c.dst) return fail(OPT_ERR_INVALID_ARG, "chunk %d: NULL pointer", i);
    if (c.rows < 1 || c.width < 1) return fail(OPT_ERR_INVALID_ARG, "chunk %d: rows=%d width=%d must be >= 1", i, c.rows, c.width);
    if (c.op < OPT_PW_COPY || c.op > OPT_PW_SIGMOID_BWD) return fail(OPT_ERR_INVALID_ARG, "chunk %d: bad op %d", i, c.op);
    const bool ext = c.op >= OPT_PW_CLAMP, binary = (c.op >= OPT_PW_SUB && c.op <= OPT_PW_MUL) || c.op >= OPT_PW_RELU_BWD;
    const bool fp8 = c.op == OPT_PW_QUANT_E4M3 || c.op == OPT_PW_DEQUANT_E4M3;
    if (fp8 && io != OPT_BF16) return fail(OPT_ERR_UNSUPPORTED, "chunk %d: FP8 quantisation is implemented for bf16 activations only", i);
    // element sizes of the two sides: quantise writes fp8, dequantise reads fp8
    const int s_esz = c.op == OPT_PW_DEQUANT_E4M3 ? 1 : esz, d_esz = c.op == OPT_PW_QUANT_E4M3 ? 1 : esz;
    if (binary) {
      if (!c.src2) return fail(OPT_ERR_INVALID_ARG, "chunk %d: binary op %d needs src2", i, c.op);
      if (c.rows > 1 && c.lds2 < c.width) return fail(OPT_ERR_INVALID_ARG, "chunk %d: row stride of src2 smaller than width", i);
      if (!aligned16(c.src2)) return fail(OPT_ERR_ALIGNMENT, "chunk %d: pointers must be 16-byte aligned", i);
      if (c.rows > 1 && c.lds2 % V) return fail(OPT_ERR_ALIGNMENT, "chunk %d: row strides must be multiples of %d elements", i, V);
    }
    if (c.rows > 1 && (c.lds < c.width || c.ldd < c.width))
      return fail(OPT_ERR_INVALID_ARG, "chunk %d: row stride smaller than width", i);
    if (!aligned16(c.src) || !aligned16(c.dst)) return fail(OPT_ERR_ALIGNMENT, "chunk %d: pointers must be 16-byte aligned", i);
    if (c.width % V) return fail(OPT_ERR_ALIGNMENT, "chunk %d: width %d is not a multiple of %d", i, c.width, V);
    if (c.rows > 1 && (c.lds % V || c.ldd % V))
      return fail(OPT_ERR_ALIGNMENT, "chunk %d: row strides must be multiples of %d elements", i, V);
    regions.push_back({(uintptr_t)c.src, c.lds * s_esz, (int64_t)c.width * s_esz, c.rows, false, i});
    regions.push_back({(uintptr_t)c.dst, c.ldd * d_esz, (int64_t)c.width * d_esz, c.rows, true, i});
    if (binary) regions.push_back({(uintptr_t)c.src2, c.lds2 * esz, (int64_t)c.width * esz, c.rows, false, i});
    bytes += (int64_t)c.rows * c.width * (s_esz + d_esz + (binary ? esz : 0));

    const int64_t wv = c.width / V;
    const bool dense = c.rows == 1 || (c.lds == c.width && c.ldd == c.width && (!binary || c.lds2 == c.width));
    const size_t cc0 = cc.size();
    if (dense) {
      const int64_t T = (int64_t)c.rows * wv;
      int64_t done = 0;
      if (T >= 2 * kFlatW) {
        const int64_t r2 = T / kFlatW;
        if (r2 > INT32_MAX) return fail(OPT_ERR_UNSUPPORTED, "chunk %d too large", i);
        cc.push_back({(const char*)c.src, (char*)c.dst, kFlatW, kFlatW, (int32_t)r2, kFlatW, c.op});
        done = r2 * kFlatW;
      }
      if (T > done)       // (a vector is 8 elements on both sides: 16 bytes of bf16 / fp32x4, 8 bytes of fp8)
        cc.push_back({(const char*)c.src + done * (c.op == OPT_PW_DEQUANT_E4M3 ? 8 : 16),
                      (char*)c.dst + done * (c.op == OPT_PW_QUANT_E4M3 ? 8 : 16), 0, 0, 1, (int32_t)(T - done), c.op});
    } else {
      if (wv > INT32_MAX) return fail(OPT_ERR_UNSUPPORTED, "chunk %d too wide", i);
      cc.push_back({(const char*)c.src, (char*)c.dst, c.lds / V, c.ldd / V, c.rows, (int32_t)wv, c.op});
    }
    if (ext)                                   // same re-tiling for the second operand; scalars ride along
      for (size_t k = cc0; k < cc.size(); ++k) {
        CChunk& e = cc[k];
        if (binary) {
          e.src2 = (const char*)c.src2 + (e.src - (const char*)c.src);     // dense pieces: same byte offset
          e.lds2_16 = dense ? e.lds16 : c.lds2 / V;
        }
        e.p0 = c.p0; e.p1 = c.p1; e.p2 = c.p2;
      }
  }
  if (opt_status st = check_independent(regions, /*allow_inplace_self=*/true)) return st;
  int num_sms = 0;
  DeviceGuard device_guard;      // the caller's current device is restored on return
  if (opt_status st = open_device(device, &num_sms)) return st;

  // ---- group canonical chunks by (rows, lds16, ldd16)
  std::map<std::tuple<int32_t, int64_t, int64_t>, std::vector<int>> buckets;
  std::vector<int> ext_ids;
  for (int i = 0; i < (int)cc.size(); ++i) {
    if (cc[i].op >= OPT_PW_CLAMP) ext_ids.push_back(i);                 // EXT mode: one group per chunk, no map
    else buckets[std::make_tuple(cc[i].rows, cc[i].lds16, cc[i].ldd16)].push_back(i);
  }

  std::vector<PwGroup> groups;
  std::vector<int2> vmap;
  std::vector<PwBlock> blocks;
  size_t smem_needed = 0;
  for (auto& kv : buckets) {
    std::vector<int>& ids = kv.second;
    std::sort(ids.begin(), ids.end(), [&](int a, int b) { return cc[a].dst < cc[b].dst; });
    size_t i0 = 0;
    while (i0 < ids.size()) {
      // greedy: extend the group while offsets from the group's bases fit the map encoding
      const char* smin = cc[ids[i0]].src;
      const char* smax = smin;
      char* dmin = cc[ids[i0]].dst;
      int64_t W = 0;
      size_t i1 = i0;
      while (i1 < ids.size()) {
        const CChunk& c = cc[ids[i1]];
        const char* nsmin = std::min(smin, c.src);
        const char* nsmax = std::max(smax, c.src + (int64_t)c.wv * 16);
        const int64_t dspan = (c.dst + (int64_t)c.wv * 16 - dmin) / 16;
        if (i1 > i0 && ((nsmax - nsmin) / 16 >= (1ll << 31) || dspan >= (1ll << 30) || W + c.wv > (1 << 24))) break;
        smin = nsmin; smax = nsmax; W += c.wv; ++i1;
      }
      if ((smax - smin) / 16 >= (1ll << 31) || W > INT32_MAX)
        return fail(OPT_ERR_UNSUPPORTED, "a single chunk spans more than 32 GB");
      PwGroup g;
      g.src = smin; g.dst = dmin;
      g.lds16 = std::get<1>(kv.first); g.ldd16 = std::get<2>(kv.first);
      g.rows = std::get<0>(kv.first); g.W = (int32_t)W;
      g.map_off = (int32_t)vmap.size();
      int txl = 0;
      while ((1 << txl) < W && txl < 8) ++txl;
      g.tx_log2 = txl;
      g.src_span = g.dst_span = g.tile_rows = g.pad = 0;
      g.ext_op = 0; g.src2 = nullptr; g.lds2_16 = 0; g.p0 = g.p1 = g.p2 = 0.f;
      // map entries, sorted by (op, dst)
      std::vector<int> order(ids.begin() + i0, ids.begin() + i1);
      std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return cc[a].op < cc[b].op; });
      char* dmax = dmin;
      bool self_inplace = false;
      for (int id : order) {
        const CChunk& c = cc[id];
        const int64_t so = (c.src - smin) / 16, dof = (c.dst - dmin) / 16;
        dmax = std::max(dmax, c.dst + (int64_t)c.wv * 16);
        self_inplace |= (c.src == c.dst);
        for (int32_t v = 0; v < c.wv; ++v) {
          int2 e;
          e.x = (int32_t)(so + v);
          e.y = (int32_t)((uint32_t)(dof + v) | ((uint32_t)c.op << 30));
          vmap.push_back(e);
        }
      }
      // STAGED mode: many narrow slices of one compact source row span (split -> f -> cat residue)
      const int64_t sspan = (smax - smin) / 16, dspan = (dmax - dmin) / 16;
      const int64_t nch = (int64_t)(i1 - i0);
      const bool rows_disjoint = g.rows == 1 || (sspan <= g.lds16 && dspan <= g.ldd16);
      if (nch > 1 && W < nch * kStageMaxAvgChunk && rows_disjoint && sspan <= kStageMaxSpan && sspan <= W + W / 4) {
        g.src_span = (int32_t)sspan;
        // rows leave through a bulk store only if the chunks tile the destination span without holes
        // (otherwise the store would clobber bytes the group does not own) and nothing is in place
        if (dspan == W && dspan <= kStageMaxSpan && !self_inplace) g.dst_span = (int32_t)dspan;
        // one wave of fat blocks: rows split evenly over the resident block slots (2 per SM), each block
        // pipelines its rows through a 3-stage source ring and a double-buffered destination row.  Two blocks
        // per SM only fit while a block stays within kStageBudget: wide rows give up the staged destination
        // row (direct 16-byte stores instead of the bulk store), which always fits (3 x 32 KB).
        int64_t need = ((int64_t)kPwInStages * g.src_span + 2 * (int64_t)g.dst_span) * 16;
        if (need > kStageBudget) { g.dst_span = 0; need = (int64_t)kPwInStages * g.src_span * 16; }
        static_assert((int64_t)kPwInStages * kStageMaxSpan * 16 <= kStageBudget, "a staged source ring must fit the budget");
        const int64_t slots = 2 * (int64_t)num_sms;
        g.tile_rows = (int32_t)std::max<int64_t>(std::min<int64_t>(4, g.rows), (g.rows + slots - 1) / slots);
        smem_needed = std::max<size_t>(smem_needed, (size_t)need);
        for (int64_t r0 = 0; r0 < g.rows; r0 += g.tile_rows)
          blocks.push_back({(int32_t)groups.size(), 0, (int32_t)r0, (int32_t)std::min<int64_t>(g.tile_rows, g.rows - r0)});
        groups.push_back(g);
        i0 = i1;
        continue;
      }
      // work items
      const int TX = 1 << txl, TY = kPwThreads / TX;
      int64_t rb = kVecPerBlock / std::min<int64_t>(W, TX);
      rb = std::max<int64_t>(TY, std::min<int64_t>(rb, g.rows));
      rb = (rb + TY - 1) / TY * TY;
      for (int64_t q0 = 0; q0 < W; q0 += TX)
        for (int64_t r0 = 0; r0 < g.rows; r0 += rb)
          blocks.push_back({(int32_t)groups.size(), (int32_t)q0, (int32_t)r0, (int32_t)std::min<int64_t>(rb, g.rows - r0)});
      groups.push_back(g);
      i0 = i1;
    }
  }
  for (int id : ext_ids) {
    const CChunk& c = cc[id];
    PwGroup g;
    memset(&g, 0, sizeof g);
    g.src = c.src; g.dst = c.dst; g.lds16 = c.lds16; g.ldd16 = c.ldd16; g.rows = c.rows; g.W = c.wv;
    g.map_off = 0;
    int txl = 0;
    while ((1 << txl) < c.wv && txl < 8) ++txl;
    g.tx_log2 = txl;
    g.ext_op = c.op; g.src2 = c.src2; g.lds2_16 = c.lds2_16; g.p0 = c.p0; g.p1 = c.p1; g.p2 = c.p2;
    const int TX = 1 << txl, TY = kPwThreads / TX;
    int64_t rb = kVecPerBlock / std::min<int64_t>(c.wv, TX);
    rb = std::max<int64_t>(TY, std::min<int64_t>(rb, g.rows));
    rb = (rb + TY - 1) / TY * TY;
    for (int64_t q0 = 0; q0 < c.wv; q0 += TX)
      for (int64_t r0 = 0; r0 < g.rows; r0 += rb)
        blocks.push_back({(int32_t)groups.size(), (int32_t)q0, (int32_t)r0, (int32_t)std::min<int64_t>(rb, g.rows - r0)});
    groups.push_back(g);
  }
  if (blocks.size() > (size_t)INT32_MAX) return fail(OPT_ERR_UNSUPPORTED, "too many work items");

  auto align_up = [](size_t x) { return (x + 255) & ~size_t(255); };
  opt_plan* p = new opt_plan();
  p->kind = kPlanPointwise; p->device = device; p->io = io; p->n_members = n;
  p->off0 = 0;
  p->off1 = align_up(groups.size() * sizeof(PwGroup));
  p->off2 = p->off1 + align_up(vmap.size() * sizeof(int2));
  const size_t total = p->off2 + align_up(blocks.size() * sizeof(PwBlock));
  std::vector<char> blob(total, 0);
  memcpy(blob.data() + p->off0, groups.data(), groups.size() * sizeof(PwGroup));
  memcpy(blob.data() + p->off1, vmap.data(), vmap.size() * sizeof(int2));
  memcpy(blob.data() + p->off2, blocks.data(), blocks.size() * sizeof(PwBlock));
  if (opt_status st = upload_tables(p, blob.data(), total)) { delete p; return st; }
  if (smem_needed > 48 * 1024) {
    // per kernel FUNCTION, not per plan (the last call wins): always the fixed budget, so that a later, smaller
    // plan never lowers the limit under a live, larger one
    cudaError_t e = io == OPT_BF16
        ? cudaFuncSetAttribute(multi_pointwise_splitcat_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kStageBudget)
        : cudaFuncSetAttribute(multi_pointwise_splitcat_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kStageBudget);
    if (e != cudaSuccess) {
      cudaFree(p->dev_tables); delete p;
      return fail(OPT_ERR_CUDA, "cudaFuncSetAttribute(max dynamic smem %zu) failed: %s", smem_needed, cudaGetErrorString(e));
    }
  }
  p->smem = smem_needed;
  p->grid = dim3((unsigned)blocks.size());
  p->block = dim3(kPwThreads);
  p->total_tiles = (int32_t)blocks.size();
  p->bytes = bytes; p->flops = 0;
  *plan = p;
  return OPT_OK;
}
