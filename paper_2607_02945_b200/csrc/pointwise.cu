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
#include <algorithm>
#include <map>
#include <tuple>

#include "common.h"

namespace optb {

struct PwGroup {
  const char* src;
  char* dst;
  int64_t lds16, ldd16;   // row stride in 16-byte vectors
  int32_t rows, W;        // rows; vectors per virtual row
  int32_t map_off;        // first map entry of this group
  int32_t tx_log2;        // log2(threads along the virtual row)
};
struct PwBlock { int32_t group, q0, r0, nrows; };

constexpr int kPwThreads = 256;
constexpr int kPwUnroll = 8;
constexpr int kFlatW = 256;          // vectors per row when a dense tensor is re-tiled
constexpr int kVecPerBlock = 4096;   // ~64 KB read + 64 KB written per block

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

template <bool BF16>
__global__ void __launch_bounds__(kPwThreads)
multi_pointwise_splitcat_kernel(const PwGroup* __restrict__ groups, const int2* __restrict__ vmap,
                                const PwBlock* __restrict__ blocks) {
  const PwBlock b = blocks[blockIdx.x];
  const PwGroup g = groups[b.group];
  const int tx = threadIdx.x & ((1 << g.tx_log2) - 1);
  const int ty = threadIdx.x >> g.tx_log2;
  const int ty_step = kPwThreads >> g.tx_log2;
  const int q = b.q0 + tx;
  if (q >= g.W) return;
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
    multi_pointwise_splitcat_kernel<true><<<p->grid, p->block, 0, s>>>(groups, vmap, blocks);
  else
    multi_pointwise_splitcat_kernel<false><<<p->grid, p->block, 0, s>>>(groups, vmap, blocks);
  return cudaGetLastError();
}

namespace {
struct CChunk {   // canonical chunk, in 16-byte vectors
  const char* src;
  char* dst;
  int64_t lds16, ldd16;
  int32_t rows, wv, op;
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
    if (c.op < OPT_PW_COPY || c.op > OPT_PW_SIGMOID) return fail(OPT_ERR_INVALID_ARG, "chunk %d: bad op %d", i, c.op);
    if (c.rows > 1 && (c.lds < c.width || c.ldd < c.width))
      return fail(OPT_ERR_INVALID_ARG, "chunk %d: row stride smaller than width", i);
    if (!aligned16(c.src) || !aligned16(c.dst)) return fail(OPT_ERR_ALIGNMENT, "chunk %d: pointers must be 16-byte aligned", i);
    if (c.width % V) return fail(OPT_ERR_ALIGNMENT, "chunk %d: width %d is not a multiple of %d", i, c.width, V);
    if (c.rows > 1 && (c.lds % V || c.ldd % V))
      return fail(OPT_ERR_ALIGNMENT, "chunk %d: row strides must be multiples of %d elements", i, V);
    regions.push_back({(uintptr_t)c.src, c.lds * esz, (int64_t)c.width * esz, c.rows, false, i});
    regions.push_back({(uintptr_t)c.dst, c.ldd * esz, (int64_t)c.width * esz, c.rows, true, i});
    bytes += 2ll * c.rows * c.width * esz;

    const int64_t wv = c.width / V;
    const bool dense = c.rows == 1 || (c.lds == c.width && c.ldd == c.width);
    if (dense) {
      const int64_t T = (int64_t)c.rows * wv;
      int64_t done = 0;
      if (T >= 2 * kFlatW) {
        const int64_t r2 = T / kFlatW;
        if (r2 > INT32_MAX) return fail(OPT_ERR_UNSUPPORTED, "chunk %d too large", i);
        cc.push_back({(const char*)c.src, (char*)c.dst, kFlatW, kFlatW, (int32_t)r2, kFlatW, c.op});
        done = r2 * kFlatW;
      }
      if (T > done)
        cc.push_back({(const char*)c.src + done * 16, (char*)c.dst + done * 16, 0, 0, 1, (int32_t)(T - done), c.op});
    } else {
      if (wv > INT32_MAX) return fail(OPT_ERR_UNSUPPORTED, "chunk %d too wide", i);
      cc.push_back({(const char*)c.src, (char*)c.dst, c.lds / V, c.ldd / V, c.rows, (int32_t)wv, c.op});
    }
  }
  if (opt_status st = check_independent(regions, /*allow_inplace_self=*/true)) return st;

  // ---- group canonical chunks by (rows, lds16, ldd16)
  std::map<std::tuple<int32_t, int64_t, int64_t>, std::vector<int>> buckets;
  for (int i = 0; i < (int)cc.size(); ++i)
    buckets[std::make_tuple(cc[i].rows, cc[i].lds16, cc[i].ldd16)].push_back(i);

  std::vector<PwGroup> groups;
  std::vector<int2> vmap;
  std::vector<PwBlock> blocks;
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
      // map entries, sorted by (op, dst)
      std::vector<int> order(ids.begin() + i0, ids.begin() + i1);
      std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return cc[a].op < cc[b].op; });
      for (int id : order) {
        const CChunk& c = cc[id];
        const int64_t so = (c.src - smin) / 16, dof = (c.dst - dmin) / 16;
        for (int32_t v = 0; v < c.wv; ++v) {
          int2 e;
          e.x = (int32_t)(so + v);
          e.y = (int32_t)((uint32_t)(dof + v) | ((uint32_t)c.op << 30));
          vmap.push_back(e);
        }
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
  if (blocks.size() > (size_t)INT32_MAX) return fail(OPT_ERR_UNSUPPORTED, "too many work items");

  int num_sms = 0;
  if (opt_status st = open_device(device, &num_sms)) return st;

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
  p->grid = dim3((unsigned)blocks.size());
  p->block = dim3(kPwThreads);
  p->total_tiles = (int32_t)blocks.size();
  p->bytes = bytes; p->flops = 0;
  *plan = p;
  return OPT_OK;
}
