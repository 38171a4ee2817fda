// opt_bias_grad_noalloc: the bias gradient of ONE Linear layer, db[n] = sum over m of dZ[m, n]
// (PAPER.md:292 batch_linear_post_grad, PAPER.md:437 training; include/optimus_b200.h), for callers that cannot
// call cudaMalloc -- code under CUDA-graph capture, tight serving loops, harnesses that forbid allocation.
//
// The planned path (bias_grad.cu, opt_bias_grad_plan_create) keeps its per-part partial sums and tickets in a
// cudaMalloc'ed plan workspace.  This entry point allocates NOTHING: its scratch is the file-scope device array
// g_na_scratch below (1 MiB + 256 B, held by every GPU that loads the library until the process exits), which bounds
// the problem: N <= OPT_NOALLOC_BIAS_GRAD_MAX_N.  Host code never uses the array's NAME as a pointer (on the host it
// is a stand-in, not a device address): once per device, with that device current, cudaGetSymbolAddress gives the
// device address, which is passed to the kernel.
//
// Every call shares the array: calls that overlap on the GPU (two streams, two threads) RACE on it; calls on one
// stream are ordered and safe.  The array keeps the last call's contents: the partial sums are fully overwritten
// before they are read, the tickets must start at zero and are cleared on the caller's stream before every launch
// (and re-armed by the last block, like the planned kernel).
//
// Same arithmetic scheme as the planned kernel -- fp32, fixed order (rows of a row group, row groups, row parts), no
// atomics on data, bitwise reproducible -- but its own partitioning, so the two paths agree within the rounding bound
// of tests/test_gpu_bias_grad.py, not bit for bit.
#include <algorithm>
#include <mutex>

#include "common.h"

namespace optb {

constexpr int kNaMaxN = OPT_NOALLOC_BIAS_GRAD_MAX_N;   // columns
constexpr int kNaMaxParts = 64;                        // row parts (grid.y)
constexpr int kNaStrip = 256;                          // columns per block: 32 lanes x one 16-byte vector of bf16
constexpr int kNaRowGroups = 8;                        // row groups per block (warps)
constexpr int kNaThreads = 32 * kNaRowGroups;
constexpr int kNaMaxStrips = kNaMaxN / kNaStrip;       // 16
constexpr int kNaMaxDevices = 64;

struct NaScratch {
  float part[kNaMaxParts * kNaMaxN];   // [part][column] partial sums: 1 MiB
  int32_t ticket[64];                  // [strip] blocks of the strip that have finished (256 B)
};
static_assert(sizeof(NaScratch) == OPT_NOALLOC_SCRATCH_BYTES, "the header states the scratch size");
static_assert(kNaMaxStrips <= 64, "one ticket per column strip");

static __device__ __align__(256) NaScratch g_na_scratch;

__global__ void __launch_bounds__(kNaThreads)
bias_grad_noalloc_kernel(const uint16_t* __restrict__ dz, int64_t ldz, void* __restrict__ db, int M, int N, int nparts,
                         int rows_per_part, int db_bf16, NaScratch* __restrict__ sc) {
  __shared__ float red[kNaRowGroups][kNaStrip + 8];
  __shared__ int is_last;
  const int strip = blockIdx.x, part = blockIdx.y;
  const int cv = threadIdx.x & 31, rg = threadIdx.x >> 5;
  const int col0 = strip * kNaStrip + cv * 8;
  const int r_begin = part * rows_per_part, r_end = min(M, r_begin + rows_per_part);
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  if (col0 < N) {                                      // N % 8 == 0: a vector is inside or outside as a whole
    const uint16_t* p = dz + col0;
    int r = r_begin + rg;
    for (; r + 3 * kNaRowGroups < r_end; r += 4 * kNaRowGroups) {       // four rows in flight per thread
      uint4 v[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) v[u] = __ldg(reinterpret_cast<const uint4*>(p + (int64_t)(r + u * kNaRowGroups) * ldz));
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const uint32_t w[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
#pragma unroll
        for (int t = 0; t < 4; ++t) { acc[2 * t] += bf16_lo(w[t]); acc[2 * t + 1] += bf16_hi(w[t]); }
      }
    }
    for (; r < r_end; r += kNaRowGroups) {
      const uint4 v = __ldg(reinterpret_cast<const uint4*>(p + (int64_t)r * ldz));
      const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (int t = 0; t < 4; ++t) { acc[2 * t] += bf16_lo(w[t]); acc[2 * t + 1] += bf16_hi(w[t]); }
    }
  }
#pragma unroll
  for (int j = 0; j < 8; ++j) red[rg][cv * 8 + j] = acc[j];
  __syncthreads();
  // row groups in group order -> this part's partial sum of column (strip, threadIdx.x)
  const int col = strip * kNaStrip + threadIdx.x;
  if (col < N) {
    float s = red[0][threadIdx.x];
#pragma unroll
    for (int g = 1; g < kNaRowGroups; ++g) s += red[g][threadIdx.x];
    sc->part[(size_t)part * kNaMaxN + col] = s;
  }
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) is_last = atomicAdd(&sc->ticket[strip], 1) == nparts - 1;
  __syncthreads();
  if (!is_last) return;
  // last block of the strip: the parts in part order, write db, re-arm the ticket
  __threadfence();
  if (col < N) {
    float s = 0.f;
    for (int q = 0; q < nparts; ++q) s += __ldcg(&sc->part[(size_t)q * kNaMaxN + col]);
    if (db_bf16) static_cast<__nv_bfloat16*>(db)[col] = __float2bfloat16_rn(s);
    else static_cast<float*>(db)[col] = s;
  }
  if (threadIdx.x == 0) sc->ticket[strip] = 0;
}

namespace {

std::mutex g_na_mu;
NaScratch* g_na_ptr[kNaMaxDevices] = {};     // device address of g_na_scratch on each device (set-up once per device)
int g_na_sms[kNaMaxDevices] = {};

// Once per device, with that device current: the device address of the scratch array.  No allocation.
opt_status na_setup(int device, NaScratch** ptr, int* sms) {
  std::lock_guard<std::mutex> lock(g_na_mu);
  if (device < 0 || device >= kNaMaxDevices) return fail(OPT_ERR_INVALID_ARG, "device %d out of range [0,%d)", device, kNaMaxDevices);
  if (!g_na_ptr[device]) {
    int n = 0;
    opt_status st = open_device(device, &n);         // checks sm_100, makes the device current
    if (st != OPT_OK) return st;
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_na_scratch);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      return fail(OPT_ERR_CUDA, "cudaGetSymbolAddress of the no-allocation scratch failed on device %d: %s", device,
                  cudaGetErrorString(e));
    }
    g_na_ptr[device] = static_cast<NaScratch*>(p);
    g_na_sms[device] = n;
  }
  *ptr = g_na_ptr[device];
  *sms = g_na_sms[device];
  return OPT_OK;
}

}  // namespace
}  // namespace optb

using namespace optb;

extern "C" opt_status opt_bias_grad_noalloc(const void* dz, int64_t ldz, void* db, int32_t M, int32_t N, opt_dtype param,
                                            int device, void* cuda_stream) {
  // host validation first: reported without a GPU, nothing launched
  if (!dz || !db) return fail(OPT_ERR_INVALID_ARG, "opt_bias_grad_noalloc: dz / db is NULL");
  if (M < 1 || N < 1) return fail(OPT_ERR_INVALID_ARG, "opt_bias_grad_noalloc: M = %d, N = %d must be >= 1", M, N);
  if (param != OPT_F32 && param != OPT_BF16) return fail(OPT_ERR_INVALID_ARG, "opt_bias_grad_noalloc: bad param dtype %d", (int)param);
  if (ldz < N) return fail(OPT_ERR_INVALID_ARG, "opt_bias_grad_noalloc: ldz = %lld < N = %d", (long long)ldz, N);
  if (N > kNaMaxN)
    return fail(OPT_ERR_UNSUPPORTED,
                "opt_bias_grad_noalloc: N = %d exceeds OPT_NOALLOC_BIAS_GRAD_MAX_N = %d, the width the static scratch "
                "of the no-allocation entry point holds; use opt_bias_grad_plan_create for wider layers", N, kNaMaxN);
  if (N % 8 != 0 || ldz % 8 != 0 || !aligned16(dz) || !aligned16(db))
    return fail(OPT_ERR_ALIGNMENT, "opt_bias_grad_noalloc: bf16 dZ needs N %% 8 == 0, ldz %% 8 == 0 and 16-byte aligned dz / db");
  {
    const uintptr_t z0 = reinterpret_cast<uintptr_t>(dz), z1 = z0 + ((uintptr_t)(M - 1) * (uintptr_t)ldz + (uintptr_t)N) * 2u;
    const uintptr_t b0 = reinterpret_cast<uintptr_t>(db), b1 = b0 + (uintptr_t)N * (uintptr_t)elem_size(param);
    if (b0 < z1 && z0 < b1) return fail(OPT_ERR_ALIAS, "opt_bias_grad_noalloc: db overlaps dz");
  }
  DeviceGuard guard;                                   // the caller's current device is left as it was
  NaScratch* sc = nullptr;
  int sms = 0;
  opt_status st = na_setup(device, &sc, &sms);
  if (st != OPT_OK) return st;
  OPT_CUDA_TRY(cudaSetDevice(device));
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  // partition: column strips x row parts, about two blocks per SM, at least 8 rows per row group and part
  const int nstrips = (N + kNaStrip - 1) / kNaStrip;
  int nparts = (2 * sms + nstrips - 1) / nstrips;
  nparts = std::min(nparts, kNaMaxParts);
  nparts = std::min(nparts, (M + 8 * kNaRowGroups - 1) / (8 * kNaRowGroups));
  nparts = std::max(nparts, 1);
  const int rows_per_part = (M + nparts - 1) / nparts;
  nparts = (M + rows_per_part - 1) / rows_per_part;    // no empty part
  // the tickets must start at zero whatever an earlier (possibly faulted) call left behind: cleared in stream order
  OPT_CUDA_TRY(cudaMemsetAsync(sc->ticket, 0, sizeof(sc->ticket), s));
  bias_grad_noalloc_kernel<<<dim3(nstrips, nparts), kNaThreads, 0, s>>>(static_cast<const uint16_t*>(dz), ldz, db, M, N, nparts,
                                                                          rows_per_part, param == OPT_BF16 ? 1 : 0, sc);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(OPT_ERR_CUDA, "opt_bias_grad_noalloc: kernel launch failed: %s", cudaGetErrorString(e));
  count_launch();
  return OPT_OK;
}
