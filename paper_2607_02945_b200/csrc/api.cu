// liboptimus_b200: plan lifecycle, launch entry points, error plumbing and the
// host-side independence check.  ABI contract: include/optimus_b200.h.
#include <algorithm>
#include <atomic>
#include <cstring>

#include "common.h"

namespace optb {

static thread_local std::string g_err;
static std::atomic<uint64_t> g_launches{0};

void set_error(const char* fmt, ...) {
  char buf[1024];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
}

opt_status fail(opt_status st, const char* fmt, ...) {
  char buf[1024];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return st;
}

void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

opt_status open_device(int device, int* num_sms) {
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return fail(OPT_ERR_NO_DEVICE, "no CUDA device available (%s)",
                e == cudaSuccess ? "device count is 0" : cudaGetErrorString(e));
  }
  if (device < 0 || device >= ndev) return fail(OPT_ERR_INVALID_ARG, "device %d out of range [0,%d)", device, ndev);
  int major = 0, minor = 0, sms = 0;
  OPT_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device));
  OPT_CUDA_TRY(cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, device));
  OPT_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
  if (major != 10)
    return fail(OPT_ERR_NO_DEVICE, "device %d is sm_%d%d; liboptimus_b200 is built for sm_100a only", device, major, minor);
  OPT_CUDA_TRY(cudaSetDevice(device));
  *num_sms = sms;
  return OPT_OK;
}

DeviceGuard::DeviceGuard() { if (cudaGetDevice(&prev_) != cudaSuccess) { cudaGetLastError(); prev_ = -1; } }
DeviceGuard::~DeviceGuard() {
  int cur = -1;
  if (prev_ >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev_) cudaSetDevice(prev_);
}

// Exact test for two strided regions that share a row pitch; conservative
// (reports overlap) otherwise.  Only called when the bounding intervals overlap.
static bool regions_overlap(const Region& a, const Region& b) {
  if (a.rows == 1 && b.rows == 1) return true;  // bounding interval is exact
  int64_t L = a.rows > 1 ? a.pitch_bytes : b.pitch_bytes;
  if ((a.rows > 1 && b.rows > 1 && a.pitch_bytes != b.pitch_bytes) || L <= 0) return true;
  uintptr_t ref = std::min(a.start, b.start);
  int64_t ca = (int64_t)((a.start - ref) % (uintptr_t)L), cb = (int64_t)((b.start - ref) % (uintptr_t)L);
  if (ca + a.row_bytes > L || cb + b.row_bytes > L) return true;  // a row wraps the pitch window
  return !(ca + a.row_bytes <= cb || cb + b.row_bytes <= ca);
}

opt_status check_independent(std::vector<Region>& regions, bool allow_inplace_self) {
  auto end_of = [](const Region& r) { return r.start + (uintptr_t)((r.rows - 1) * r.pitch_bytes + r.row_bytes); };
  std::sort(regions.begin(), regions.end(), [](const Region& a, const Region& b) { return a.start < b.start; });
  // sweep: `active` holds regions whose bounding interval is still open
  std::vector<size_t> active;
  for (size_t i = 0; i < regions.size(); ++i) {
    const Region& r = regions[i];
    size_t w = 0;
    for (size_t k = 0; k < active.size(); ++k)
      if (end_of(regions[active[k]]) > r.start) active[w++] = active[k];
    active.resize(w);
    for (size_t k : active) {
      const Region& q = regions[k];
      if (!r.is_output && !q.is_output) continue;       // inputs may alias inputs (batch_linear_lhs)
      if (!regions_overlap(q, r)) continue;
      if (allow_inplace_self && q.member == r.member && q.is_output != r.is_output && q.start == r.start &&
          q.pitch_bytes == r.pitch_bytes && q.row_bytes == r.row_bytes && q.rows == r.rows)
        continue;                                       // in-place pointwise chunk
      return fail(OPT_ERR_ALIAS,
                  "members %d (%s) and %d (%s) overlap in memory: group members must be independent "
                  "(PAPER.md:251)", q.member, q.is_output ? "output" : "input", r.member,
                  r.is_output ? "output" : "input");
    }
    active.push_back(i);
  }
  return OPT_OK;
}

opt_status upload_tables(opt_plan* p, const void* host_blob, size_t bytes) {
  OPT_CUDA_TRY(cudaMalloc(&p->dev_tables, bytes));
  p->table_bytes = bytes;
  cudaError_t e = cudaMemcpy(p->dev_tables, host_blob, bytes, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    cudaFree(p->dev_tables);
    p->dev_tables = nullptr;
    return fail(OPT_ERR_CUDA, "table upload failed: %s", cudaGetErrorString(e));
  }
  return OPT_OK;
}

static cudaError_t launch_kind(const opt_plan* p, cudaStream_t s) {
  switch (p->kind) {
    case kPlanPointwise: return launch_pointwise(p, s);
    case kPlanLayerNorm: return launch_layernorm(p, s);
    case kPlanLinearBf16: return launch_linear_bf16(p, s);
    case kPlanLinearF32: return launch_linear_f32(p, s);
    case kPlanLinear2: case kPlanLnLinear2: return launch_linear2(p, s);
    case kPlanLinearSkinny: return launch_linear_skinny(p, s);
    case kPlanLayerNormBwd: return launch_layernorm_bwd(p, s);
    case kPlanBiasGrad: return launch_bias_grad(p, s);
    default: return cudaErrorInvalidValue;
  }
}

// The kernel goes to the PLAN's device whatever the caller's current device is (restored afterwards).
static cudaError_t launch_any(const opt_plan* p, cudaStream_t s) {
  int cur = -1;
  cudaError_t e = cudaGetDevice(&cur);
  if (e != cudaSuccess) return e;
  if (cur == p->device) return launch_kind(p, s);
  if ((e = cudaSetDevice(p->device)) != cudaSuccess) return e;
  e = launch_kind(p, s);
  cudaSetDevice(cur);
  return e;
}

}  // namespace optb

using namespace optb;

extern "C" {

opt_status opt_plan_launch(const opt_plan* plan, void* cuda_stream) {
  if (!plan) return fail(OPT_ERR_INVALID_ARG, "opt_plan_launch: plan is NULL");
  cudaError_t e = launch_any(plan, static_cast<cudaStream_t>(cuda_stream));
  if (e != cudaSuccess) return fail(OPT_ERR_CUDA, "kernel launch failed: %s", cudaGetErrorString(e));
  count_launch();
  return OPT_OK;
}

opt_status opt_plan_launch_host(const opt_plan* plan, const opt_host_copy* copies, int32_t ncopies,
                                void* cuda_stream) {
  if (!plan) return fail(OPT_ERR_INVALID_ARG, "opt_plan_launch_host: plan is NULL");
  if (ncopies < 0 || (ncopies > 0 && !copies)) return fail(OPT_ERR_INVALID_ARG, "opt_plan_launch_host: bad copy list");
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  for (int32_t i = 0; i < ncopies; ++i) {
    if (!copies[i].host || !copies[i].device) return fail(OPT_ERR_INVALID_ARG, "copy %d has a NULL pointer", i);
    if (copies[i].to_device)
      OPT_CUDA_TRY(cudaMemcpyAsync(copies[i].device, copies[i].host, copies[i].bytes, cudaMemcpyHostToDevice, s));
  }
  cudaError_t e = launch_any(plan, s);
  if (e != cudaSuccess) return fail(OPT_ERR_CUDA, "kernel launch failed: %s", cudaGetErrorString(e));
  count_launch();
  for (int32_t i = 0; i < ncopies; ++i)
    if (!copies[i].to_device)
      OPT_CUDA_TRY(cudaMemcpyAsync(copies[i].host, copies[i].device, copies[i].bytes, cudaMemcpyDeviceToHost, s));
  return OPT_OK;
}

opt_status opt_plan_info(const opt_plan* plan, int64_t* flops, int64_t* bytes, int32_t* launches, int32_t* tiles) {
  if (!plan) return fail(OPT_ERR_INVALID_ARG, "opt_plan_info: plan is NULL");
  if (flops) *flops = plan->flops;
  if (bytes) *bytes = plan->bytes;
  if (launches) *launches = 1;
  if (tiles) *tiles = plan->total_tiles;
  return OPT_OK;
}

opt_status opt_plan_destroy(opt_plan* plan) {
  if (!plan) return OPT_OK;
  if (plan->dev_tables) cudaFree(plan->dev_tables);
  if (plan->workspace) cudaFree(plan->workspace);
  delete plan;
  return OPT_OK;
}

const char* opt_last_error(void) { return g_err.c_str(); }

uint64_t opt_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

const char* opt_version(void) { return "liboptimus_b200 0.1 (sm_100a)"; }

}  // extern "C"
