// Internal header of liboptimus_b200 (not installed; the public ABI is
// include/optimus_b200.h).  Plan object, error plumbing, the host-side
// independence (alias) check, and small device helpers shared by the kernels.
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <cuda_fp8.h>

#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

#include "optimus_b200.h"

namespace optb {

// ------------------------------------------------------------------ errors --
void set_error(const char* fmt, ...);
opt_status fail(opt_status st, const char* fmt, ...);
void count_launch();

#define OPT_CUDA_TRY(expr)                                                                   \
  do {                                                                                       \
    cudaError_t e__ = (expr);                                                                \
    if (e__ != cudaSuccess)                                                                  \
      return ::optb::fail(OPT_ERR_CUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), \
                          __FILE__, __LINE__);                                               \
  } while (0)

inline int elem_size(opt_dtype dt) { return dt == OPT_F32 ? 4 : 2; }
inline int vec_elems(opt_dtype dt) { return 16 / elem_size(dt); }   // elements per 16-byte vector
inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// opens the device (must be sm_100) -- makes it the thread's current device -- and returns its SM count
opt_status open_device(int device, int* num_sms);
// every *_plan_create holds one of these: the caller's current device is restored when plan creation returns
struct DeviceGuard {
  DeviceGuard();
  ~DeviceGuard();
  int prev_ = -1;
};

// ------------------------------------------------------------ alias check ---
// A strided 2-D byte region: rows x row_bytes, row pitch pitch_bytes.
struct Region {
  uintptr_t start;
  int64_t pitch_bytes;
  int64_t row_bytes;
  int64_t rows;
  bool is_output;
  int32_t member;
};
// PAPER.md:251 independence: no output may overlap an input or another output.
// allow_inplace_self: a member whose input region is identical to its output
// region (pointwise in place) is accepted.
opt_status check_independent(std::vector<Region>& regions, bool allow_inplace_self);

// ---------------------------------------------------------------- the plan --
enum PlanKind { kPlanPointwise = 1, kPlanLayerNorm = 2, kPlanLinearBf16 = 3, kPlanLinearF32 = 4, kPlanLinear2 = 5, kPlanLayerNormBwd = 6, kPlanLnLinear2 = 7, kPlanLinearSkinny = 8, kPlanBiasGrad = 9 };

}  // namespace optb

struct opt_plan {
  int kind = 0;
  int device = 0;
  void* dev_tables = nullptr;   // one device allocation holding every table of the plan
  void* workspace = nullptr;    // optional scratch owned by the plan (LayerNorm backward / bias gradient: per-block partial sums)
  size_t table_bytes = 0;
  // offsets of sub-tables inside dev_tables (meaning depends on kind)
  size_t off0 = 0, off1 = 0, off2 = 0, off3 = 0;
  dim3 grid{1, 1, 1}, block{1, 1, 1};
  size_t smem = 0;
  int32_t n_members = 0;
  int32_t total_tiles = 0;
  int32_t n_chunks = 0, nstages = 0, stage_bytes = 0, ncta = 1;
  int32_t ln_tile_max = 0, ln_pmax = 0;                 // staged LayerNorm: bytes of a stage's row tile / of one parameter vector   // grouped GEMM: schedule chunks, smem ring shape
  int32_t io = 0, param = 0;
  int64_t flops = 0, bytes = 0;
};

namespace optb {
// per-kind launchers (exactly one kernel launch each)
cudaError_t launch_pointwise(const opt_plan* p, cudaStream_t s);
cudaError_t launch_layernorm(const opt_plan* p, cudaStream_t s);
cudaError_t launch_linear_bf16(const opt_plan* p, cudaStream_t s);
cudaError_t launch_linear_f32(const opt_plan* p, cudaStream_t s);
cudaError_t launch_linear2(const opt_plan* p, cudaStream_t s);
cudaError_t launch_linear_skinny(const opt_plan* p, cudaStream_t s);
bool skinny_linear_member(const opt_linear_member& m);
opt_status plan_skinny_linear(const opt_linear_member* members, int32_t n, opt_plan* p);
cudaError_t launch_layernorm_bwd(const opt_plan* p, cudaStream_t s);
cudaError_t launch_bias_grad(const opt_plan* p, cudaStream_t s);

// host->device upload of a table blob; allocates p->dev_tables
opt_status upload_tables(opt_plan* p, const void* host_blob, size_t bytes);
}  // namespace optb

// ---------------------------------------------------------- device helpers --
#ifdef __CUDACC__
namespace optb {

// Activation in fp32.  FAST=true: MUFU approximations (tanh.approx, ex2.approx,
// rcp.approx), good to ~2^-11 relative -- only for results rounded to bf16.
// FAST=false: libdevice tanhf/expf for fp32 outputs (reading Q10).
template <bool FAST>
__device__ __forceinline__ float act_f32(float x, int act) {
  if (act == 1) {            // relu, NaN propagates (torch semantics, Q13)
    return (x > 0.f || x != x) ? x : 0.f;
  } else if (act == 2) {     // tanh
    if (FAST) {
      float y;
      asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
      return fabsf(x) < 0.0078125f ? x : y;   // tanh(x) = x(1 - x^2/3 ..): below 2^-7 the identity is within 2^-15, and keeps subnormals
    } else {
      return tanhf(x);
    }
  } else if (act == 3) {     // sigmoid: t = 2^(-|x| log2 e) in (0,1];  x >= 0: 1/(1+t);  x < 0: t/(1+t)
    if (FAST) {              // (1+t) stays in [1,2], so both tails keep full relative accuracy, subnormal results included
      float t, r;
      asm("ex2.approx.f32 %0, %1;" : "=f"(t) : "f"(fabsf(x) * -1.4426950408889634f));
      asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(1.f + t));
      return x >= 0.f ? r : (x != x ? x : t * r);
    } else {
      return x >= 0.f ? 1.f / (1.f + expf(-x)) : expf(x) / (1.f + expf(x));
    }
  }
  return x;
}

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);   // .x = lo (low 16 bits)
  return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ float bf16_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t u) { return __uint_as_float(u & 0xFFFF0000u); }

// FP8 (OCP E4M3) quantisation of four bf16 values held as two packed pairs (reading Q24: the product value x scale
// is formed in fp32, then one saturating round-to-nearest-even; NaN -> NaN).  Lowest column in the low byte.  ONE
// definition for the stand-alone op (OPT_PW_QUANT_E4M3) and the fused epilogues (grouped Linear, batched LayerNorm).
__device__ __forceinline__ uint32_t quant4_e4m3(uint32_t a, uint32_t b, float scale) {
  const uint32_t lo = __nv_cvt_float2_to_fp8x2(make_float2(bf16_lo(a) * scale, bf16_hi(a) * scale), __NV_SATFINITE, __NV_E4M3);
  const uint32_t hi = __nv_cvt_float2_to_fp8x2(make_float2(bf16_lo(b) * scale, bf16_hi(b) * scale), __NV_SATFINITE, __NV_E4M3);
  return lo | (hi << 16);
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


}  // namespace optb
#endif
