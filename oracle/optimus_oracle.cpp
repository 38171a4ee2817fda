// optimus_oracle.cpp -- CPU ORACLE. TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct fp64 definitions of the ops on the hot path
// of Optimus' horizontally fused groups (arxiv/paper_2607_02945).  One op at a
// time, the UNFUSED graph: "given the same input, pattern r_s and r_d have the
// same output" (section 2.2) -- so the oracle of a fused group is
// the original N independent ops run one by one.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may call this.  It shares no code with
// paper_2607_02945_b200/ (no headers, helpers, tables or constants).
//
// Every function below is pinned by tests/test_oracle_pins.py (worked example
// of PAPER.md Listing 1/2, closed forms, brute force, identities); nothing is
// "parity unpinned".
//
// Storage dtypes: 0 = fp32, 1 = bf16 (raw 16-bit patterns).  Inputs are
// widened exactly to double; every sum is taken in double in index order; a
// result is rounded ONCE, directly from double to the storage dtype with
// round-to-nearest-even (reading Q3).
//
// OpenMP only parallelises over independent rows; it never changes the order
// of any floating-point sum.
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int kF32 = 0, kBF16 = 1;

inline double widen(const void* p, int64_t i, int dt) {
  if (dt == kF32) return (double)((const float*)p)[i];
  uint32_t u = (uint32_t)((const uint16_t*)p)[i] << 16;   // bf16 -> fp32 is exact
  float f;
  std::memcpy(&f, &u, 4);
  return (double)f;
}

// double -> bf16 bits, round-to-nearest-even, done on the double's own bit
// pattern (never through float: double rounding differs on some ties).
// bf16 = 1 sign, 8 exponent (bias 127), 7 fraction bits.
uint16_t f64_to_bf16_bits(double d) {
  uint64_t b;
  std::memcpy(&b, &d, 8);
  const uint16_t sign = (uint16_t)((b >> 63) << 15);
  const int64_t e = (int64_t)((b >> 52) & 0x7FF);
  const uint64_t frac = b & 0xFFFFFFFFFFFFFull;
  if (e == 0x7FF) {                                   // inf / nan
    if (frac) return (uint16_t)(sign | 0x7FC0);       // quiet NaN
    return (uint16_t)(sign | 0x7F80);
  }
  if (e == 0) return sign;                            // double subnormal: far below bf16 range
  // value = 1.frac * 2^(e-1023)
  int64_t eb = e - 1023 + 127;                        // bf16 biased exponent if normal
  uint64_t sig = (1ull << 52) | frac;                 // 53-bit significand
  int shift = 52 - 7;                                 // keep 1+7 bits
  if (eb <= 0) {                                      // bf16 subnormal (or underflow)
    int64_t extra = 1 - eb;
    if (extra > 10) return sign;                      // shift >= 56: sig < 2^53 is below half a min subnormal -> 0
    shift += (int)extra;
    eb = 0;
  }
  uint64_t kept = sig >> shift;
  uint64_t rem = sig & ((1ull << shift) - 1);
  uint64_t half = 1ull << (shift - 1);
  if (rem > half || (rem == half && (kept & 1))) kept += 1;
  // kept includes the implicit bit for normals: (eb<<7) + kept - (1<<7) handles carry.
  uint64_t out;
  if (eb == 0) out = kept;                            // subnormal; carry into exponent 1 is natural
  else out = ((uint64_t)eb << 7) + (kept - (1ull << 7));
  if (out >= 0x7F80) out = 0x7F80;                    // overflow -> inf
  return (uint16_t)(sign | (uint16_t)out);
}

inline double act_apply(double x, int act) {
  switch (act) {
    case 1:  // relu: torch semantics, NaN propagates (Q13)
      return x > 0.0 ? x : (std::isnan(x) ? x : 0.0);
    case 2:
      return std::tanh(x);
    case 3:  // sigmoid, overflow-free form
      if (x >= 0.0) return 1.0 / (1.0 + std::exp(-x));
      else { double e = std::exp(x); return e / (1.0 + e); }
    default:
      return x;
  }
}

}  // namespace

extern "C" {

void oracle_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

int oracle_get_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// ---- storage rounding (Q3): once per op output, double -> storage directly.
void oracle_round_to_storage(const double* z, int64_t n, int dt, void* out) {
  if (dt == kF32) {
    float* o = (float*)out;
    for (int64_t i = 0; i < n; ++i) o[i] = (float)z[i];   // C cast double->float is RNE
  } else {
    uint16_t* o = (uint16_t*)out;
    for (int64_t i = 0; i < n; ++i) o[i] = f64_to_bf16_bits(z[i]);
  }
}

void oracle_widen(const void* p, int64_t n, int dt, double* out) {
  for (int64_t i = 0; i < n; ++i) out[i] = widen(p, i, dt);
}

// ---- linear: Z[m,n] = sum_{k<K} X[m,k] * W[n,k] + b[n]   (torch nn.Linear
// layout, W is [N,K]; PAPER.md:148 "A x B", :292 batch_linear; reading Q1).
// Sum in index order k = 0..K-1, in double, bias added last.
// z is dense [M,N] double.  bias may be NULL.
void oracle_linear(const void* x, int64_t ldx, const void* w, int64_t ldw, const void* bias,
                   int32_t M, int32_t N, int32_t K, int dt, double* z) {
#pragma omp parallel for schedule(static)
  for (int32_t m = 0; m < M; ++m) {
    std::vector<double> xr((size_t)K);
    for (int32_t k = 0; k < K; ++k) xr[k] = widen(x, (int64_t)m * ldx + k, dt);
    for (int32_t n = 0; n < N; ++n) {
      double acc = 0.0;
      for (int32_t k = 0; k < K; ++k) acc += xr[k] * widen(w, (int64_t)n * ldw + k, dt);
      if (bias) acc += widen(bias, n, dt);
      z[(int64_t)m * N + n] = acc;
    }
  }
}

// ---- the same linear on an activation matrix that is ALREADY in double (dense [M,K]): the first layer of a
// vertically fused LayerNorm -> Linear chain, whose normalised input is never materialised and therefore never
// rounded (reading Q25; "chained transformations").  Weights and bias are storage dtype.
// Same loop nest and summation order as oracle_linear (k = 0..K-1, bias added last).
void oracle_linear_f64x(const double* x, const void* w, int64_t ldw, const void* bias,
                        int32_t M, int32_t N, int32_t K, int dt, double* z) {
#pragma omp parallel for schedule(static)
  for (int32_t m = 0; m < M; ++m) {
    for (int32_t n = 0; n < N; ++n) {
      double acc = 0.0;
      for (int32_t k = 0; k < K; ++k) acc += x[(int64_t)m * K + k] * widen(w, (int64_t)n * ldw + k, dt);
      if (bias) acc += widen(bias, n, dt);
      z[(int64_t)m * N + n] = acc;
    }
  }
}

// ---- bias gradient of y = x W^T + b: db[n] = sum_{m<M} dZ[m,n], rows added in index order m = 0..M-1, in double
// (the third output of the backward of a Linear; batch_linear_post_grad; training).
void oracle_colsum(const void* dz, int64_t ldz, int32_t M, int32_t N, int dt, double* db) {
  for (int32_t n = 0; n < N; ++n) {
    double acc = 0.0;
    for (int32_t m = 0; m < M; ++m) acc += widen(dz, (int64_t)m * ldz + n, dt);
    db[n] = acc;
  }
}

// ---- the same linear written as broadcast-multiply then reduce over K with a
// different loop nest (k outermost) -- the decompose_mm formulation of
// PAPER.md:475.  Only used by the pin test P5 as an independent second formula.
void oracle_linear_mulreduce(const void* x, int64_t ldx, const void* w, int64_t ldw,
                             const void* bias, int32_t M, int32_t N, int32_t K, int dt, double* z) {
  for (int64_t i = 0; i < (int64_t)M * N; ++i) z[i] = 0.0;
  for (int32_t k = 0; k < K; ++k)
    for (int32_t m = 0; m < M; ++m) {
      const double a = widen(x, (int64_t)m * ldx + k, dt);
      for (int32_t n = 0; n < N; ++n) z[(int64_t)m * N + n] += a * widen(w, (int64_t)n * ldw + k, dt);
    }
  if (bias)
    for (int32_t m = 0; m < M; ++m)
      for (int32_t n = 0; n < N; ++n) z[(int64_t)m * N + n] += widen(bias, n, dt);
}

// ---- activation, elementwise on double, in place (batch_relu / batch_sigmoid
// / batch_aten_tanh).  act: 0 none, 1 relu, 2 tanh, 3 sigmoid.
void oracle_activation(double* z, int64_t n, int act) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) z[i] = act_apply(z[i], act);
}

// ---- pointwise on a strided 2-D storage tensor -> dense double [rows,width].
void oracle_pointwise(const void* src, int64_t lds, int32_t rows, int32_t width, int op, int dt,
                      double* out) {
#pragma omp parallel for schedule(static)
  for (int32_t r = 0; r < rows; ++r)
    for (int32_t c = 0; c < width; ++c)
      out[(int64_t)r * width + c] = act_apply(widen(src, (int64_t)r * lds + c, dt), op);
}

// ---- the remaining horizontal pointwise patterns of Table 1: batch_clamp,
// batch_nan_to_num (unary, scalar parameters) and batch_aten_sub / _div / _mul (binary), torch
// semantics, on strided 2-D storage tensors -> dense double [rows,width].
//   op 4 clamp:      y = min(max(x, lo), hi), NaN propagates            (torch.clamp)
//   op 5 nan_to_num: NaN -> p0, +inf -> p1, -inf -> p2, else x          (torch.nan_to_num)
//   op 6 / 7 / 8:    a - b, a / b, a * b                                (aten.sub / div / mul)
//   op 11 relu_bwd:  y = (b <= 0) ? 0 : a   -- a = incoming gradient, b = the ReLU's forward output (or its input:
//                    same mask); the backward of the ReLU epilogue of a grouped Linear in a post-grad graph
//                    (batch_linear_post_grad; training QPS is the headline)
//   op 12 tanh_bwd:    y = a (1 - b^2)    -- b = the STORED forward output tanh(z)    (torch tanh_backward)
//   op 13 sigmoid_bwd: y = a (1 - b) b    -- b = the STORED forward output sigmoid(z) (torch sigmoid_backward)
//                    the backward of the other two epilogues of the grouped Linear (same passages as op 11)
// b may be NULL for the unary ops.
void oracle_pointwise_ext(const void* a, int64_t lda, const void* b, int64_t ldb, int32_t rows, int32_t width,
                          int op, double p0, double p1, double p2, int dt, double* out) {
#pragma omp parallel for schedule(static)
  for (int32_t r = 0; r < rows; ++r)
    for (int32_t c = 0; c < width; ++c) {
      const double x = widen(a, (int64_t)r * lda + c, dt);
      double y;
      switch (op) {
        case 4:
          if (std::isnan(x)) { y = x; break; }
          y = x < p0 ? p0 : x;
          y = y > p1 ? p1 : y;
          break;
        case 5:
          y = std::isnan(x) ? p0 : (std::isinf(x) ? (x > 0 ? p1 : p2) : x);
          break;
        case 6: y = x - widen(b, (int64_t)r * ldb + c, dt); break;
        case 7: y = x / widen(b, (int64_t)r * ldb + c, dt); break;
        case 8: y = x * widen(b, (int64_t)r * ldb + c, dt); break;
        case 11: y = widen(b, (int64_t)r * ldb + c, dt) <= 0.0 ? 0.0 : x; break;
        case 12: { const double t = widen(b, (int64_t)r * ldb + c, dt); y = x * (1.0 - t * t); break; }
        case 13: { const double t = widen(b, (int64_t)r * ldb + c, dt); y = x * ((1.0 - t) * t); break; }
        default: y = x; break;
      }
      out[(int64_t)r * width + c] = y;
    }
}

// ---- FP8 (OCP E4M3: 1 sign, 4 exponent bits with bias 7, 3 mantissa bits; no infinity, S.1111.111 = NaN,
// largest finite 448) quantisation of saved activations -- activation_quantization_aten_pass (PAPER.md:341-345,
// :487-489: "quantized into a lower-precision format, such as FP8, in the forward pass ... dequantized back to
// their original precision before use", optional scaling).
//   quantise:   code = e4m3_rne_satfinite(x * scale)    (|v| > 448 and +-inf saturate to +-448, NaN -> NaN)
//   dequantise: y    = value(code) * scale
static double e4m3_value(uint8_t c) {
  const int e = (c >> 3) & 0xF, m = c & 7;
  double v;
  if (e == 0xF && m == 7) return std::nan("");
  if (e == 0) v = std::ldexp((double)m, -9);                 // subnormal: m * 2^-6 * 2^-3
  else v = std::ldexp(8.0 + m, e - 10);                      // (1 + m/8) * 2^(e-7)
  return (c & 0x80) ? -v : v;
}
static uint8_t f64_to_e4m3(double x) {
  if (std::isnan(x)) return 0x7F;
  const uint8_t sign = std::signbit(x) ? 0x80 : 0;
  const double a = std::fabs(x);
  if (a >= 448.0) return sign | 0x7E;                        // satfinite (also inf)
  // nearest representable code in [0x00, 0x7E], ties to the even code: the codes are monotone in value
  int lo = 0, hi = 0x7E;
  while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (e4m3_value((uint8_t)mid) <= a) lo = mid; else hi = mid; }
  const double vl = e4m3_value((uint8_t)lo), vh = e4m3_value((uint8_t)hi);
  const double dl = a - vl, dh = vh - a;
  int c = dl < dh ? lo : (dh < dl ? hi : ((lo & 1) ? hi : lo));
  return sign | (uint8_t)c;
}
void oracle_quant_e4m3(const void* src, int64_t lds, int32_t rows, int32_t width, double scale, int dt, uint8_t* out) {
#pragma omp parallel for schedule(static)
  for (int32_t r = 0; r < rows; ++r)
    for (int32_t c = 0; c < width; ++c) out[(int64_t)r * width + c] = f64_to_e4m3(widen(src, (int64_t)r * lds + c, dt) * scale);
}
void oracle_dequant_e4m3(const uint8_t* src, int64_t lds, int32_t rows, int32_t width, double scale, double* out) {
#pragma omp parallel for schedule(static)
  for (int32_t r = 0; r < rows; ++r)
    for (int32_t c = 0; c < width; ++c) out[(int64_t)r * width + c] = e4m3_value(src[(int64_t)r * lds + c]) * scale;
}

// ---- layer_norm over the last dim (batch_layernorm; torch
// semantics, reading Q4): mu = sum(x)/D; v = sum((x-mu)^2)/D (biased);
// y_j = (x_j-mu)/sqrt(v+eps) * gamma_j + beta_j.  gamma/beta may be NULL (1/0).
// y dense [rows,D] double.  xhat (optional, may be NULL) receives the
// pre-affine normalised row, for the invariant pins.
void oracle_layernorm(const void* x, int64_t ldx, const void* gamma, const void* beta,
                      int32_t rows, int32_t D, double eps, int dt, int param_dt,
                      double* y, double* xhat) {
#pragma omp parallel for schedule(static)
  for (int32_t r = 0; r < rows; ++r) {
    double s = 0.0;
    for (int32_t j = 0; j < D; ++j) s += widen(x, (int64_t)r * ldx + j, dt);
    const double mu = s / (double)D;
    double q = 0.0;
    for (int32_t j = 0; j < D; ++j) {
      const double d = widen(x, (int64_t)r * ldx + j, dt) - mu;
      q += d * d;
    }
    const double v = q / (double)D;
    const double sd = std::sqrt(v + eps);
    for (int32_t j = 0; j < D; ++j) {
      const double xh = (widen(x, (int64_t)r * ldx + j, dt) - mu) / sd;
      if (xhat) xhat[(int64_t)r * D + j] = xh;
      const double g = gamma ? widen(gamma, j, param_dt) : 1.0;
      const double b = beta ? widen(beta, j, param_dt) : 0.0;
      y[(int64_t)r * D + j] = xh * g + b;
    }
  }
}

// ---- layer_norm backward (torch native_layer_norm_backward): with
//   mu, v as in the forward, rstd = 1/sqrt(v+eps), xhat = (x-mu) rstd, g_j = dy_j gamma_j:
//   dx_j     = rstd * ( g_j - mean_j(g) - xhat_j * mean_j(g xhat) )        per row
//   dgamma_j = sum_rows dy_j xhat_j ;  dbeta_j = sum_rows dy_j             (rows summed in index order)
// dx dense [rows,D]; dgamma / dbeta [D] (may be NULL).  gamma may be NULL (= 1).
void oracle_layernorm_backward(const void* x, int64_t ldx, const void* dy, int64_t lddy, const void* gamma,
                               int32_t rows, int32_t D, double eps, int dt, int param_dt,
                               double* dx, double* dgamma, double* dbeta) {
  std::vector<double> xh_all(dgamma ? (size_t)rows * D : 0);
#pragma omp parallel for schedule(static)
  for (int32_t r = 0; r < rows; ++r) {
    double s = 0.0;
    for (int32_t j = 0; j < D; ++j) s += widen(x, (int64_t)r * ldx + j, dt);
    const double mu = s / (double)D;
    double q = 0.0;
    for (int32_t j = 0; j < D; ++j) { const double d = widen(x, (int64_t)r * ldx + j, dt) - mu; q += d * d; }
    const double rstd = 1.0 / std::sqrt(q / (double)D + eps);
    double sg = 0.0, sgx = 0.0;
    for (int32_t j = 0; j < D; ++j) {
      const double xh = (widen(x, (int64_t)r * ldx + j, dt) - mu) * rstd;
      const double g = widen(dy, (int64_t)r * lddy + j, dt) * (gamma ? widen(gamma, j, param_dt) : 1.0);
      sg += g; sgx += g * xh;
      if (dgamma) xh_all[(size_t)r * D + j] = xh;
    }
    const double mg = sg / (double)D, mgx = sgx / (double)D;
    for (int32_t j = 0; j < D; ++j) {
      const double xh = (widen(x, (int64_t)r * ldx + j, dt) - mu) * rstd;
      const double g = widen(dy, (int64_t)r * lddy + j, dt) * (gamma ? widen(gamma, j, param_dt) : 1.0);
      dx[(int64_t)r * D + j] = rstd * (g - mg - xh * mgx);
    }
  }
  for (int32_t j = 0; j < D && (dgamma || dbeta); ++j) {
    double a = 0.0, b = 0.0;
    for (int32_t r = 0; r < rows; ++r) {
      const double d = widen(dy, (int64_t)r * lddy + j, dt);
      if (dgamma) a += d * xh_all[(size_t)r * D + j];
      b += d;
    }
    if (dgamma) dgamma[j] = a;
    if (dbeta) dbeta[j] = b;
  }
}

// ---- split along dim 1 (torch.split(x, sizes, dim=1)):
// piece j = x[:, s_j : s_j + w_j], s_j = sum_{t<j} w_t.  Raw element copy
// (elem_size bytes per element); piece j is written densely [rows, w_j] at
// pieces[j].  Returns 0, or -1 if the sizes do not sum to `width`.
int oracle_split(const void* x, int64_t ldx, int32_t rows, int32_t width, int32_t elem_size,
                 const int32_t* sizes, int32_t npieces, void** pieces) {
  int64_t tot = 0;
  for (int32_t j = 0; j < npieces; ++j) tot += sizes[j];
  if (tot != width) return -1;
  int64_t s = 0;
  for (int32_t j = 0; j < npieces; ++j) {
    for (int32_t r = 0; r < rows; ++r)
      std::memcpy((char*)pieces[j] + (int64_t)r * sizes[j] * elem_size,
                  (const char*)x + ((int64_t)r * ldx + s) * elem_size,
                  (size_t)sizes[j] * elem_size);
    s += sizes[j];
  }
  return 0;
}

// ---- cat along dim 1 (torch.cat(pieces, dim=1)):
// out[:, d_j : d_j + w_j] = piece_j, d_j = sum_{t<j} w_t, pieces dense
// [rows, w_j].  Raw element copy.
void oracle_cat(void* const* pieces, const int32_t* sizes, int32_t npieces, int32_t rows,
                int32_t elem_size, void* out, int64_t ldo) {
  int64_t d = 0;
  for (int32_t j = 0; j < npieces; ++j) {
    for (int32_t r = 0; r < rows; ++r)
      std::memcpy((char*)out + ((int64_t)r * ldo + d) * elem_size,
                  (const char*)pieces[j] + (int64_t)r * sizes[j] * elem_size,
                  (size_t)sizes[j] * elem_size);
    d += sizes[j];
  }
}

}  // extern "C"
