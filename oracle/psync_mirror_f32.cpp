// psync fp32 MIRROR -- a DIAGNOSTIC, NOT THE GRADED ORACLE, and test infrastructure only.
//
// The graded truth is oracle/psync_oracle.cpp (double arithmetic on fp32 storage, written from the paper;
// nothing in that file knows about this one).  This separate library restates, on the CPU, the fp32
// OPERATION LIST that DESIGN.md readings R9 / R10 say the CUDA path uses, so that a GPU result can be
// compared BIT FOR BIT -- which checks the summation order, the placement of the fused multiply-adds and
// the device-side coefficients, things a 1e-5 tolerance cannot see.  It is a regression check of the
// kernels against their own documented arithmetic; it is not parity evidence and no parity claim rests
// on it.  ("a second build of the same oracle ... in float, same order".)
//
// Operation list (R9 / R10), per element:
//   S    = 0;  S = S + G_k            one fp32 add per kept worker, in the order listed (ascending k)
//   G    = S * inv_N                  inv_N = 1.0f / (float)n formed in fp32 (R8); the clip factor for Alg. 2
//   SGD        theta = fma(-gamma, G, theta)
//   momentum   v = fma(mu, v, G);  theta = fma(-gamma, v, theta)
//   RMSProp    ms  = fma(rho, ms, (1-rho) * (G * G))
//              mom = fma(mu, mom, (gamma * G) * rsqrt(ms + eps))     rsqrt = correctly rounded 1/sqrt
//              theta = theta - mom
//   EMA        ema = fma(alpha, ema, (1-alpha) * operand)            operand = new theta (POST) / old (PRE)
// Every other operation is one IEEE fp32 operation, round-to-nearest-even (compile with -ffp-contract=off).
//
// Pinned (tests/test_oracle_fp32_mirror.py, -m "not gpu") by exact rational arithmetic rounded once per
// stated operation (mpmath decides the square root), by the hand-worked dyadic examples, and by closeness
// to the double oracle.  Shares no code with oracle/psync_oracle.cpp nor with the CUDA path.

#include <cmath>
#include <cstdint>
#include <cstring>

namespace {

constexpr int M_OK = 0, M_EINVAL = -1;
constexpr int M_F32 = 0, M_BF16 = 1;
constexpr int M_SGD = 0, M_MOMENTUM = 1, M_RMSPROP_MOM = 2;
constexpr int M_EMA_POST = 0, M_EMA_PRE = 1, M_EMA_OFF = 2;

inline float grad_f32(const void* g, int dtype, int64_t i) {
  if (dtype == M_F32) return static_cast<const float*>(g)[i];
  const uint32_t u = static_cast<uint32_t>(static_cast<const uint16_t*>(g)[i]) << 16;  // bf16 widens exactly
  float f;
  std::memcpy(&f, &u, sizeof f);
  return f;
}

struct CoeffsF {
  float gamma, alpha, one_minus_alpha, mu, rho, one_minus_rho, eps, inv_N;
};

inline CoeffsF make_coeffs(int32_t n, float gamma_t, float alpha, float mu, float rho, float eps) {
  CoeffsF c;
  c.gamma = gamma_t;
  c.alpha = alpha;
  c.one_minus_alpha = 1.0f - alpha;
  c.mu = mu;
  c.rho = rho;
  c.one_minus_rho = 1.0f - rho;
  c.eps = eps;
  c.inv_N = 1.0f / static_cast<float>(n);
  return c;
}

// Correctly rounded fp32 reciprocal square root, RN-even, of a positive finite normal x.
// y0 = (float)(1 / sqrt((double)x)) is within one fp32 ulp of the answer; the three neighbouring candidates
// are then compared EXACTLY: y is the rounding of 1/sqrt(x) iff it lies between the two midpoints around
// it, and 1/sqrt(x) < m  <=>  m*m*x > 1 (all positive).  m has <= 25 significant bits, so m*m is exact in
// double and m*m*x is evaluated exactly as hi + lo with one fma.  (1/sqrt(x) is never a midpoint: that
// would need m*m*x == 1 with m of 25 bits and x of 24 bits, and then m*m*x has an odd significand > 1.)
inline float rsqrt_rn(float x) {
  if (!(x > 0.0f) || !std::isfinite(x)) return 1.0f / std::sqrt(x);  // 0, negative, inf, NaN: IEEE special values
  const double xd = static_cast<double>(x);
  float y = static_cast<float>(1.0 / std::sqrt(xd));
  auto below = [xd](double m) {  // true iff 1/sqrt(x) < m
    const double p = m * m;      // exact (<= 50 bits)
    const double hi = p * xd;
    const double lo = std::fma(p, xd, -hi);  // p*x = hi + lo exactly
    return hi > 1.0 || (hi == 1.0 && lo > 0.0);
  };
  for (int it = 0; it < 2; ++it) {
    const float up = std::nextafterf(y, INFINITY), dn = std::nextafterf(y, 0.0f);
    const double m_hi = 0.5 * (static_cast<double>(y) + static_cast<double>(up));
    const double m_lo = 0.5 * (static_cast<double>(y) + static_cast<double>(dn));
    if (!below(m_hi))
      y = up;  // the true value is above the upper midpoint
    else if (below(m_lo))
      y = dn;  // ... or below the lower one
    else
      break;
  }
  return y;
}

inline void apply_element(float S, const CoeffsF& c, int opt, int ema_mode, float* theta, float* ema, float* state0,
                          float* state1, int64_t i) {
  const float G = S * c.inv_N;
  const float th = theta[i];
  float th_new;
  if (opt == M_SGD) {
    th_new = std::fmaf(-c.gamma, G, th);
  } else if (opt == M_MOMENTUM) {
    const float v = std::fmaf(c.mu, state0[i], G);
    state0[i] = v;
    th_new = std::fmaf(-c.gamma, v, th);
  } else {
    const float g2 = G * G;
    const float ms = std::fmaf(c.rho, state0[i], c.one_minus_rho * g2);
    const float step = (c.gamma * G) * rsqrt_rn(ms + c.eps);
    const float mom = std::fmaf(c.mu, state1[i], step);
    state0[i] = ms;
    state1[i] = mom;
    th_new = th - mom;
  }
  theta[i] = th_new;
  if (ema_mode != M_EMA_OFF) {
    const float operand = (ema_mode == M_EMA_POST) ? th_new : th;
    ema[i] = std::fmaf(c.alpha, ema[i], c.one_minus_alpha * operand);
  }
}

bool args_ok(int64_t P, int32_t M, const int64_t* shard_off, int32_t N, int opt, int ema_mode, const float* theta,
             const float* ema, const float* state0, const float* state1) {
  if (P < 0 || M < 1 || N < 1 || !shard_off || !theta) return false;
  if (shard_off[0] != 0 || shard_off[M] != P) return false;
  for (int32_t j = 0; j < M; ++j)
    if (shard_off[j + 1] < shard_off[j]) return false;
  if (opt < M_SGD || opt > M_RMSPROP_MOM || ema_mode < M_EMA_POST || ema_mode > M_EMA_OFF) return false;
  if (ema_mode != M_EMA_OFF && !ema) return false;
  if (opt != M_SGD && !state0) return false;
  if (opt == M_RMSPROP_MOM && !state1) return false;
  return true;
}

}  // namespace

extern "C" {

float mirror_rsqrt_rn(float x) { return rsqrt_rn(x); }

// One kept ROW per server (per_shard) and/or a per-row count; per_shard = 0, n_kept = status = NULL is the
// plain step.  slices != 0: grads is [W*M], entry k*M + j -> the len_j elements of worker k's G[j].
int mirror_aggregate_update_rows(int64_t P, int32_t M, const int64_t* shard_off, int32_t N, int32_t W,
                                 const void* const* grads, int grad_dtype, int slices, int per_shard,
                                 const int32_t* kept, int32_t kept_stride, const int32_t* n_kept,
                                 const int32_t* status, float* theta, float* ema, float* state0, float* state1,
                                 int opt, int ema_mode, float gamma_t, float alpha, float mu, float rho, float eps) {
  if (!args_ok(P, M, shard_off, N, opt, ema_mode, theta, ema, state0, state1)) return M_EINVAL;
  if (!grads || !kept || W < N || kept_stride < 1) return M_EINVAL;
  if (grad_dtype != M_F32 && grad_dtype != M_BF16) return M_EINVAL;
  for (int32_t j = 0; j < M; ++j) {
    const int32_t row = per_shard ? j : 0;
    if (status && status[row] != M_OK) continue;
    const int32_t n_j = n_kept ? n_kept[row] : N;
    if (n_j < 1 || n_j > kept_stride || n_j > W) return M_EINVAL;
    const int32_t* kept_j = kept + static_cast<int64_t>(row) * kept_stride;
    const CoeffsF c = make_coeffs(n_j, gamma_t, alpha, mu, rho, eps);
    const int64_t lo = shard_off[j], hi = shard_off[j + 1];
    for (int64_t i = lo; i < hi; ++i) {
      float S = 0.0f;
      for (int32_t n = 0; n < n_j; ++n) {
        const int32_t k = kept_j[n];
        S += slices ? grad_f32(grads[static_cast<int64_t>(k) * M + j], grad_dtype, i - lo)
                    : grad_f32(grads[k], grad_dtype, i);
      }
      apply_element(S, c, opt, ema_mode, theta, ema, state0, state1, i);
    }
  }
  return M_OK;
}

// S holds fp32 values (stored in double for the shim's sake): one fp32 addition per call and element.
int mirror_accumulate(double* S, const void* grad, int grad_dtype, int64_t P) {
  if (!S || !grad || P < 0) return M_EINVAL;
  for (int64_t i = 0; i < P; ++i)
    S[i] = static_cast<double>(static_cast<float>(S[i]) + grad_f32(grad, grad_dtype, i));
  return M_OK;
}

int mirror_apply_sum(int64_t P, int32_t M, const int64_t* shard_off, int32_t N, const double* S, float* theta,
                     float* ema, float* state0, float* state1, int opt, int ema_mode, float gamma_t, float alpha,
                     float mu, float rho, float eps) {
  if (!args_ok(P, M, shard_off, N, opt, ema_mode, theta, ema, state0, state1) || !S) return M_EINVAL;
  const CoeffsF c = make_coeffs(N, gamma_t, alpha, mu, rho, eps);
  for (int64_t i = 0; i < P; ++i) apply_element(static_cast<float>(S[i]), c, opt, ema_mode, theta, ema, state0, state1, i);
  return M_OK;
}

int mirror_ema(float* ema, const float* theta, int64_t P, float alpha) {
  if (!ema || !theta || P < 0) return M_EINVAL;
  const float oma = 1.0f - alpha;
  for (int64_t i = 0; i < P; ++i) ema[i] = std::fmaf(alpha, ema[i], oma * theta[i]);
  return M_OK;
}

// Alg. 2: K gradients one at a time; the i-th is scaled by gscales[i] (default 1) in the slot of inv_N.
int mirror_async_apply(int64_t P, int32_t M, const int64_t* shard_off, int32_t K, int32_t W,
                       const void* const* grads, int grad_dtype, const int32_t* order, const float* gammas,
                       const float* gscales, float* theta, float* ema, float* state0, float* state1, int opt,
                       int ema_mode, float gamma_t, float alpha, float mu, float rho, float eps) {
  if (!args_ok(P, M, shard_off, 1, opt, ema_mode, theta, ema, state0, state1)) return M_EINVAL;
  if (!grads || !order || K < 0 || K > W) return M_EINVAL;
  if (grad_dtype != M_F32 && grad_dtype != M_BF16) return M_EINVAL;
  for (int32_t i = 0; i < K; ++i) {
    if (order[i] < 0 || order[i] >= W || !grads[order[i]]) return M_EINVAL;
    CoeffsF c = make_coeffs(1, gammas ? gammas[i] : gamma_t, alpha, mu, rho, eps);
    c.inv_N = gscales ? gscales[i] : 1.0f;
    for (int64_t e = 0; e < P; ++e)
      apply_element(grad_f32(grads[order[i]], grad_dtype, e), c, opt, ema_mode, theta, ema, state0, state1, e);
  }
  return M_OK;
}

}  // extern "C"
