// psync CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, obviously-correct CPU statement of the parameter-server step of
// "Revisiting Distributed Synchronous SGD" (arXiv 1702.05800), Algorithm 4
// (de-interleaved in SURVEY.md section 2a):
//
//     G = {}; while |G| < N: wait for (G, t'); keep iff t' == t      (Alg. 4 l.2-6, L145-158)
//     theta(t+1)[j] <- theta(t)[j] - (gamma_t / N) * sum_{G in G} G[j] (Alg. 4 l.8,  L160)
//     ema(t)[j]     =  alpha * ema(t-1)[j] + (1 - alpha) * theta[j]    (Alg. 4 l.9,  L162; L40)
//
// with "the first N of N+b workers by arrival time are kept, the slowest b are
// dropped" (section 3).  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load this library.  It shares no code,
// header, table or helper with the CUDA path (paper_1702_05800_b200/csrc) and
// includes nothing but the C/C++ standard library.
//
// Arithmetic: every floating-point step is done in double on the fp32 (or bf16)
// stored inputs, and each stored result is rounded once to fp32 by
// static_cast<float>.  The scalar coefficients cross the interface as fp32 and the
// derived coefficients (1/N, 1-alpha, 1-rho) are formed in fp32 first, then widened
// (reading R8) -- the CUDA path does the same, so both sides multiply by
// the same real numbers.
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): selection against
// numpy's stable lexsort and exhaustive permutations; b=0 against numpy's mean;
// N=1 against the arg-min worker; exact rational brute force (fractions.Fraction,
// mpmath for the square root) for P <= 64; closed forms for constant gradients
// (SGD, momentum, RMSProp second moment) and the constant-theta EMA; optimizer
// reductions (mu=0, rho=1); a hand-worked dyadic example (tests/golden/).
// The functions added for SURVEY.md section 8(f) are pinned the same way: per-server rows and the
// time-out rule (tests/test_oracle_per_server.py), Alg. 2 (tests/test_oracle_async.py), learning-rate
// schedule and clip factors (tests/test_oracle_helpers.py), straggler statistics and the Fig. 5
// interpolation, the latter against the two values the paper prints (tests/test_oracle_stragglers.py);
// the per-(worker, server) slice layout (tests/test_oracle_slices.py); the staleness bookkeeping of Alg. 2
// (tests/test_oracle_staleness.py), Alg. 2 per server (tests/test_oracle_async.py) and the clip factors
// of sliced gradients (tests/test_oracle_helpers.py).
// (The fp32 diagnostic mirror of the GPU's operation list is a SEPARATE library, oracle/psync_mirror_f32.cpp;
// nothing of it is in this file.)
// Nothing here is "parity unpinned".
//
// Optional OpenMP (-fopenmp): the element loop is split over threads; per-element
// arithmetic and order are untouched, so results are bit-identical to one thread.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <utility>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// Status codes (values fixed by the oracle's own contract; tests compare numbers).
constexpr int ORACLE_OK = 0;
constexpr int ORACLE_EINVAL = -1;
constexpr int ORACLE_ETOOFEW = -2;

// Gradient element types.
constexpr int ORACLE_F32 = 0;
constexpr int ORACLE_BF16 = 1;

// Optimizers (a4 in SURVEY.md section 8a).
constexpr int ORACLE_SGD = 0;
constexpr int ORACLE_MOMENTUM = 1;
constexpr int ORACLE_RMSPROP_MOM = 2;

// EMA operand (reading R3).
constexpr int ORACLE_EMA_POST = 0;  // ema uses the freshly updated theta(t+1)
constexpr int ORACLE_EMA_PRE = 1;   // ema uses theta(t), the literal indexing of L162
constexpr int ORACLE_EMA_OFF = 2;

// bf16 -> double: a bf16 value is the upper 16 bits of an fp32 value; widening is exact.
inline double widen_bf16(uint16_t h) {
  uint32_t u = static_cast<uint32_t>(h) << 16;
  float f;
  std::memcpy(&f, &u, sizeof f);
  return static_cast<double>(f);
}

inline double grad_at(const void* g, int dtype, int64_t i) {
  if (dtype == ORACLE_F32) return static_cast<double>(static_cast<const float*>(g)[i]);
  return widen_bf16(static_cast<const uint16_t*>(g)[i]);
}

struct Coeffs {
  double gamma, alpha, one_minus_alpha, mu, rho, one_minus_rho, eps, inv_N;
};

// Derived coefficients formed in fp32, then widened (reading R8).
inline Coeffs make_coeffs(int32_t N, float gamma_t, float alpha, float mu, float rho, float eps) {
  Coeffs c;
  c.gamma = static_cast<double>(gamma_t);
  c.alpha = static_cast<double>(alpha);
  c.one_minus_alpha = static_cast<double>(1.0f - alpha);
  c.mu = static_cast<double>(mu);
  c.rho = static_cast<double>(rho);
  c.one_minus_rho = static_cast<double>(1.0f - rho);
  c.eps = static_cast<double>(eps);
  c.inv_N = static_cast<double>(1.0f / static_cast<float>(N));
  return c;
}

// One element of Alg. 4 l.8-9 given S = sum of the kept gradients at this element.
inline void apply_element(double S, const Coeffs& c, int opt, int ema_mode, float* theta, float* ema,
                          float* state0, float* state1, int64_t i) {
  const double G = S * c.inv_N;  // the mean gradient, (1/N) * sum   (L160)
  const double th = static_cast<double>(theta[i]);
  double th_new;
  if (opt == ORACLE_SGD) {
    // theta(t+1) = theta(t) - gamma_t * G                         (L40, L160)
    th_new = th - c.gamma * G;
  } else if (opt == ORACLE_MOMENTUM) {
    // v <- mu v + G ; theta <- theta - gamma_t v                   (reading R6)
    const double v = c.mu * static_cast<double>(state0[i]) + G;
    state0[i] = static_cast<float>(v);
    th_new = th - c.gamma * v;
  } else {
    // RMSProp with momentum, "decay" rho and "momentum" mu (L305, L315); the paper gives
    // no equations -- DESIGN.md reading R5:
    //   ms  <- rho ms + (1-rho) G^2
    //   mom <- mu mom + gamma_t G / sqrt(ms + eps)
    //   theta <- theta - mom
    const double ms = c.rho * static_cast<double>(state0[i]) + c.one_minus_rho * (G * G);
    const double mom = c.mu * static_cast<double>(state1[i]) + c.gamma * G / std::sqrt(ms + c.eps);
    state0[i] = static_cast<float>(ms);
    state1[i] = static_cast<float>(mom);
    th_new = th - mom;
  }
  const float th_new_f = static_cast<float>(th_new);
  theta[i] = th_new_f;
  if (ema_mode != ORACLE_EMA_OFF) {
    // ema = alpha * ema + (1 - alpha) * theta                      (L40, L162)
    // POST uses the stored (fp32) theta(t+1); PRE uses the stored theta(t).
    const double operand = (ema_mode == ORACLE_EMA_POST) ? static_cast<double>(th_new_f) : th;
    ema[i] = static_cast<float>(c.alpha * static_cast<double>(ema[i]) + c.one_minus_alpha * operand);
  }
}

bool args_ok(int64_t P, int32_t M, const int64_t* shard_off, int32_t N, int opt, int ema_mode,
             const float* theta, const float* ema, const float* state0, const float* state1) {
  if (P < 0 || M < 1 || N < 1 || !shard_off || !theta) return false;
  if (shard_off[0] != 0 || shard_off[M] != P) return false;
  for (int32_t j = 0; j < M; ++j)
    if (shard_off[j + 1] < shard_off[j]) return false;
  if (opt < ORACLE_SGD || opt > ORACLE_RMSPROP_MOM) return false;
  if (ema_mode < ORACLE_EMA_POST || ema_mode > ORACLE_EMA_OFF) return false;
  if (ema_mode != ORACLE_EMA_OFF && !ema) return false;
  if (opt != ORACLE_SGD && !state0) return false;
  if (opt == ORACLE_RMSPROP_MOM && !state1) return false;
  return true;
}

}  // namespace

extern "C" {

// ---------------------------------------------------------------------------------------------
// Selection: the first N of W = N+b workers by arrival time (L130; Alg. 4 l.3-6, L148-158).
//   arrival[W]  fp32 seconds; non-finite (NaN, +-inf) = never arrived (reading R13)
//   tags[W]     or NULL; worker k is eligible iff tags[k] == t  (Alg. 4 l.5: "if t' == t")
//   kept[N]     OUT ascending worker indices;  t_nth OUT (or NULL) the N-th smallest arrival
// Ties on arrival time go to the lower worker index (reading R1).  Fewer than N eligible
// workers -> ORACLE_ETOOFEW and kept / t_nth are left untouched.
// ---------------------------------------------------------------------------------------------
int oracle_select_first_n(const float* arrival, const int32_t* tags, int32_t t, int32_t N, int32_t b,
                          int32_t* kept, float* t_nth) {
  if (!arrival || !kept || N < 1 || b < 0) return ORACLE_EINVAL;
  const int32_t W = N + b;
  std::vector<std::pair<float, int32_t>> pairs;
  for (int32_t k = 0; k < W; ++k) {
    const bool eligible = std::isfinite(arrival[k]) && (tags == nullptr || tags[k] == t);
    if (eligible) pairs.emplace_back(arrival[k], k);
  }
  if (static_cast<int32_t>(pairs.size()) < N) return ORACLE_ETOOFEW;
  // Full sort by (time, worker index) with IEEE comparisons on the fp32 values (-0.0 == +0.0).
  std::sort(pairs.begin(), pairs.end(), [](const std::pair<float, int32_t>& x, const std::pair<float, int32_t>& y) {
    return x.first < y.first || (x.first == y.first && x.second < y.second);
  });
  std::vector<int32_t> first(N);
  for (int32_t i = 0; i < N; ++i) first[i] = pairs[i].second;
  std::sort(first.begin(), first.end());
  for (int32_t i = 0; i < N; ++i) kept[i] = first[i];
  if (t_nth) *t_nth = pairs[N - 1].first;
  return ORACLE_OK;
}

// ---------------------------------------------------------------------------------------------
// One whole step, Alg. 4 l.8-9, written per shard j and per element as the definition reads.
//   grads[W]     host pointers, each to P elements of grad_dtype laid out like theta
//   kept[N]      worker indices to aggregate, summed in the order given (ascending from select)
//   shard_off    [M+1], theta[j] = [shard_off[j], shard_off[j+1])
// theta, ema, state0, state1 are updated in place (fp32 storage).
// ---------------------------------------------------------------------------------------------
int oracle_aggregate_update(int64_t P, int32_t M, const int64_t* shard_off, int32_t N, int32_t W,
                            const void* const* grads, int grad_dtype, const int32_t* kept, float* theta,
                            float* ema, float* state0, float* state1, int opt, int ema_mode, float gamma_t,
                            float alpha, float mu, float rho, float eps) {
  if (!args_ok(P, M, shard_off, N, opt, ema_mode, theta, ema, state0, state1)) return ORACLE_EINVAL;
  if (!grads || !kept || W < N) return ORACLE_EINVAL;
  if (grad_dtype != ORACLE_F32 && grad_dtype != ORACLE_BF16) return ORACLE_EINVAL;
  for (int32_t n = 0; n < N; ++n)
    if (kept[n] < 0 || kept[n] >= W || !grads[kept[n]]) return ORACLE_EINVAL;
  const Coeffs c = make_coeffs(N, gamma_t, alpha, mu, rho, eps);
  for (int32_t j = 0; j < M; ++j) {  // parameter server j owns theta[j]   (L42)
    const int64_t lo = shard_off[j], hi = shard_off[j + 1];
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t i = lo; i < hi; ++i) {
      double S = 0.0;  // sum_{G in kept set} G[j]                  (L160)
      for (int32_t n = 0; n < N; ++n) S += grad_at(grads[kept[n]], grad_dtype, i);
      apply_element(S, c, opt, ema_mode, theta, ema, state0, state1, i);
    }
  }
  return ORACLE_OK;
}

// ---------------------------------------------------------------------------------------------
// The same step split in two so that a caller can stream the kept buffers one at a time (the
// paper-scale configs hold 10-20 GB of gradients): S[i] += G_k[i] for each kept k in ascending
// order, then oracle_apply_sum.  Per element the additions happen in the same order as in
// oracle_aggregate_update, so the two are bit-identical (tested).
// ---------------------------------------------------------------------------------------------
int oracle_accumulate(double* S, const void* grad, int grad_dtype, int64_t P) {
  if (!S || !grad || P < 0) return ORACLE_EINVAL;
  if (grad_dtype != ORACLE_F32 && grad_dtype != ORACLE_BF16) return ORACLE_EINVAL;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
  for (int64_t i = 0; i < P; ++i) S[i] += grad_at(grad, grad_dtype, i);
  return ORACLE_OK;
}

int oracle_apply_sum(int64_t P, int32_t M, const int64_t* shard_off, int32_t N, const double* S, float* theta,
                     float* ema, float* state0, float* state1, int opt, int ema_mode, float gamma_t, float alpha,
                     float mu, float rho, float eps) {
  if (!args_ok(P, M, shard_off, N, opt, ema_mode, theta, ema, state0, state1) || !S) return ORACLE_EINVAL;
  const Coeffs c = make_coeffs(N, gamma_t, alpha, mu, rho, eps);
  for (int32_t j = 0; j < M; ++j) {
    const int64_t lo = shard_off[j], hi = shard_off[j + 1];
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t i = lo; i < hi; ++i) apply_element(S[i], c, opt, ema_mode, theta, ema, state0, state1, i);
  }
  return ORACLE_OK;
}

// ema <- alpha * ema + (1 - alpha) * theta   (L40; Alg. 2 l.4 L87; Alg. 4 l.9 L162)
int oracle_ema(float* ema, const float* theta, int64_t P, float alpha) {
  if (!ema || !theta || P < 0) return ORACLE_EINVAL;
  const double a = static_cast<double>(alpha);
  const double oma = static_cast<double>(1.0f - alpha);
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
  for (int64_t i = 0; i < P; ++i)
    ema[i] = static_cast<float>(a * static_cast<double>(ema[i]) + oma * static_cast<double>(theta[i]));
  return ORACLE_OK;
}

// =============================================================================================
// NEXT-1: Algorithm 4 run LITERALLY per parameter server j.  The listing is
// titled "Sync-SGD Parameter Server j" (L134) and its wait loop (l.3-6, L148-158) runs on each
// server separately, so server j keeps the first N gradients that reach *it*: arrival times are a
// matrix arrival[M][W] (row j = the times at server j) and each server has its own kept set.
//   arrival[M*W]  row-major; tags[M*W] or NULL; kept[M*N] row j = server j's kept workers ascending
//   t_nth[M] or NULL; status[M]: ORACLE_OK or ORACLE_ETOOFEW per server (a failed server's kept
//   row and t_nth entry are left untouched).  Returns ORACLE_EINVAL on bad arguments, else OK.
// Each row is exactly oracle_select_first_n on that row.
// =============================================================================================
int oracle_select_first_n_sharded(const float* arrival, const int32_t* tags, int32_t t, int32_t N, int32_t b,
                                  int32_t M, int32_t* kept, float* t_nth, int32_t* status) {
  if (!arrival || !kept || !status || N < 1 || b < 0 || M < 1) return ORACLE_EINVAL;
  const int64_t W = static_cast<int64_t>(N) + b;
  for (int32_t j = 0; j < M; ++j)  // parameter server j waits for its own first N arrivals
    status[j] = oracle_select_first_n(arrival + j * W, tags ? tags + j * W : nullptr, t, N, b,
                                      kept + static_cast<int64_t>(j) * N, t_nth ? t_nth + j : nullptr);
  return ORACLE_OK;
}

// =============================================================================================
// NEXT-2: the time-out rule.  The paper only names it: "An alternative of
// using time-outs instead of backup workers is also being explored" (section 6).  Reading
// (R19): the server stops waiting at time `timeout`; every eligible worker (finite
// arrival, tag == t) whose gradient arrived by then (arrival <= timeout, IEEE compare on fp32) is
// kept, the rest are dropped; the update divides by the number actually kept, |G| (the mean of
// the gradients in hand, as L160 divides by N = |G|).  Fewer than min_keep (>= 1) kept ->
// ORACLE_ETOOFEW and nothing is written.
//   kept[W] OUT: the first *n_kept entries are the kept workers ascending; the rest untouched.
// =============================================================================================
int oracle_select_timeout(const float* arrival, const int32_t* tags, int32_t t, int32_t W, float timeout,
                          int32_t min_keep, int32_t* kept, int32_t* n_kept) {
  if (!arrival || !kept || !n_kept || W < 1 || min_keep < 1 || std::isnan(timeout)) return ORACLE_EINVAL;
  std::vector<int32_t> in_time;
  for (int32_t k = 0; k < W; ++k) {
    const bool eligible = std::isfinite(arrival[k]) && (tags == nullptr || tags[k] == t);
    if (eligible && arrival[k] <= timeout) in_time.push_back(k);
  }
  if (static_cast<int32_t>(in_time.size()) < min_keep) return ORACLE_ETOOFEW;
  for (size_t i = 0; i < in_time.size(); ++i) kept[i] = in_time[i];
  *n_kept = static_cast<int32_t>(in_time.size());
  return ORACLE_OK;
}

// =============================================================================================
// Alg. 4 l.8-9 with one kept ROW per parameter server and a per-row count (NEXT-1, NEXT-2):
//   row(j) = per_shard ? j : 0
//   kept_j = kept[row * kept_stride .. + n_j),  n_j = n_kept ? n_kept[row] : N
//   server j is skipped (theta[j], state[j], ema[j] untouched) when status && status[row] != OK
//   theta(t+1)[j] = theta(t)[j] - (gamma_t / n_j) * sum_{k in kept_j} G_k[j]           (L160)
// The divisor 1/n_j is formed in fp32 (reading R8), like 1/N.
// =============================================================================================
int oracle_aggregate_update_rows(int64_t P, int32_t M, const int64_t* shard_off, int32_t N, int32_t W,
                                 const void* const* grads, int grad_dtype, int per_shard, const int32_t* kept,
                                 int32_t kept_stride, const int32_t* n_kept, const int32_t* status, float* theta,
                                 float* ema, float* state0, float* state1, int opt, int ema_mode, float gamma_t,
                                 float alpha, float mu, float rho, float eps) {
  if (!args_ok(P, M, shard_off, N, opt, ema_mode, theta, ema, state0, state1)) return ORACLE_EINVAL;
  if (!grads || !kept || W < N || kept_stride < 1) return ORACLE_EINVAL;
  if (grad_dtype != ORACLE_F32 && grad_dtype != ORACLE_BF16) return ORACLE_EINVAL;
  for (int32_t j = 0; j < M; ++j) {  // validate every live row before anything is written
    const int32_t row = per_shard ? j : 0;
    if (status && status[row] != ORACLE_OK) continue;
    const int32_t n_j = n_kept ? n_kept[row] : N;
    if (n_j < 1 || n_j > kept_stride || n_j > W) return ORACLE_EINVAL;
    const int32_t* kept_j = kept + static_cast<int64_t>(row) * kept_stride;
    for (int32_t n = 0; n < n_j; ++n)
      if (kept_j[n] < 0 || kept_j[n] >= W || !grads[kept_j[n]]) return ORACLE_EINVAL;
  }
  for (int32_t j = 0; j < M; ++j) {  // parameter server j owns theta[j]   (L42)
    const int32_t row = per_shard ? j : 0;
    if (status && status[row] != ORACLE_OK) continue;  // this server never collected its gradients
    const int32_t n_j = n_kept ? n_kept[row] : N;
    const int32_t* kept_j = kept + static_cast<int64_t>(row) * kept_stride;
    const Coeffs c = make_coeffs(n_j, gamma_t, alpha, mu, rho, eps);
    const int64_t lo = shard_off[j], hi = shard_off[j + 1];
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t i = lo; i < hi; ++i) {
      double S = 0.0;  // sum over server j's own kept set
      for (int32_t n = 0; n < n_j; ++n) S += grad_at(grads[kept_j[n]], grad_dtype, i);
      apply_element(S, c, opt, ema_mode, theta, ema, state0, state1, i);
    }
  }
  return ORACLE_OK;
}

// =============================================================================================
// NEXT-1, companion layout (SURVEY.md section 8b last line, 8f NEXT-1): what parameter server j RECEIVES.
// Alg. 4 is the program of ONE server j (L134): it waits for "(G, t') from any worker" (l.4, L152) and uses
// only G[j] (l.8, L160) -- worker k sends server j the slice G_k[j] of its gradient, as server j owns
// only theta[j] (L42).  So the gradients of one step are W*M separate buffers, one per (worker, server):
//   grad_slices[k*M + j] -> the len_j = shard_off[j+1] - shard_off[j] elements of G_k[j]
// (element i of that buffer belongs to parameter shard_off[j] + i), each its own allocation with its own
// alignment; nothing is assumed about where they lie relative to one another.  Entries of workers that
// are not kept by server j are never dereferenced (they may be NULL); an empty server (len_j = 0) needs
// no buffers at all.  Everything else -- kept rows, per-row counts, status, the divisor 1/n_j formed in
// fp32, the update and the EMA -- is oracle_aggregate_update_rows' (per_shard = 0: row 0 serves every
// server, n_kept = NULL: exactly N workers, status = NULL: every server is live):
//   theta(t+1)[j] = theta(t)[j] - (gamma_t / n_j) * sum_{k in kept_j, ascending} G_k[j]            (L160)
// =============================================================================================
int oracle_aggregate_update_slices(int64_t P, int32_t M, const int64_t* shard_off, int32_t N, int32_t W,
                                   const void* const* grad_slices, int grad_dtype, int per_shard,
                                   const int32_t* kept, int32_t kept_stride, const int32_t* n_kept,
                                   const int32_t* status, float* theta, float* ema, float* state0, float* state1,
                                   int opt, int ema_mode, float gamma_t, float alpha, float mu, float rho, float eps) {
  if (!args_ok(P, M, shard_off, N, opt, ema_mode, theta, ema, state0, state1)) return ORACLE_EINVAL;
  if (!grad_slices || !kept || W < N || kept_stride < 1) return ORACLE_EINVAL;
  if (grad_dtype != ORACLE_F32 && grad_dtype != ORACLE_BF16) return ORACLE_EINVAL;
  for (int32_t j = 0; j < M; ++j) {  // validate every live row before anything is written
    const int32_t row = per_shard ? j : 0;
    if (status && status[row] != ORACLE_OK) continue;
    const int32_t n_j = n_kept ? n_kept[row] : N;
    if (n_j < 1 || n_j > kept_stride || n_j > W) return ORACLE_EINVAL;
    const int32_t* kept_j = kept + static_cast<int64_t>(row) * kept_stride;
    const int64_t len_j = shard_off[j + 1] - shard_off[j];
    for (int32_t n = 0; n < n_j; ++n) {
      if (kept_j[n] < 0 || kept_j[n] >= W) return ORACLE_EINVAL;
      if (len_j > 0 && !grad_slices[static_cast<int64_t>(kept_j[n]) * M + j]) return ORACLE_EINVAL;
    }
  }
  for (int32_t j = 0; j < M; ++j) {  // parameter server j owns theta[j]   (L42)
    const int32_t row = per_shard ? j : 0;
    if (status && status[row] != ORACLE_OK) continue;  // this server never collected its gradients
    const int32_t n_j = n_kept ? n_kept[row] : N;
    const int32_t* kept_j = kept + static_cast<int64_t>(row) * kept_stride;
    const Coeffs c = make_coeffs(n_j, gamma_t, alpha, mu, rho, eps);
    const int64_t lo = shard_off[j], len_j = shard_off[j + 1] - shard_off[j];
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t i = 0; i < len_j; ++i) {  // element i of what server j received = parameter lo + i
      double S = 0.0;                      // sum_{G in kept set of server j} G[j]              (L160)
      for (int32_t n = 0; n < n_j; ++n)
        S += grad_at(grad_slices[static_cast<int64_t>(kept_j[n]) * M + j], grad_dtype, i);
      apply_element(S, c, opt, ema_mode, theta, ema, state0, state1, lo + i);
    }
  }
  return ORACLE_OK;
}

// =============================================================================================
// NEXT-3: Algorithm 2, "Async-SGD Parameter Server j" --
// the paper's comparison method:
//     for t = 0, 1, ...:  wait for gradient G from any worker               (L85)
//                         theta(t+1)[j] <- theta(t)[j] - gamma_t G[j]       (L86)
//                         ema(t)[j] = alpha ema(t-1)[j] + (1-alpha) theta(t)[j]   (L87)
// Every arriving gradient is one iteration; nothing is dropped and no tag is checked.
//
// oracle_order_by_arrival: the order in which the W gradients reach the server = ascending
// (arrival time, worker index) over the workers whose time is finite (reading R13: non-finite =
// never arrived).  order[0..*n_arrived) OUT; the rest of order[] is left untouched.
// =============================================================================================
int oracle_order_by_arrival(const float* arrival, int32_t W, int32_t* order, int32_t* n_arrived) {
  if (!arrival || !order || !n_arrived || W < 1) return ORACLE_EINVAL;
  std::vector<std::pair<float, int32_t>> pairs;
  for (int32_t k = 0; k < W; ++k)
    if (std::isfinite(arrival[k])) pairs.emplace_back(arrival[k], k);
  std::stable_sort(pairs.begin(), pairs.end(),
                   [](const std::pair<float, int32_t>& x, const std::pair<float, int32_t>& y) {
                     return x.first < y.first;  // stable: equal times keep ascending worker index
                   });
  for (size_t i = 0; i < pairs.size(); ++i) order[i] = pairs[i].second;
  *n_arrived = static_cast<int32_t>(pairs.size());
  return ORACLE_OK;
}

// oracle_async_apply: K iterations of Alg. 2, one per gradient, in the order given:
//   for i = 0..K-1:  G = grads[order[i]] (times gscales[i] if given);  gamma = gammas ? gammas[i] : gamma_t
//                    every element: optimizer step with G (no averaging: the divisor is 1), then EMA
// written as the paper's loop reads -- outer loop over arrivals, inner loop over the parameters of
// each server j -- with theta / state / ema stored as fp32 after every iteration (they are the
// server's stored state between arrivals).  The optimizer variants and the EMA operand are those of
// the synchronous step (readings R3, R5, R6); EMA_PRE is the literal indexing of L87.
int oracle_async_apply(int64_t P, int32_t M, const int64_t* shard_off, int32_t K, int32_t W,
                       const void* const* grads, int grad_dtype, const int32_t* order, const float* gammas,
                       const float* gscales, float* theta, float* ema, float* state0, float* state1, int opt,
                       int ema_mode, float gamma_t, float alpha, float mu, float rho, float eps) {
  if (!args_ok(P, M, shard_off, 1, opt, ema_mode, theta, ema, state0, state1)) return ORACLE_EINVAL;
  if (!grads || !order || K < 0 || K > W) return ORACLE_EINVAL;
  if (grad_dtype != ORACLE_F32 && grad_dtype != ORACLE_BF16) return ORACLE_EINVAL;
  for (int32_t i = 0; i < K; ++i)
    if (order[i] < 0 || order[i] >= W || !grads[order[i]]) return ORACLE_EINVAL;
  for (int32_t i = 0; i < K; ++i) {  // iteration t+i: "wait for gradient G from any worker"
    const void* G = grads[order[i]];
    Coeffs c = make_coeffs(1, gammas ? gammas[i] : gamma_t, alpha, mu, rho, eps);
    // global-norm clipping (L313; R22): the i-th gradient is scaled by gscales[i] before the update.
    // apply_element multiplies the gradient by c.inv_N, which is 1 here, so the clip factor takes its place.
    if (gscales) c.inv_N = static_cast<double>(gscales[i]);
    for (int32_t j = 0; j < M; ++j) {  // parameter server j
      const int64_t lo = shard_off[j], hi = shard_off[j + 1];
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
      for (int64_t e = lo; e < hi; ++e)
        apply_element(grad_at(G, grad_dtype, e), c, opt, ema_mode, theta, ema, state0, state1, e);
    }
  }
  return ORACLE_OK;
}

// =============================================================================================
// Alg. 2 run LITERALLY per parameter server j on what it receives.  The listing is "Async-SGD Parameter Server j"
// (L78): each server has its own loop "wait for gradient G from any worker" (L85) and applies G[j] (L86), so the
// order in which the gradients are applied, and how many have arrived, may differ from server to server (the
// same remark as for Alg. 4).  Row r(j) = per_shard ? j : 0 of `order` (stride order_stride) lists the
// workers in the order server j applies them, K_j = n_arrived ? n_arrived[r] : K of them.
//   slices != 0: grads is [W*M], entry k*M + j -> the len_j elements of worker k's G_k[j] (element i = parameter
//                shard_off[j] + i); else grads is [W] flat buffers.
//   gammas[i]  learning rate of the server's i-th iteration of this batch (or NULL: gamma_t for all);
//   gscales[k] global-norm clip factor of WORKER k's gradient (L313), or NULL (= 1);
//   status[r]  != OK: server j applies nothing (its slice is untouched).
// Per server the arithmetic is oracle_async_apply's: outer loop over the arrivals, inner loop over the server's
// parameters, one optimizer step (divisor 1) and one EMA per arrival, stored as fp32 after every iteration.
// =============================================================================================
int oracle_async_apply_rows(int64_t P, int32_t M, const int64_t* shard_off, int32_t K, int32_t W,
                            const void* const* grads, int grad_dtype, int slices, int per_shard, const int32_t* order,
                            int32_t order_stride, const int32_t* n_arrived, const int32_t* status, const float* gammas,
                            const float* gscales, float* theta, float* ema, float* state0, float* state1, int opt,
                            int ema_mode, float gamma_t, float alpha, float mu, float rho, float eps) {
  if (!args_ok(P, M, shard_off, 1, opt, ema_mode, theta, ema, state0, state1)) return ORACLE_EINVAL;
  if (!grads || !order || K < 0 || K > W || order_stride < 1) return ORACLE_EINVAL;
  if (grad_dtype != ORACLE_F32 && grad_dtype != ORACLE_BF16) return ORACLE_EINVAL;
  for (int32_t j = 0; j < M; ++j) {  // validate every live row before anything is written
    const int32_t row = per_shard ? j : 0;
    if (status && status[row] != ORACLE_OK) continue;
    const int32_t K_j = n_arrived ? n_arrived[row] : K;
    if (K_j < 0 || K_j > order_stride || K_j > W) return ORACLE_EINVAL;
    const int64_t len_j = shard_off[j + 1] - shard_off[j];
    for (int32_t i = 0; i < K_j; ++i) {
      const int32_t k = order[static_cast<int64_t>(row) * order_stride + i];
      if (k < 0 || k >= W) return ORACLE_EINVAL;
      if (len_j > 0 && !grads[slices ? static_cast<int64_t>(k) * M + j : k]) return ORACLE_EINVAL;
    }
  }
  for (int32_t j = 0; j < M; ++j) {  // parameter server j
    const int32_t row = per_shard ? j : 0;
    if (status && status[row] != ORACLE_OK) continue;
    const int32_t K_j = n_arrived ? n_arrived[row] : K;
    const int64_t lo = shard_off[j], len_j = shard_off[j + 1] - shard_off[j];
    for (int32_t i = 0; i < K_j; ++i) {  // its i-th iteration: "wait for gradient G from any worker"   (L85)
      const int32_t k = order[static_cast<int64_t>(row) * order_stride + i];
      Coeffs c = make_coeffs(1, gammas ? gammas[i] : gamma_t, alpha, mu, rho, eps);
      if (gscales) c.inv_N = static_cast<double>(gscales[k]);  // the clip factor takes the place of 1/N = 1
      const void* G = slices ? grads[static_cast<int64_t>(k) * M + j] : grads[k];
      const int64_t g0 = slices ? 0 : lo;  // where server j's part starts in that buffer
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
      for (int64_t e = 0; e < len_j; ++e)  // theta(t+1)[j] <- theta(t)[j] - gamma_t G[j]; then the EMA   (L86-87)
        apply_element(grad_at(G, grad_dtype, g0 + e), c, opt, ema_mode, theta, ema, state0, state1, lo + e);
    }
  }
  return ORACLE_OK;
}

// =============================================================================================
// Staleness of the gradients Alg. 2 applies (NEXT-3, remainder): "Staleness of a gradient is measured as the
// number of updates that have occurred between its corresponding read and update operations" (Table 1,
// PAPER.md:L103-110).  The server counts its updates t = 0, 1, ... (Alg. 2's loop variable, L84).  Worker k
// read theta when the counter stood at read_iter[k] (Alg. 1 l.2, L64); the gradient it computed from that
// copy is the i-th one the server applies in this batch, as update number t0 + lag + i, so
//     staleness_i = (t0 + lag + i) - read_iter[order[i]]
// updates were applied in between.  `lag` >= 0 is the fixed-lag simulation of section 2.1 (L114: "simulated
// staleness by using old gradients for the parameter updates"): every gradient waits `lag` further updates
// before it is applied, which adds exactly `lag` to its staleness.  After its gradient has been applied the
// worker reads again (Alg. 1 is a loop: send, then read, L62-75): read_iter_out[k] = t0 + lag + i + 1, the counter
// right after its own update; workers not in `order` keep their value.
//   read_iter[W] int64 (>= 0, <= the update index it is compared with, else EINVAL: a gradient cannot be
//   computed from parameters that do not exist yet);  order[K] distinct worker indices;  t0 >= 0
//   staleness[K] int64 OUT;  read_iter_out[W] int64 OUT (may alias read_iter);
//   stats[6] double OUT: min, mean, median, max, standard deviation (population: divide by K), count --
//   the columns of Table 1.  K = 0: stats = NaN, NaN, NaN, NaN, NaN, 0.
// =============================================================================================
int oracle_staleness(const int64_t* read_iter, int32_t W, const int32_t* order, int32_t K, int64_t t0, int32_t lag,
                     int64_t* staleness, int64_t* read_iter_out, double* stats) {
  if (!read_iter || !order || !staleness || !read_iter_out || !stats || W < 1 || K < 0 || K > W || t0 < 0 || lag < 0)
    return ORACLE_EINVAL;
  std::vector<char> seen(W, 0);
  for (int32_t i = 0; i < K; ++i) {
    const int32_t k = order[i];
    if (k < 0 || k >= W || seen[k]) return ORACLE_EINVAL;
    seen[k] = 1;
    if (read_iter[k] < 0 || read_iter[k] > t0 + lag + i) return ORACLE_EINVAL;
  }
  std::vector<int64_t> next(read_iter, read_iter + W);
  for (int32_t i = 0; i < K; ++i) {  // the i-th gradient to arrive is update number t0 + lag + i
    const int64_t applied_as = t0 + lag + i;
    staleness[i] = applied_as - read_iter[order[i]];
    next[order[i]] = applied_as + 1;  // the worker's next read sees its own update
  }
  for (int32_t k = 0; k < W; ++k) read_iter_out[k] = next[k];
  const double nan = std::numeric_limits<double>::quiet_NaN();
  if (K == 0) {
    stats[0] = stats[1] = stats[2] = stats[3] = stats[4] = nan;
    stats[5] = 0.0;
    return ORACLE_OK;
  }
  std::vector<int64_t> sorted(staleness, staleness + K);
  std::sort(sorted.begin(), sorted.end());
  double sum = 0.0;
  for (int32_t i = 0; i < K; ++i) sum += static_cast<double>(staleness[i]);
  const double mean = sum / K;
  double ss = 0.0;
  for (int32_t i = 0; i < K; ++i) ss += (static_cast<double>(staleness[i]) - mean) * (static_cast<double>(staleness[i]) - mean);
  stats[0] = static_cast<double>(sorted.front());
  stats[1] = mean;
  stats[2] = (K % 2) ? static_cast<double>(sorted[K / 2])
                     : 0.5 * (static_cast<double>(sorted[K / 2 - 1]) + static_cast<double>(sorted[K / 2]));
  stats[3] = static_cast<double>(sorted.back());
  stats[4] = std::sqrt(ss / K);
  stats[5] = static_cast<double>(K);
  return ORACLE_OK;
}

// =============================================================================================
// NEXT-4 helpers.
//
// Learning-rate schedule of A.2 / A.3 (L305, L315): gamma_t = gamma_0 * beta^(t * s) with
// s = N/(2T) for Sync-Opt and s = 1/(2T) for Async-Opt, T = |X|/B mini-batches per epoch
// ("exponentially decreased with decay rate beta = 0.94 as gamma_0 beta^(tN/(2T))").  out[i] is the
// rate of iteration t0 + i, computed in double and rounded once to fp32.
// =============================================================================================
int oracle_lr_schedule(float gamma0, float beta, int64_t t0, int32_t K, double s, float* out) {
  if (!out || K < 0 || t0 < 0 || !(beta > 0.0f)) return ORACLE_EINVAL;
  for (int32_t i = 0; i < K; ++i)
    out[i] = static_cast<float>(static_cast<double>(gamma0) *
                                std::pow(static_cast<double>(beta), static_cast<double>(t0 + i) * s));
  return ORACLE_OK;
}

// Global-norm clipping of Async-Opt (A.3, L313: "collect the gradient across all layers of the deep
// model, compute the global norm ||G|| and then clip all gradient accordingly").  The paper gives no
// formula; reading R22 (the TensorFlow operation it ran on, L197): G <- G * clip / max(||G||, clip),
// ||G|| the Euclidean norm over ALL P elements of one worker's gradient.  scales[k] is that factor for
// worker k's buffer, computed in double and rounded once to fp32 (1 when the norm is within the bound;
// a non-finite norm gives a NaN/0 factor per IEEE, as the definition reads).
int oracle_clip_scales(const void* const* grads, int32_t W, int64_t P, int grad_dtype, float clip, float* scales) {
  if (!grads || !scales || W < 1 || P < 0 || !(clip > 0.0f)) return ORACLE_EINVAL;
  if (grad_dtype != ORACLE_F32 && grad_dtype != ORACLE_BF16) return ORACLE_EINVAL;
  for (int32_t k = 0; k < W; ++k) {
    if (!grads[k]) return ORACLE_EINVAL;
    double sumsq = 0.0;
    for (int64_t i = 0; i < P; ++i) {
      const double g = grad_at(grads[k], grad_dtype, i);
      sumsq += g * g;
    }
    const double norm = std::sqrt(sumsq);
    const double c = static_cast<double>(clip);
    scales[k] = static_cast<float>(c / std::max(norm, c));
  }
  return ORACLE_OK;
}

// The same factor when worker k's gradient lies as M per-(worker, server) slices (grads is [W*M], entry k*M + j ->
// the len_j elements of G_k[j]; reading R24).  "Collect the gradient across all layers ... compute the global norm"
// (L313): the norm is over ALL of worker k's slices -- the squares are added server by server, element by element,
// i.e. in the order of the flat vector.  Every slice of a non-empty server must be present.
int oracle_clip_scales_slices(const void* const* grads, int32_t W, int32_t M, const int64_t* shard_off, int grad_dtype,
                              float clip, float* scales) {
  if (!grads || !scales || !shard_off || W < 1 || M < 1 || !(clip > 0.0f)) return ORACLE_EINVAL;
  if (grad_dtype != ORACLE_F32 && grad_dtype != ORACLE_BF16) return ORACLE_EINVAL;
  if (shard_off[0] != 0) return ORACLE_EINVAL;
  for (int32_t j = 0; j < M; ++j)
    if (shard_off[j + 1] < shard_off[j]) return ORACLE_EINVAL;
  for (int32_t k = 0; k < W; ++k)
    for (int32_t j = 0; j < M; ++j)
      if (shard_off[j + 1] > shard_off[j] && !grads[static_cast<int64_t>(k) * M + j]) return ORACLE_EINVAL;
  for (int32_t k = 0; k < W; ++k) {
    double sumsq = 0.0;
    for (int32_t j = 0; j < M; ++j) {  // server j's part of worker k's gradient
      const void* G = grads[static_cast<int64_t>(k) * M + j];
      const int64_t len_j = shard_off[j + 1] - shard_off[j];
      for (int64_t i = 0; i < len_j; ++i) {
        const double g = grad_at(G, grad_dtype, i);
        sumsq += g * g;
      }
    }
    const double norm = std::sqrt(sumsq);
    const double c = static_cast<double>(clip);
    scales[k] = static_cast<float>(c / std::max(norm, c));
  }
  return ORACLE_OK;
}

// =============================================================================================
// Straggler statistics -- the PROCEDURE of section 3.1 (L171-193), on whatever arrival times are
// supplied: "we collected for each iteration both the start time of the iteration and the time when
// the kth gradient ... arrived at the parameter server" (L171; Fig. 3 is the CDF of these per k),
// "Mean and median times, across all iterations, to collect k gradients" (Fig. 4), and "We can
// multiply this with the mean iteration times (Figure 4) to obtain the running time required to
// converge for each setting of N and b" (Fig. 6).
//   arrival[T][W]  times since each iteration's start; non-finite = never arrived
//   sorted[T][W]   OUT: row t ascending; entry k = time the (k+1)-th gradient arrived; missing = +inf
//   count[W], mean[W], median[W]  OUT over the iterations in which a (k+1)-th gradient arrived
//                  (mean/median are NaN where count is 0; median of an even count = mean of the two
//                  middle values)
//   iters[W] or NULL, est_time[W] OUT or NULL: est_time[k] = mean[k] * iters[k], iters[k] = iterations
//                  to converge when aggregating k+1 gradients (Fig. 5, supplied by the caller)
// =============================================================================================
int oracle_kth_arrival_stats(const float* arrival, int32_t T, int32_t W, float* sorted, int32_t* count,
                             double* mean, double* median, const double* iters, double* est_time) {
  if (!arrival || !sorted || !count || !mean || !median || T < 1 || W < 1) return ORACLE_EINVAL;
  if ((iters == nullptr) != (est_time == nullptr)) return ORACLE_EINVAL;
  const float inf = std::numeric_limits<float>::infinity();
  for (int32_t t = 0; t < T; ++t) {
    std::vector<float> row;
    for (int32_t k = 0; k < W; ++k)
      if (std::isfinite(arrival[static_cast<int64_t>(t) * W + k])) row.push_back(arrival[static_cast<int64_t>(t) * W + k]);
    std::sort(row.begin(), row.end());
    for (int32_t k = 0; k < W; ++k)
      sorted[static_cast<int64_t>(t) * W + k] = k < static_cast<int32_t>(row.size()) ? row[k] : inf;
  }
  for (int32_t k = 0; k < W; ++k) {
    std::vector<float> col;
    for (int32_t t = 0; t < T; ++t)
      if (std::isfinite(sorted[static_cast<int64_t>(t) * W + k])) col.push_back(sorted[static_cast<int64_t>(t) * W + k]);
    count[k] = static_cast<int32_t>(col.size());
    if (col.empty()) {
      mean[k] = median[k] = std::numeric_limits<double>::quiet_NaN();
    } else {
      double sum = 0.0;
      for (float v : col) sum += static_cast<double>(v);
      mean[k] = sum / static_cast<double>(col.size());
      std::sort(col.begin(), col.end());
      const size_t n = col.size();
      median[k] = (n % 2) ? static_cast<double>(col[n / 2])
                          : 0.5 * (static_cast<double>(col[n / 2 - 1]) + static_cast<double>(col[n / 2]));
    }
    if (est_time) est_time[k] = mean[k] * iters[k];
  }
  return ORACLE_OK;
}

// Iterations to converge as a function of N, for Fig. 6's estimate: "we can estimate the iterations required
// from Figure 5 (linearly interpolating for values of N for which we did not collect data)" (L193).
//   N_pts[n_pts] strictly ascending worker counts with measured iterations iters_pts[n_pts]
//   iters[W] OUT: entry k is the value for N = k+1 gradients; below the first / above the last measured N the
//   nearest measured value is held (the paper interpolates only; reading R23).
int oracle_interp_iterations(const int32_t* N_pts, const double* iters_pts, int32_t n_pts, int32_t W, double* iters) {
  if (!N_pts || !iters_pts || !iters || n_pts < 1 || W < 1) return ORACLE_EINVAL;
  for (int32_t p = 1; p < n_pts; ++p)
    if (N_pts[p] <= N_pts[p - 1]) return ORACLE_EINVAL;
  for (int32_t k = 0; k < W; ++k) {
    const int32_t N = k + 1;
    if (N <= N_pts[0]) {
      iters[k] = iters_pts[0];
    } else if (N >= N_pts[n_pts - 1]) {
      iters[k] = iters_pts[n_pts - 1];
    } else {
      int32_t p = 0;
      while (N_pts[p + 1] < N) ++p;  // N_pts[p] < N <= N_pts[p+1]
      const double num = (iters_pts[p + 1] - iters_pts[p]) * static_cast<double>(N - N_pts[p]);
      iters[k] = iters_pts[p] + num / static_cast<double>(N_pts[p + 1] - N_pts[p]);
    }
  }
  return ORACLE_OK;
}

// Threads the element loops use (1 without OpenMP); bench.py reports it as cpu_baseline.cores.
int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void oracle_set_num_threads(int n) {
#ifdef _OPENMP
  if (n >= 1) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

}  // extern "C"
