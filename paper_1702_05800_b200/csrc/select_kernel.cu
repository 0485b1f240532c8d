// K1: keep the first N of the W = N+b workers by arrival time -- one warp, no sort.
//
// Defines: PAPER.md section 3 (L130): "as soon as the parameter servers receive gradients from
// any N workers, they stop waiting ... The slowest b workers' gradients will be dropped", and
// Alg. 4 l.3-6 (L148-158): a gradient counts only if its tag t' equals the server's t.
//
// Method (B200: one warp's ballots and shuffles are enough for W <= 1024 keys, ~microseconds):
//   1. each fp32 arrival time becomes an order-preserving uint32 key (after -0.0 -> +0.0);
//      ineligible workers (non-finite time or stale tag) get the key 0xFFFFFFFF, which no
//      finite time maps to and which sorts last;
//   2. the N-th smallest key tau is found by a 32-pass MSB-first radix select
//      (per pass: count the still-matching keys whose current bit is 0, warp-reduce);
//   3. worker k is kept iff key_k < tau, or key_k == tau and k is among the first
//      (N - #{key < tau}) such workers in index order (ties go to the lower index, reading R1).
// Lanes own CONTIGUOUS index ranges, so a warp exclusive scan of the per-lane kept counts
// gives every lane its output offset and the list comes out in ascending worker order.

#include "psync_kernels.cuh"

namespace psync {
namespace {

constexpr uint32_t kIneligible = 0xFFFFFFFFu;
constexpr int kStatusOk = 0;
constexpr int kStatusTooFew = -2;

__device__ __forceinline__ uint32_t arrival_key(float a) {
  uint32_t u = __float_as_uint(a);
  if ((u & 0x7F800000u) == 0x7F800000u) return kIneligible;  // NaN, +inf, -inf: never arrived
  if (u == 0x80000000u) u = 0u;                              // -0.0 == +0.0
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

__device__ __forceinline__ float key_to_time(uint32_t key) {
  const uint32_t u = (key & 0x80000000u) ? (key & 0x7FFFFFFFu) : ~key;
  return __uint_as_float(u);
}

__device__ __forceinline__ int warp_exclusive_scan(int v, int lane, int* total) {
  int incl = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int up = __shfl_up_sync(0xFFFFFFFFu, incl, d);
    if (lane >= d) incl += up;
  }
  *total = __shfl_sync(0xFFFFFFFFu, incl, 31);
  return incl - v;
}

__global__ void __launch_bounds__(32) select_first_n_kernel(const float* __restrict__ arrival,
                                                            const int32_t* __restrict__ tags, int32_t t, int32_t N,
                                                            int32_t W, int32_t* __restrict__ kept,
                                                            float* __restrict__ t_nth, int32_t* __restrict__ status) {
  // key of worker k lives at s_key[(k % c) * 32 + k / c]: lane k / c owns workers [lane*c, lane*c + c)
  // and reads row i of its range at s_key[i * 32 + lane] -- conflict-free.
  __shared__ uint32_t s_key[kMaxWorkers];
  const int lane = threadIdx.x;
  const int c = (W + 31) >> 5;  // keys per lane, 1..32

  int n_elig = 0;
  for (int k = lane; k < c * 32; k += 32) {  // coalesced global reads
    uint32_t key = kIneligible;
    if (k < W) {
      key = arrival_key(arrival[k]);
      if (tags != nullptr && tags[k] != t) key = kIneligible;  // Alg. 4 l.5-6: t' != t -> dropped
    }
    n_elig += (key != kIneligible);
    s_key[(k % c) * 32 + (k / c)] = key;
  }
  n_elig = __reduce_add_sync(0xFFFFFFFFu, n_elig);
  __syncwarp();
  if (n_elig < N) {  // |G| can never reach N this step
    if (lane == 0) *status = kStatusTooFew;
    return;
  }

  // radix select: tau = key of rank N-1 (0-based) among all keys (ineligible keys sort last)
  uint32_t prefix = 0u;
  int r = N - 1;
  for (int bit = 31; bit >= 0; --bit) {
    const uint32_t hi_mask = (bit == 31) ? 0u : (0xFFFFFFFFu << (bit + 1));
    int zeros = 0;
    for (int i = 0; i < c; ++i) {
      const uint32_t key = s_key[i * 32 + lane];
      zeros += (((key & hi_mask) == prefix) && (((key >> bit) & 1u) == 0u));
    }
    zeros = __reduce_add_sync(0xFFFFFFFFu, zeros);
    if (r >= zeros) {
      r -= zeros;
      prefix |= (1u << bit);
    }
  }
  const uint32_t tau = prefix;
  const int eq_take = r + 1;  // how many of the workers tied at tau are kept, lowest indices first

  int n_less = 0, n_eq = 0;
  for (int i = 0; i < c; ++i) {
    const uint32_t key = s_key[i * 32 + lane];
    n_less += (key < tau);
    n_eq += (key == tau);
  }
  int total_eq, total_kept;
  const int eq_before = warp_exclusive_scan(n_eq, lane, &total_eq);
  int my_eq = eq_take - eq_before;
  my_eq = my_eq < 0 ? 0 : (my_eq > n_eq ? n_eq : my_eq);
  int out = warp_exclusive_scan(n_less + my_eq, lane, &total_kept);  // total_kept == N

  for (int i = 0; i < c; ++i) {  // ascending worker index within the lane's range
    const uint32_t key = s_key[i * 32 + lane];
    bool keep = key < tau;
    if (key == tau && my_eq > 0) {
      keep = true;
      --my_eq;
    }
    if (keep) kept[out++] = lane * c + i;
  }
  if (lane == 0) {
    *status = kStatusOk;
    if (t_nth != nullptr) *t_nth = key_to_time(tau);
  }
}

}  // namespace

cudaError_t launch_select_first_n(const float* d_arrival, const int32_t* d_tags, int32_t t, int32_t N, int32_t W,
                                  int32_t* d_kept, float* d_t_nth, int32_t* d_status, cudaStream_t stream) {
  select_first_n_kernel<<<1, 32, 0, stream>>>(d_arrival, d_tags, t, N, W, d_kept, d_t_nth, d_status);
  return cudaGetLastError();
}

}  // namespace psync
