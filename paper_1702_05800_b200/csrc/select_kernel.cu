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
//   2. the N-th smallest key tau is found by a 16-pass MSB-first radix select, two bits per pass
//      (per pass: count the still-matching keys per digit value, warp-reduce);
//   3. worker k is kept iff key_k < tau, or key_k == tau and k is among the first
//      (N - #{key < tau}) such workers in index order (ties go to the lower index, reading R1).
// Lanes own CONTIGUOUS index ranges, so a warp exclusive scan of the per-lane kept counts
// gives every lane its output offset and the list comes out in ascending worker order.
// The keys stay in registers (C per lane, templated), the select takes two bits per pass.

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

// Programmatic dependent launch (PDL): launched with programmatic stream serialization, this kernel
// may become resident while its predecessor in the stream (typically the previous step's fused
// kernel) drains, which hides its launch latency.  It touches no memory before griddepcontrol.wait
// (which returns once the predecessor has completed and its writes are visible), so ordinary stream
// semantics are preserved for any predecessor.  It releases its successor (the fused kernel, which
// waits the same way before reading kept[]) immediately.
__device__ __forceinline__ void pdl_wait_for_predecessor() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_release_successor() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// C = keys per lane (W <= 32*C); the keys live in registers, every loop is unrolled.
template <int C>
__global__ void __launch_bounds__(32) select_first_n_kernel(const float* arrival,  // plain pointers: a predecessor
                                                            const int32_t* tags,   // under PDL typically writes these
                                                            int32_t t, int32_t N,
                                                            int32_t W, int32_t* __restrict__ kept,
                                                            float* __restrict__ t_nth, int32_t* __restrict__ status) {
  const int lane = threadIdx.x;
  const int base = lane * C;  // lane owns workers [base, base + C): ascending order falls out of the scan
  pdl_release_successor();    // the fused kernel behind us may get resident; it waits before reading kept[]
  pdl_wait_for_predecessor();

  // one CTA (one warp) per row: row j = parameter server j's own arrival times (Alg. 4 per server, L134)
  const int64_t row = blockIdx.x;
  arrival += row * W;
  if (tags != nullptr) tags += row * W;
  kept += row * N;
  if (t_nth != nullptr) t_nth += row;
  status += row;

  uint32_t key[C];
  int n_elig = 0;
#pragma unroll
  for (int i = 0; i < C; ++i) {
    const int k = base + i;
    uint32_t v = kIneligible;
    if (k < W) {
      v = arrival_key(arrival[k]);
      if (tags != nullptr && tags[k] != t) v = kIneligible;  // Alg. 4 l.5-6: t' != t -> dropped
    }
    key[i] = v;
    n_elig += (v != kIneligible);
  }
  n_elig = __reduce_add_sync(0xFFFFFFFFu, n_elig);
  if (n_elig < N) {  // |G| can never reach N this step
    if (lane == 0) *status = kStatusTooFew;
    return;
  }

  // radix select, two bits per pass: tau = key of rank N-1 (0-based); ineligible keys sort last
  uint32_t prefix = 0u;
  int r = N - 1;
#pragma unroll 1
  for (int shift = 30; shift >= 0; shift -= 2) {
    const uint32_t hi_mask = (shift == 30) ? 0u : (0xFFFFFFFFu << (shift + 2));
    uint32_t c01 = 0u, c2 = 0u;  // counts of digit 0 (low half) and 1 (high half), and of digit 2
#pragma unroll
    for (int i = 0; i < C; ++i) {
      const bool match = (key[i] & hi_mask) == prefix;
      const uint32_t d = (key[i] >> shift) & 3u;
      c01 += (match && d == 0u) ? 1u : 0u;
      c01 += (match && d == 1u) ? 0x10000u : 0u;
      c2 += (match && d == 2u) ? 1u : 0u;
    }
    c01 = __reduce_add_sync(0xFFFFFFFFu, c01);
    c2 = __reduce_add_sync(0xFFFFFFFFu, c2);
    const int n0 = static_cast<int>(c01 & 0xFFFFu), n1 = static_cast<int>(c01 >> 16), n2 = static_cast<int>(c2);
    uint32_t digit;
    if (r < n0) {
      digit = 0u;
    } else if (r < n0 + n1) {
      digit = 1u;
      r -= n0;
    } else if (r < n0 + n1 + n2) {
      digit = 2u;
      r -= n0 + n1;
    } else {
      digit = 3u;
      r -= n0 + n1 + n2;
    }
    prefix |= digit << shift;
  }
  const uint32_t tau = prefix;
  const int eq_take = r + 1;  // how many of the workers tied at tau are kept, lowest indices first

  int n_less = 0, n_eq = 0;
#pragma unroll
  for (int i = 0; i < C; ++i) {
    n_less += (key[i] < tau);
    n_eq += (key[i] == tau);
  }
  int total_eq, total_kept;
  const int eq_before = warp_exclusive_scan(n_eq, lane, &total_eq);
  int my_eq = eq_take - eq_before;
  my_eq = my_eq < 0 ? 0 : (my_eq > n_eq ? n_eq : my_eq);
  int out = warp_exclusive_scan(n_less + my_eq, lane, &total_kept);  // total_kept == N

#pragma unroll
  for (int i = 0; i < C; ++i) {  // ascending worker index within the lane's range
    bool keep = key[i] < tau;
    if (key[i] == tau && my_eq > 0) {
      keep = true;
      --my_eq;
    }
    if (keep) kept[out++] = base + i;
  }
  if (lane == 0) {
    *status = kStatusOk;
    if (t_nth != nullptr) *t_nth = key_to_time(tau);
  }
}

// K1b: the time-out rule (reading R19).  Worker k is kept iff it is eligible
// (finite arrival, tag == t) and arrival[k] <= timeout; kept[] comes out ascending because lanes own
// contiguous index ranges; fewer than min_keep -> ETOOFEW, n_kept[row] = 0 and the kept row is not written.
__global__ void __launch_bounds__(32) select_timeout_kernel(const float* arrival,  // plain pointers (as above)
                                                            const int32_t* tags, int32_t t, int32_t W,
                                                            float timeout, int32_t min_keep,
                                                            int32_t* __restrict__ kept, int32_t* __restrict__ n_kept,
                                                            int32_t* __restrict__ status) {
  const int lane = threadIdx.x;
  pdl_release_successor();
  pdl_wait_for_predecessor();
  const int64_t row = blockIdx.x;
  arrival += row * W;
  if (tags != nullptr) tags += row * W;
  kept += row * W;
  const int C = (W + 31) / 32;  // workers per lane
  const int base = lane * C;
  int mine = 0;
  for (int i = 0; i < C; ++i) {
    const int k = base + i;
    if (k < W) {
      const float a = arrival[k];
      const bool finite = (__float_as_uint(a) & 0x7F800000u) != 0x7F800000u;
      mine += (finite && a <= timeout && (tags == nullptr || tags[k] == t)) ? 1 : 0;
    }
  }
  int total;
  int out = warp_exclusive_scan(mine, lane, &total);
  if (total < min_keep) {
    if (lane == 0) {
      status[row] = kStatusTooFew;
      n_kept[row] = 0;  // a consumer that ignores the status must still see an empty row, never a stale count
    }
    return;
  }
  for (int i = 0; i < C; ++i) {
    const int k = base + i;
    if (k < W) {
      const float a = arrival[k];
      const bool finite = (__float_as_uint(a) & 0x7F800000u) != 0x7F800000u;
      if (finite && a <= timeout && (tags == nullptr || tags[k] == t)) kept[out++] = k;
    }
  }
  if (lane == 0) {
    n_kept[row] = total;
    status[row] = kStatusOk;
  }
}

}  // namespace

namespace {
cudaLaunchConfig_t one_warp_per_row(int32_t rows, cudaStream_t stream, cudaLaunchAttribute* attr) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(static_cast<unsigned>(rows));
  cfg.blockDim = dim3(32);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = stream;
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cfg;
}
}  // namespace

cudaError_t launch_select_first_n(const float* d_arrival, const int32_t* d_tags, int32_t t, int32_t N, int32_t W,
                                  int32_t rows, int32_t* d_kept, float* d_t_nth, int32_t* d_status,
                                  cudaStream_t stream) {
  using Kernel = void (*)(const float*, const int32_t*, int32_t, int32_t, int32_t, int32_t*, float*, int32_t*);
  Kernel kernel = select_first_n_kernel<32>;
  if (W <= 32) kernel = select_first_n_kernel<1>;
  else if (W <= 64) kernel = select_first_n_kernel<2>;
  else if (W <= 128) kernel = select_first_n_kernel<4>;
  else if (W <= 256) kernel = select_first_n_kernel<8>;
  else if (W <= 512) kernel = select_first_n_kernel<16>;
  cudaLaunchAttribute attr[1];
  const cudaLaunchConfig_t cfg = one_warp_per_row(rows, stream, attr);
  return cudaLaunchKernelEx(&cfg, kernel, d_arrival, d_tags, t, N, W, d_kept, d_t_nth, d_status);
}

cudaError_t launch_select_timeout(const float* d_arrival, const int32_t* d_tags, int32_t t, int32_t W, int32_t rows,
                                  float timeout, int32_t min_keep, int32_t* d_kept, int32_t* d_n_kept,
                                  int32_t* d_status, cudaStream_t stream) {
  cudaLaunchAttribute attr[1];
  const cudaLaunchConfig_t cfg = one_warp_per_row(rows, stream, attr);
  return cudaLaunchKernelEx(&cfg, select_timeout_kernel, d_arrival, d_tags, t, W, timeout, min_keep, d_kept,
                            d_n_kept, d_status);
}

}  // namespace psync
