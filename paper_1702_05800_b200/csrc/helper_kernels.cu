// K5 / K6: the two helpers the asynchronous baseline of the paper needs around K4.
//
// K5 -- global-norm clipping (PAPER.md A.3, L313: "gradient clipping is also needed for stabilization, which
// requires each worker to collect the gradient across all layers of the deep model, compute the global norm ||G||
// and then clip all gradient accordingly").  Reading R22: G <- G * clip / max(||G||_2, clip).  Only the FACTOR is
// computed here; K4 applies it while it streams the gradient (it takes the place of the 1/N multiplier), so the
// clipped gradient is never written.  The norm needs one extra pass over the W buffers (W*P*sizeof(grad) bytes, an
// HBM-bound stream) -- the paper's point that clipping serialises the update behind the whole gradient.
// Deterministic: fixed chunking, fixed-order tree reductions, no atomics.
//
// K6 -- gamma_t = gamma_0 * beta^(t s) (A.2 L305, A.3 L315) for K consecutive iterations, for K4's d_gamma table.

#include "psync_device.cuh"

namespace psync {
namespace {

using namespace dev;

constexpr int kClipThreads = 256;
constexpr int kClipUnitsPerThread = 32;                                   // 16-byte units per thread per chunk
constexpr int64_t kClipChunkUnits = int64_t{kClipThreads} * kClipUnitsPerThread;  // 8192 units = 128 KB per CTA

__device__ __forceinline__ double block_sum(double v, double* s_warp) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v += __shfl_down_sync(0xFFFFFFFFu, v, d);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) s_warp[warp] = v;
  __syncthreads();
  double total = 0.0;
  if (threadIdx.x == 0)
    for (int w = 0; w < (blockDim.x + 31) / 32; ++w) total += s_warp[w];  // fixed order
  return total;  // valid in thread 0
}

template <bool BF16>
__device__ __forceinline__ float unit_sumsq(const uint4& r) {
  float s = 0.f;
  if (BF16) {
    const uint32_t w[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float lo = __uint_as_float(w[i] << 16), hi = __uint_as_float(w[i] & 0xFFFF0000u);
      s = __fmaf_rn(lo, lo, s);
      s = __fmaf_rn(hi, hi, s);
    }
  } else {
    const float x = __uint_as_float(r.x), y = __uint_as_float(r.y), z = __uint_as_float(r.z), w = __uint_as_float(r.w);
    s = __fmaf_rn(x, x, s);
    s = __fmaf_rn(y, y, s);
    s = __fmaf_rn(z, z, s);
    s = __fmaf_rn(w, w, s);
  }
  return s;
}

// grid (chunks, W): CTA (c, k) writes the sum of squares of chunk c of worker k's buffer to work[k * chunks + c].
template <bool BF16>
__global__ void __launch_bounds__(kClipThreads) sumsq_chunks_kernel(const void* const* __restrict__ grads, int64_t P,
                                                                    double* __restrict__ work) {
  constexpr int E = BF16 ? 8 : 4;
  __shared__ double s_warp[kClipThreads / 32];
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const char* g = static_cast<const char*>(grads[blockIdx.y]);
  const int64_t n_units = ((reinterpret_cast<uintptr_t>(g) & 15u) == 0) ? P / E : 0;  // misaligned: all scalar
  const int64_t u0 = static_cast<int64_t>(blockIdx.x) * kClipChunkUnits;
  double acc = 0.0;
  constexpr int U = 8;
  for (int b = 0; b < kClipUnitsPerThread; b += U) {
    uint4 r[U];
    bool on[U];
#pragma unroll
    for (int v = 0; v < U; ++v) {
      const int64_t u = u0 + static_cast<int64_t>(b + v) * kClipThreads + threadIdx.x;
      on[v] = u < n_units;
      r[v] = on[v] ? ldg_stream16(g + u * 16) : make_uint4(0u, 0u, 0u, 0u);
    }
#pragma unroll
    for (int v = 0; v < U; ++v)
      if (on[v]) acc += static_cast<double>(unit_sumsq<BF16>(r[v]));  // fp32 inside a 16-byte unit, double across
  }
  // elements the vector path does not cover (tail, or everything if misaligned): chunk 0 takes them
  if (blockIdx.x == 0)
    for (int64_t i = n_units * E + threadIdx.x; i < P; i += kClipThreads) {
      const float x = load_grad_scalar<BF16>(g, i);
      acc += static_cast<double>(x) * static_cast<double>(x);
    }
  const double total = block_sum(acc, s_warp);
  if (threadIdx.x == 0) work[static_cast<int64_t>(blockIdx.y) * gridDim.x + blockIdx.x] = total;
}

// K5s -- the same sums for gradients that lie as per-(worker, server) slices (grads [W*M], entry k*M + j -> G_k[j]).
// grid (n_chunks, W): CTA (c, k) finds its (server j, chunk) in chunk_start (the work-list prefix sum for chunks of
// 8192 16-byte units), sums the squares of that chunk of slice (k, j) and writes work[k * n_chunks + c].  A slice may
// start at any element: the < 16 bytes before its first 16-byte boundary inside the chunk and the tail go element by
// element, everything between as 128-bit loads.
template <bool BF16>
__global__ void __launch_bounds__(kClipThreads) sumsq_slices_kernel(const void* const* __restrict__ grads, int32_t M,
                                                                    const int64_t* shard_off, const int64_t* chunk_start,
                                                                    double* __restrict__ work) {
  constexpr int E = BF16 ? 8 : 4;
  constexpr int ESZ = BF16 ? 2 : 4;
  constexpr int64_t CE = kClipChunkUnits * E;  // elements per chunk
  __shared__ double s_warp[kClipThreads / 32];
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int64_t c = blockIdx.x;
  double acc = 0.0;
  if (chunk_start[M] == static_cast<int64_t>(gridDim.x)) {  // else: a chunk list of another layout -- sums stay 0
    const int j = upper_slot_warp(chunk_start, M, c);
    const int64_t len_j = shard_off[j + 1] - shard_off[j];
    const int64_t lo = (c - chunk_start[j]) * CE;
    const int64_t hi = (len_j - lo < CE) ? len_j : lo + CE;
    const char* g = static_cast<const char*>(grads[static_cast<int64_t>(blockIdx.y) * M + j]);
    const int mis = static_cast<int>((reinterpret_cast<uintptr_t>(g + lo * ESZ) & 15u) / ESZ);
    int64_t head = mis ? (16 / ESZ - mis) : 0;
    if (head > hi - lo) head = hi - lo;
    const int64_t n_units = (hi - lo - head) / E;
    const char* base = g + (lo + head) * ESZ;  // 16-byte aligned
    constexpr int U = 8;
    for (int b = 0; b < kClipUnitsPerThread; b += U) {
      uint4 r[U];
      bool on[U];
#pragma unroll
      for (int v = 0; v < U; ++v) {
        const int64_t u = static_cast<int64_t>(b + v) * kClipThreads + threadIdx.x;
        on[v] = u < n_units;
        r[v] = on[v] ? ldg_stream16(base + u * 16) : make_uint4(0u, 0u, 0u, 0u);
      }
#pragma unroll
      for (int v = 0; v < U; ++v)
        if (on[v]) acc += static_cast<double>(unit_sumsq<BF16>(r[v]));
    }
    const int64_t tail0 = lo + head + n_units * E;
    const int64_t n_peel = head + (hi - tail0);  // < 2 E
    if (threadIdx.x < n_peel) {
      const int64_t i = threadIdx.x < head ? lo + threadIdx.x : tail0 + (threadIdx.x - head);
      const float x = load_grad_scalar<BF16>(g, i);
      acc += static_cast<double>(x) * static_cast<double>(x);
    }
  }
  const double total = block_sum(acc, s_warp);
  if (threadIdx.x == 0) work[static_cast<int64_t>(blockIdx.y) * gridDim.x + blockIdx.x] = total;
}

// one CTA per worker: fixed-order sum of its chunk partials, then the clip factor (`work` comes from the
// predecessor kernel: a plain pointer, see K7b)
__global__ void __launch_bounds__(kClipThreads) clip_finalize_kernel(const double* work, int chunks,
                                                                     float clip, float* __restrict__ scales) {
  __shared__ double s_warp[kClipThreads / 32];
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const double* row = work + static_cast<int64_t>(blockIdx.x) * chunks;
  double acc = 0.0;
  for (int c = threadIdx.x; c < chunks; c += kClipThreads) acc += row[c];
  const double total = block_sum(acc, s_warp);
  if (threadIdx.x == 0) {
    const double c = static_cast<double>(clip);
    scales[blockIdx.x] = static_cast<float>(c / fmax(sqrt(total), c));
  }
}

__global__ void lr_schedule_kernel(float gamma0, float beta, int64_t t0, int32_t K, double s, float* __restrict__ out) {
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < K)
    out[i] = static_cast<float>(static_cast<double>(gamma0) *
                                pow(static_cast<double>(beta), static_cast<double>(t0 + i) * s));
}

// K6c -- the same table when the iteration count t lives on the DEVICE (Alg. 2's t, L84, advances by the number of
// gradients that actually arrived, which only the device knows without a host sync).  One CTA: t0 = t_set >= 0 ? t_set :
// *t_counter + max_r n_add[r]  (rows = 1: the one order's count; rows = M: the largest count of any server -- every
// worker gradient that reached a server is one iteration of the schedule); *t_counter <- t0; out[i] = gamma_{t0 + i}.
__global__ void __launch_bounds__(1024) lr_schedule_counted_kernel(float gamma0, float beta, int64_t* t_counter,
                                                                   int64_t t_set, const int32_t* n_add, int32_t rows,
                                                                   int32_t K, double s, float* out) {
  __shared__ int s_max;
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  if (threadIdx.x == 0) s_max = 0;
  __syncthreads();
  if (t_set < 0 && n_add != nullptr) {
    int m = 0;
    for (int r = threadIdx.x; r < rows; r += blockDim.x) m = max(m, n_add[r]);
    if (m > 0) atomicMax(&s_max, m);
  }
  const int64_t before = *t_counter;
  __syncthreads();  // every thread has read the counter before thread 0 replaces it
  const int64_t t0 = t_set >= 0 ? t_set : before + s_max;
  if (threadIdx.x == 0) *t_counter = t0;
  const int i = threadIdx.x;
  if (i < K)
    out[i] = static_cast<float>(static_cast<double>(gamma0) *
                                pow(static_cast<double>(beta), static_cast<double>(t0 + i) * s));
}

// ---- K7: straggler statistics, the procedure of section 3.1 -----------------------------
__device__ __forceinline__ uint32_t time_key(float a) {  // order-preserving; 0xFFFFFFFF = never arrived
  uint32_t u = __float_as_uint(a);
  if ((u & 0x7F800000u) == 0x7F800000u) return 0xFFFFFFFFu;
  if (u == 0x80000000u) u = 0u;
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float key_time(uint32_t key) {
  return __uint_as_float((key & 0x80000000u) ? (key & 0x7FFFFFFFu) : ~key);
}

// K7a: one CTA per iteration: rank-sort its W arrival times; entry k of the row = when the (k+1)-th gradient arrived
__global__ void __launch_bounds__(1024) sort_rows_kernel(const float* arrival, int32_t W,  // plain: a predecessor may write it
                                                         float* __restrict__ sorted) {
  __shared__ uint32_t s_key[kMaxWorkers];
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int i = threadIdx.x;
  const int64_t row = static_cast<int64_t>(blockIdx.x) * W;
  uint32_t key = 0xFFFFFFFFu;
  if (i < W) {
    key = time_key(arrival[row + i]);
    s_key[i] = key;
  }
  const int n = __syncthreads_count(key != 0xFFFFFFFFu);
  if (i < W && i >= n) sorted[row + i] = __int_as_float(0x7F800000);  // no (i+1)-th arrival this iteration: +inf
  if (key != 0xFFFFFFFFu) {
    int rank = 0;
    for (int j = 0; j < W; ++j) {
      const uint32_t kj = s_key[j];
      rank += (kj < key || (kj == key && j < i)) ? 1 : 0;
    }
    sorted[row + rank] = key_time(key);
  }
}

// (`sorted` and `iters` are written by the predecessor kernel, which may still be running when this grid becomes
// resident under programmatic dependent launch: they are plain pointers, never ld.global.nc / __restrict__.)
// K7b: one CTA per k: count / mean (fixed-order double sum) / median (radix select over the T keys of column k)
__global__ void __launch_bounds__(256) column_stats_kernel(const float* sorted, int32_t T, int32_t W,
                                                           int32_t* __restrict__ count, double* __restrict__ mean,
                                                           double* __restrict__ median, const double* iters,
                                                           double* __restrict__ est_time) {
  __shared__ double s_warp[8];
  __shared__ int s_cnt[4];
  __shared__ int s_n;
  __shared__ double s_sum;
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int k = blockIdx.x;
  double acc = 0.0;
  int mine = 0;
  for (int t = threadIdx.x; t < T; t += 256) {
    const float v = sorted[static_cast<int64_t>(t) * W + k];
    if (time_key(v) != 0xFFFFFFFFu) {
      acc += static_cast<double>(v);
      ++mine;
    }
  }
  const double total = block_sum(acc, s_warp);
  if (threadIdx.x == 0) {
    s_sum = total;
    s_n = 0;
  }
  __syncthreads();
  atomicAdd(&s_n, mine);  // integer: the result does not depend on the order
  __syncthreads();
  const int c = s_n;
  double med = __longlong_as_double(0x7FF8000000000000LL);  // NaN when nobody ever delivered a (k+1)-th gradient
  if (c > 0) {
    double v[2];
    for (int which = 0; which < 2; ++which) {
      int r = which == 0 ? (c - 1) / 2 : c / 2;
      uint32_t prefix = 0u;
      for (int shift = 30; shift >= 0; shift -= 2) {
        const uint32_t hi_mask = (shift == 30) ? 0u : (0xFFFFFFFFu << (shift + 2));
        if (threadIdx.x < 4) s_cnt[threadIdx.x] = 0;
        __syncthreads();
        int c0 = 0, c1 = 0, c2 = 0, c3 = 0;
        for (int t = threadIdx.x; t < T; t += 256) {
          const uint32_t key = time_key(sorted[static_cast<int64_t>(t) * W + k]);
          if (key != 0xFFFFFFFFu && (key & hi_mask) == prefix) {
            const uint32_t d = (key >> shift) & 3u;
            c0 += d == 0u;
            c1 += d == 1u;
            c2 += d == 2u;
            c3 += d == 3u;
          }
        }
        if (c0) atomicAdd(&s_cnt[0], c0);
        if (c1) atomicAdd(&s_cnt[1], c1);
        if (c2) atomicAdd(&s_cnt[2], c2);
        if (c3) atomicAdd(&s_cnt[3], c3);
        __syncthreads();
        const int n0 = s_cnt[0], n1 = s_cnt[1], n2 = s_cnt[2];
        uint32_t digit;
        if (r < n0) digit = 0u;
        else if (r < n0 + n1) { digit = 1u; r -= n0; }
        else if (r < n0 + n1 + n2) { digit = 2u; r -= n0 + n1; }
        else { digit = 3u; r -= n0 + n1 + n2; }
        prefix |= digit << shift;
        __syncthreads();
      }
      v[which] = static_cast<double>(key_time(prefix));
    }
    med = (c & 1) ? v[0] : 0.5 * (v[0] + v[1]);
  }
  if (threadIdx.x == 0) {
    const double m = c > 0 ? s_sum / static_cast<double>(c) : __longlong_as_double(0x7FF8000000000000LL);
    count[k] = c;
    mean[k] = m;
    median[k] = med;
    if (est_time != nullptr) est_time[k] = m * iters[k];
  }
}

// K7c: iterations(N) for N = 1..W by linear interpolation of measured points (Fig. 5 -> Fig. 6);
// the nearest measured value is held outside the measured range.  Explicitly rounded double operations.
__global__ void interp_iterations_kernel(const InterpPoints pts, int32_t W, double* __restrict__ iters) {
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= W) return;
  const int N = k + 1;
  double v;
  if (N <= pts.N[0]) {
    v = pts.iters[0];
  } else if (N >= pts.N[pts.n - 1]) {
    v = pts.iters[pts.n - 1];
  } else {
    int p = 0;
    while (pts.N[p + 1] < N) ++p;
    const double num = __dmul_rn(__dsub_rn(pts.iters[p + 1], pts.iters[p]), static_cast<double>(N - pts.N[p]));
    v = __dadd_rn(pts.iters[p], __ddiv_rn(num, static_cast<double>(pts.N[p + 1] - pts.N[p])));
  }
  iters[k] = v;
}

int clip_chunks(int64_t P, int dtype) {
  const int E = dtype == 1 ? 8 : 4;
  const int64_t c = (P / E + kClipChunkUnits - 1) / kClipChunkUnits;
  return static_cast<int>(c < 1 ? 1 : c);
}

void pdl_config(cudaLaunchConfig_t* cfg, cudaLaunchAttribute* attr, dim3 grid, dim3 block, cudaStream_t stream) {
  *cfg = {};
  cfg->gridDim = grid;
  cfg->blockDim = block;
  cfg->stream = stream;
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg->attrs = attr;
  cfg->numAttrs = 1;
}

// ---- K8: staleness of the gradients Alg. 2 applies (Table 1; fixed lag: section 2.1) -------
// One CTA, thread i owns the i-th applied gradient: staleness_i = (t + lag + i) - read_iter[order[i]]; the worker's next
// read sees t + lag + i + 1.  Validation (a worker twice in one batch, a read from the future) happens before anything
// is written.  Statistics: min / max by reduction, mean = sum / K (integer sum, exact), the population standard
// deviation summed by one thread in index order (the order the oracle uses), the median from a rank sort.
// One CTA per row: row r of every array is parameter server r's own bookkeeping (its counter, what each worker last read
// from IT, the order its gradients reached IT); rows = 1 is the single-order form.
__global__ void __launch_bounds__(1024) staleness_kernel(int64_t* read_iter_rows, int32_t W, const int32_t* order_rows,
                                                         const int32_t* n_arrived_rows, int32_t K_arg,
                                                         int64_t* t_counter_rows, int32_t lag, int64_t* staleness_rows,
                                                         double* stats_rows, int32_t* status_rows) {
  const int64_t row = blockIdx.x;
  int64_t* read_iter = read_iter_rows + row * W;
  const int32_t* order = order_rows + row * W;
  const int32_t* n_arrived = n_arrived_rows ? n_arrived_rows + row : nullptr;
  int64_t* t_counter = t_counter_rows + row;
  int64_t* staleness = staleness_rows + row * W;
  double* stats = stats_rows + row * 6;
  int32_t* status = status_rows + row;
  __shared__ int s_seen[kMaxWorkers];
  __shared__ long long s_val[kMaxWorkers];
  __shared__ long long s_sorted[kMaxWorkers];
  __shared__ int s_bad;
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int i = threadIdx.x;
  const int K = n_arrived ? *n_arrived : K_arg;
  if (i < W) s_seen[i] = 0;
  if (i == 0) s_bad = (K < 0 || K > W) ? 1 : 0;
  __syncthreads();
  const long long t0 = *t_counter;
  int k = -1;
  long long st = 0;
  if (s_bad == 0 && i < K) {
    k = order[i];
    if (k < 0 || k >= W) {
      atomicExch(&s_bad, 1);
    } else {
      if (atomicAdd(&s_seen[k], 1) != 0) atomicExch(&s_bad, 1);  // the same worker twice in one batch
      const long long r = read_iter[k];
      st = t0 + lag + i - r;
      if (r < 0 || st < 0) atomicExch(&s_bad, 1);  // computed from parameters that did not exist yet
    }
  }
  if (t0 < 0 || lag < 0) s_bad = 1;
  __syncthreads();
  if (s_bad != 0) {
    if (i == 0) *status = -1;  // PSYNC_EINVAL; nothing else is written
    return;
  }
  if (i < K) {
    staleness[i] = st;
    read_iter[k] = t0 + lag + i + 1;
    s_val[i] = st;
  }
  __syncthreads();
  if (i < K) {  // rank sort (ties by index)
    int rank = 0;
    for (int j = 0; j < K; ++j) {
      const long long v = s_val[j];
      rank += (v < st || (v == st && j < i)) ? 1 : 0;
    }
    s_sorted[rank] = st;
  }
  __syncthreads();
  if (i == 0) {
    *status = 0;
    *t_counter = t0 + K;
    if (K == 0) {
      const double nan = __longlong_as_double(0x7FF8000000000000LL);
      stats[0] = stats[1] = stats[2] = stats[3] = stats[4] = nan;
      stats[5] = 0.0;
    } else {
      double sum = 0.0;
      for (int j = 0; j < K; ++j) sum = __dadd_rn(sum, static_cast<double>(s_val[j]));
      const double mean = __ddiv_rn(sum, static_cast<double>(K));
      double ss = 0.0;
      for (int j = 0; j < K; ++j) {
        const double d = __dsub_rn(static_cast<double>(s_val[j]), mean);
        ss = __dadd_rn(ss, __dmul_rn(d, d));
      }
      stats[0] = static_cast<double>(s_sorted[0]);
      stats[1] = mean;
      stats[2] = (K & 1) ? static_cast<double>(s_sorted[K / 2])
                         : __dmul_rn(0.5, __dadd_rn(static_cast<double>(s_sorted[K / 2 - 1]), static_cast<double>(s_sorted[K / 2])));
      stats[3] = static_cast<double>(s_sorted[K - 1]);
      stats[4] = __dsqrt_rn(__ddiv_rn(ss, static_cast<double>(K)));
      stats[5] = static_cast<double>(K);
    }
  }
}

}  // namespace

size_t clip_workspace_bytes(int32_t W, int64_t P, int dtype) {
  return sizeof(double) * static_cast<size_t>(W) * static_cast<size_t>(clip_chunks(P, dtype));
}

cudaError_t launch_clip_scales(const void* const* d_grads, int32_t W, int64_t P, int dtype, float clip, float* d_scales,
                               void* d_work, cudaStream_t stream) {
  const int chunks = clip_chunks(P, dtype);
  cudaLaunchConfig_t cfg;
  cudaLaunchAttribute attr[1];
  pdl_config(&cfg, attr, dim3(static_cast<unsigned>(chunks), static_cast<unsigned>(W)), dim3(kClipThreads), stream);
  double* work = static_cast<double*>(d_work);
  cudaError_t err = dtype == 1 ? cudaLaunchKernelEx(&cfg, sumsq_chunks_kernel<true>, d_grads, P, work)
                               : cudaLaunchKernelEx(&cfg, sumsq_chunks_kernel<false>, d_grads, P, work);
  if (err != cudaSuccess) return err;
  pdl_config(&cfg, attr, dim3(static_cast<unsigned>(W)), dim3(kClipThreads), stream);
  return cudaLaunchKernelEx(&cfg, clip_finalize_kernel, static_cast<const double*>(work), chunks, clip, d_scales);
}

int64_t clip_chunk_elems(int dtype) { return kClipChunkUnits * (dtype == 1 ? 8 : 4); }

size_t clip_slices_workspace_bytes(int32_t W, int32_t M, int64_t n_chunks) {
  return sizeof(int64_t) * (static_cast<size_t>(M) + 1) +
         sizeof(double) * static_cast<size_t>(W) * static_cast<size_t>(n_chunks < 1 ? 1 : n_chunks);
}

cudaError_t launch_clip_scales_slices(const void* const* d_grads, int32_t W, int32_t M, const int64_t* d_shard_off,
                                      int64_t n_chunks, int dtype, float clip, float* d_scales, void* d_work,
                                      cudaStream_t stream) {
  if (n_chunks > 0x7FFFFFFF) return cudaErrorInvalidConfiguration;
  int64_t* chunk_start = static_cast<int64_t*>(d_work);
  double* work = reinterpret_cast<double*>(chunk_start + M + 1);
  cudaError_t err = launch_shard_worklist_elems(d_shard_off, M, static_cast<int32_t>(clip_chunk_elems(dtype)), chunk_start,
                                                stream);
  if (err != cudaSuccess) return err;
  cudaLaunchConfig_t cfg;
  cudaLaunchAttribute attr[1];
  const int chunks = static_cast<int>(n_chunks);
  if (chunks > 0) {
    pdl_config(&cfg, attr, dim3(static_cast<unsigned>(chunks), static_cast<unsigned>(W)), dim3(kClipThreads), stream);
    err = dtype == 1 ? cudaLaunchKernelEx(&cfg, sumsq_slices_kernel<true>, d_grads, M, d_shard_off,
                                          static_cast<const int64_t*>(chunk_start), work)
                     : cudaLaunchKernelEx(&cfg, sumsq_slices_kernel<false>, d_grads, M, d_shard_off,
                                          static_cast<const int64_t*>(chunk_start), work);
    if (err != cudaSuccess) return err;
  }
  pdl_config(&cfg, attr, dim3(static_cast<unsigned>(W)), dim3(kClipThreads), stream);
  return cudaLaunchKernelEx(&cfg, clip_finalize_kernel, static_cast<const double*>(work), chunks, clip, d_scales);
}

cudaError_t launch_kth_arrival_stats(const float* d_arrival, int32_t T, int32_t W, float* d_sorted, int32_t* d_count,
                                     double* d_mean, double* d_median, const double* d_iters, double* d_est_time,
                                     cudaStream_t stream) {
  cudaLaunchConfig_t cfg;
  cudaLaunchAttribute attr[1];
  pdl_config(&cfg, attr, dim3(static_cast<unsigned>(T)), dim3(static_cast<unsigned>((W + 31) / 32 * 32)), stream);
  cudaError_t err = cudaLaunchKernelEx(&cfg, sort_rows_kernel, d_arrival, W, d_sorted);
  if (err != cudaSuccess) return err;
  pdl_config(&cfg, attr, dim3(static_cast<unsigned>(W)), dim3(256), stream);
  return cudaLaunchKernelEx(&cfg, column_stats_kernel, static_cast<const float*>(d_sorted), T, W, d_count, d_mean,
                            d_median, d_iters, d_est_time);
}

cudaError_t launch_interp_iterations(const InterpPoints& pts, int32_t W, double* d_iters, cudaStream_t stream) {
  cudaLaunchConfig_t cfg;
  cudaLaunchAttribute attr[1];
  pdl_config(&cfg, attr, dim3(static_cast<unsigned>((W + 127) / 128)), dim3(128), stream);
  return cudaLaunchKernelEx(&cfg, interp_iterations_kernel, pts, W, d_iters);
}

cudaError_t launch_lr_schedule(float gamma0, float beta, int64_t t0, int32_t K, double s, float* d_gamma,
                               cudaStream_t stream) {
  cudaLaunchConfig_t cfg;
  cudaLaunchAttribute attr[1];
  pdl_config(&cfg, attr, dim3(static_cast<unsigned>((K + 127) / 128)), dim3(128), stream);
  return cudaLaunchKernelEx(&cfg, lr_schedule_kernel, gamma0, beta, t0, K, s, d_gamma);
}

cudaError_t launch_lr_schedule_counted(float gamma0, float beta, int64_t* d_t, int64_t t_set, const int32_t* d_n_add,
                                       int32_t rows, int32_t K, double s, float* d_gamma, cudaStream_t stream) {
  cudaLaunchConfig_t cfg;
  cudaLaunchAttribute attr[1];
  pdl_config(&cfg, attr, dim3(1), dim3(1024), stream);
  return cudaLaunchKernelEx(&cfg, lr_schedule_counted_kernel, gamma0, beta, d_t, t_set, d_n_add, rows, K, s, d_gamma);
}

cudaError_t launch_staleness(int64_t* d_read_iter, int32_t W, int32_t rows, const int32_t* d_order,
                             const int32_t* d_n_arrived, int32_t K, int64_t* d_t, int32_t lag, int64_t* d_staleness,
                             double* d_stats, int32_t* d_status, cudaStream_t stream) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(static_cast<unsigned>(rows));
  cfg.blockDim = dim3(static_cast<unsigned>((W + 31) / 32 * 32));
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, staleness_kernel, d_read_iter, W, d_order, d_n_arrived, K, d_t, lag, d_staleness,
                            d_stats, d_status);
}

}  // namespace psync

// ---- K5n: psync_clip_scales_static -- K5 for callers that must not allocate device memory ----------------------------
// Some users of this library are not allowed to call cudaMalloc where the clip factors are needed: code that runs
// inside a framework's allocator-owned region (every byte of the device already handed to a caching pool, so a raw
// cudaMalloc fails or fragments it), a plugin that is given buffers and a stream and nothing else, or a latency-critical
// loop in which cudaMalloc's implicit device synchronisation is unacceptable.  K5 needs scratch memory for its per-chunk
// partial sums (double [W][chunks]); the ordinary entry point makes the caller bring it (d_work).  This variant keeps that
// scratch inside the library image instead: one fixed array in device global memory, reserved on every GPU that loads
// libpsync.so from the moment the module is loaded until the process exits (kClipStaticBytes = 2 MiB per GPU).
//
// What follows from that, and what the header repeats for the caller:
//  * the problem must fit: W * chunks <= kClipStaticPartials (chunks = ceil(P*sizeof(grad) / 128 KiB), at least 1);
//    larger requests are refused (PSYNC_EUNSUPPORTED), never truncated;
//  * every call on a device uses the SAME array.  Two calls whose kernels can be on the GPU at the same time (different
//    streams, or different host threads on different streams) overwrite each other's partial sums.  Calls on one stream
//    are ordered by the stream and are safe;
//  * the array keeps whatever the previous call left in it.  Nothing has to be cleared: sumsq_chunks_kernel stores
//    (does not accumulate into) every one of the W * chunks slots that clip_finalize_kernel reads, in every call;
//  * inside host code the name g_clip_static_scratch is only a handle for the runtime, not a device address.  The
//    address a kernel can use is looked up once per device with cudaGetSymbolAddress while that device is current and
//    remembered; that look-up (which may also load the module onto the device) happens in the first call made on each
//    device, so make that first call outside any stream capture.
namespace psync {
namespace {

constexpr size_t kClipStaticBytes = size_t{2} << 20;                      // == PSYNC_CLIP_STATIC_SCRATCH_BYTES
constexpr size_t kClipStaticPartials = kClipStaticBytes / sizeof(double);  // 262,144 partial sums
static __device__ __align__(256) double g_clip_static_scratch[kClipStaticPartials];

constexpr int kClipStaticMaxDevices = 64;
double* g_clip_static_addr[kClipStaticMaxDevices] = {};  // device address of the array on device i, once looked up

// Device address of the scratch array on the CURRENT device (nullptr + *err on failure).  Host threads may race here:
// they all obtain the same address for the same device, and an aligned pointer store is atomic on the hosts CUDA runs on.
double* clip_static_scratch(cudaError_t* err) {
  int dev = -1;
  *err = cudaGetDevice(&dev);
  if (*err != cudaSuccess) return nullptr;
  const bool cached = dev >= 0 && dev < kClipStaticMaxDevices;
  if (cached) {
    double* p = __atomic_load_n(&g_clip_static_addr[dev], __ATOMIC_ACQUIRE);
    if (p != nullptr) return p;
  }
  double* p = nullptr;
  *err = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_clip_static_scratch);
  if (*err != cudaSuccess || p == nullptr) {
    if (*err == cudaSuccess) *err = cudaErrorInvalidSymbol;
    return nullptr;
  }
  if (cached) __atomic_store_n(&g_clip_static_addr[dev], p, __ATOMIC_RELEASE);
  return p;
}

}  // namespace
}  // namespace psync

#include "../../include/psync.h"

static_assert(PSYNC_CLIP_STATIC_SCRATCH_BYTES == psync::kClipStaticBytes, "psync.h and the scratch array disagree");

// The C entry point lives in this file because the scratch array has file scope (see psync.h for the contract).
// It calls no cudaMalloc / cudaFree and nothing that allocates: one cudaGetDevice, on the first call per device one
// cudaGetSymbolAddress, then the two launches of K5.
extern "C" PSYNC_API int psync_clip_scales_static(const void* const* d_grads, int32_t W, int64_t P, int32_t grad_dtype,
                                                  float clip, float* d_scales, void* stream) {
  if (d_grads == nullptr || d_scales == nullptr) return PSYNC_EINVAL;
  if (W < 1 || W > PSYNC_MAX_WORKERS || P < 0 || !(clip > 0.0f)) return PSYNC_EINVAL;
  if (grad_dtype != PSYNC_F32 && grad_dtype != PSYNC_BF16) return PSYNC_EINVAL;
  if (psync::clip_workspace_bytes(W, P, grad_dtype) > psync::kClipStaticBytes) return PSYNC_EUNSUPPORTED;  // does not fit
  cudaError_t err = cudaSuccess;
  double* scratch = psync::clip_static_scratch(&err);
  if (scratch == nullptr) return PSYNC_ECUDA;
  return psync::launch_clip_scales(d_grads, W, P, grad_dtype, clip, d_scales, scratch, static_cast<cudaStream_t>(stream)) ==
                 cudaSuccess
             ? PSYNC_OK
             : PSYNC_ECUDA;
}
