// K2: fused aggregate + update + EMA -- Alg. 4 l.8-9 in ONE pass over HBM.
// K3: standalone EMA.
//
//   S[i]   = sum over the kept workers k, ascending k, of G_k[i]          (fp32, fixed order)
//   G[i]   = S[i] * (1/N)
//   theta, state <- optimizer(theta, state, G)      (SGD | momentum | RMSProp with momentum)
//   ema    <- alpha ema + (1 - alpha) theta*        (theta* = new theta, or old theta for PRE)
//
// The path is a pure stream: N*sizeof(grad) + 8*(2 + n_state) bytes per parameter, ~0.25 flop/B,
// so the HBM roofline bounds it and no tensor core is involved (there is no contraction).
// B200 design:
//   * only the N kept buffers are dereferenced, through a device pointer table indexed by the
//     selection kernel's kept[] -- no host sync between K1 and K2, dropped buffers never touched;
//   * 128-bit read-only streaming loads (ld.global.nc, L1 no-allocate), U independent loads in
//     flight per thread per batch, accumulated strictly in worker order afterwards, so the result
//     does not depend on the launch geometry;
//   * one tile per CTA (grid = number of tiles, no tile loop): the hardware CTA scheduler balances the
//     tiles over the SMs dynamically;
//   * theta / state / ema are loaded after the gradient stream (its registers are dead by then),
//     updated in registers and stored once.
// The flat element space is processed without regard to shard cuts: the step is elementwise and
// all arrays share one layout, so server j's slice gets exactly Alg. 4's result (DESIGN.md s.4).

#include "psync_device.cuh"

namespace psync {
namespace {

using namespace dev;

// ---- per-server rows (Alg. 4 per parameter server j): which server owns element i ----------------
// Smallest j with off[j+1] > i, i.e. off[j] <= i < off[j+1] (empty servers are skipped).  The table is
// tiny and read by every CTA, so these loads hit L1/L2; all threads of a CTA search the same i.
__device__ __forceinline__ int find_server(const int64_t* __restrict__ off, int M, int64_t i) {
  int lo = 0, hi = M - 1;
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(off + mid + 1) > i) hi = mid; else lo = mid + 1;
  }
  return lo;
}

// Elements [i0, i1) one at a time, each with its own server's kept row read from global memory: the slow,
// always-correct path for tiles that straddle a server boundary, misaligned buffers and the tail.
template <bool BF16, int OPT, int EMA>
__device__ void rows_scalar_range(const FusedParams& p, int64_t i0, int64_t i1, int64_t tid, int64_t threads) {
  for (int64_t i = i0 + tid; i < i1; i += threads) {
    const int row = p.per_shard ? find_server(p.shard_off, p.M, i) : 0;
    if (p.status != nullptr && p.status[row] != 0) continue;  // this server did not collect its gradients
    const int N = p.n_kept ? p.n_kept[row] : p.N;
    const float inv_N = p.n_kept ? 1.0f / static_cast<float>(N) : p.inv_N;
    const int32_t* kept = p.kept + static_cast<int64_t>(row) * p.kept_stride;
    float S = 0.f;
    for (int n = 0; n < N; ++n) S += load_grad_scalar<BF16>(static_cast<const char*>(p.grads[kept[n]]), i);
    update_in_memory<OPT, EMA>(p, S, inv_N, i);
  }
}

// ---- the fused kernel ------------------------------------------------------------------------
// A "unit" is 16 bytes of one gradient buffer: E = 4 (fp32) or 8 (bf16) consecutive parameters.
// A tile is THREADS x UPT units; slot j of thread tid is unit tile*THREADS*UPT + j*THREADS + tid, so
// each warp-level load covers 512 contiguous bytes of one worker's buffer.
//
// One tile through the 128-bit path: sum the N buffers of s_ptr[] in ascending order, update, store.
// CONSTN: N and 1/N come straight from the kernel parameters (constant bank) instead of registers.
template <int THREADS, int UPT, int U, bool BF16, int OPT, int EMA, bool CONSTN>
__device__ __forceinline__ void vector_tile(const FusedParams& p, const char* const* s_ptr, const int N_arg,
                                            const float inv_N_arg, const int64_t tile, const int64_t n_units) {
  const int N = CONSTN ? p.N : N_arg;
  const float inv_N = CONSTN ? p.inv_N : inv_N_arg;
  constexpr int E = BF16 ? 8 : 4;
  constexpr int Q = E / 4;  // float4 groups of theta per unit
  constexpr int64_t TILE_UNITS = static_cast<int64_t>(THREADS) * UPT;
  int64_t unit[UPT];
  bool live[UPT];
#pragma unroll
  for (int j = 0; j < UPT; ++j) {
    const int64_t u = tile * TILE_UNITS + static_cast<int64_t>(j) * THREADS + threadIdx.x;
    live[j] = u < n_units;
    unit[j] = live[j] ? u : (n_units - 1);  // dead slots re-read a valid unit and store nothing
  }

  float acc[UPT][E];
#pragma unroll
  for (int j = 0; j < UPT; ++j)
#pragma unroll
    for (int e = 0; e < E; ++e) acc[j][e] = 0.f;

  int n = 0;
  for (; n + U <= N; n += U) {  // full batches: U x UPT independent 16-byte loads in flight
    uint4 r[U][UPT];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const char* g = s_ptr[n + u];
#pragma unroll
      for (int j = 0; j < UPT; ++j) r[u][j] = ldg_stream16(g + unit[j] * 16);
    }
#pragma unroll
    for (int u = 0; u < U; ++u)  // strictly ascending worker order per element
#pragma unroll
      for (int j = 0; j < UPT; ++j) accumulate_unit<BF16>(acc[j], r[u][j]);
  }
  if (n < N) {  // last, partial batch: same shape, predicated
    uint4 r[U][UPT];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const bool on = (n + u) < N;
      const char* g = s_ptr[on ? (n + u) : (N - 1)];
#pragma unroll
      for (int j = 0; j < UPT; ++j) r[u][j] = on ? ldg_stream16(g + unit[j] * 16) : make_uint4(0u, 0u, 0u, 0u);
    }
#pragma unroll
    for (int u = 0; u < U; ++u)
      if ((n + u) < N) {
#pragma unroll
        for (int j = 0; j < UPT; ++j) accumulate_unit<BF16>(acc[j], r[u][j]);
      }
  }

  // theta / state / ema: loaded once the gradient registers are dead; other resident warps hide the latency
  float4 th[UPT][Q], em[UPT][Q], a0[UPT][Q], a1[UPT][Q];
#pragma unroll
  for (int j = 0; j < UPT; ++j) {
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      const int64_t e = unit[j] * E + 4 * q;
      th[j][q] = ld_state16(p.theta + e);
      if (EMA != EMA_OFF) em[j][q] = ld_state16(p.ema + e);
      if (OPT != OPT_SGD) a0[j][q] = ld_state16(p.s0 + e);
      if (OPT == OPT_RMSPROP_MOM) a1[j][q] = ld_state16(p.s1 + e);
    }
  }

#pragma unroll
  for (int j = 0; j < UPT; ++j) {
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      float* t4 = reinterpret_cast<float*>(&th[j][q]);
      float* e4 = reinterpret_cast<float*>(&em[j][q]);
      float* x4 = reinterpret_cast<float*>(&a0[j][q]);
      float* y4 = reinterpret_cast<float*>(&a1[j][q]);
#pragma unroll
      for (int l = 0; l < 4; ++l) update_element<OPT, EMA>(acc[j][4 * q + l], inv_N, t4[l], e4[l], x4[l], y4[l], p);
      if (live[j]) {
        const int64_t e = unit[j] * E + 4 * q;
        st_state16(p.theta + e, th[j][q]);
        if (EMA != EMA_OFF) st_state16(p.ema + e, em[j][q]);
        if (OPT != OPT_SGD) st_state16(p.s0 + e, a0[j][q]);
        if (OPT == OPT_RMSPROP_MOM) st_state16(p.s1 + e, a1[j][q]);
      }
    }
  }
}

// Stage kept row `row` as a table of N base pointers in shared memory; returns the OR of their low bits.
template <int THREADS>
__device__ __forceinline__ unsigned stage_row(const FusedParams& p, const char** s_ptr, int row, int N) {
  const int32_t* kept = p.kept + static_cast<int64_t>(row) * p.kept_stride;
  unsigned misalign = 0;
  for (int n = threadIdx.x; n < N; n += THREADS) {
    const char* g = static_cast<const char*>(p.grads[kept[n]]);
    s_ptr[n] = g;
    misalign |= static_cast<unsigned>(reinterpret_cast<uintptr_t>(g)) & 15u;
  }
  return misalign;
}

// ROWS = false: one kept row of exactly N workers for the whole parameter vector (reading R11).
// ROWS = true : kept rows indexed on the device -- a device-side count (time-out rule, L259) and/or
//               one kept row per parameter server j (Alg. 4 literally per server, L134-164): a tile that
//               lies inside one server's slice stages that server's row and takes the same 128-bit path;
//               the at most M-1 tiles that straddle a boundary go element by element.
template <int THREADS, int UPT, int U, int MINB, bool BF16, int OPT, int EMA, bool ROWS>
__global__ void __launch_bounds__(THREADS, MINB) fused_aggregate_update_ema(const FusedParams p) {
  constexpr int E = BF16 ? 8 : 4;
  constexpr int64_t TILE_UNITS = static_cast<int64_t>(THREADS) * UPT;
  __shared__ const char* s_ptr[kMaxWorkers];

  // Programmatic dependent launch: this CTA may be resident before the selection kernel (or the previous
  // fused launch) has finished; nothing is read before the wait.  The successor is released at once --
  // it, too, waits for this whole grid before touching memory.
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  const int64_t n_units = p.P / E;
  const int64_t n_tiles = (n_units + TILE_UNITS - 1) / TILE_UNITS;
  const int64_t tail0 = n_units * E;  // fewer than E trailing parameters

  if (!ROWS) {
    if (p.status != nullptr && *p.status != 0) return;  // selection failed: leave everything untouched
    const unsigned misalign = stage_row<THREADS>(p, s_ptr, 0, p.N);  // a variable count takes the ROWS kernel
    const bool vec_ok = (__syncthreads_or(static_cast<int>(misalign)) == 0) && (p.base_aligned != 0);
    if (!vec_ok) {
      scalar_range<BF16, OPT, EMA>(p, s_ptr, 0, p.P, static_cast<int64_t>(blockIdx.x) * THREADS + threadIdx.x,
                                   static_cast<int64_t>(gridDim.x) * THREADS);
      return;
    }
    if (blockIdx.x < n_tiles)  // one tile per CTA, no tile loop: its loop-carried registers cost a spill at 64
      vector_tile<THREADS, UPT, U, BF16, OPT, EMA, true>(p, s_ptr, 0, 0.f, blockIdx.x, n_units);
    if (tail0 < p.P && blockIdx.x == 0) scalar_range<BF16, OPT, EMA>(p, s_ptr, tail0, p.P, threadIdx.x, THREADS);
  } else {
    const int64_t tile = blockIdx.x;
    if (tile < n_tiles) {
      const int64_t e0 = tile * TILE_UNITS * E;
      const int64_t e1 = (e0 + TILE_UNITS * E < tail0) ? e0 + TILE_UNITS * E : tail0;  // tile = elements [e0, e1)
      // per_shard == 0 here means one row with a device-side count (time-out rule, L259): no lookup
      const int row = p.per_shard ? find_server(p.shard_off, p.M, e0) : 0;
      const bool one_server = p.per_shard ? (__ldg(p.shard_off + row + 1) >= e1) : true;  // CTA-uniform
      const bool failed = one_server && p.status != nullptr && p.status[row] != 0;  // that server's tile is skipped
      if (!failed) {
        bool fast = one_server && p.base_aligned != 0;
        int N = 0;
        float inv_N = 0.f;
        if (fast) {
          N = p.n_kept ? p.n_kept[row] : p.N;
          inv_N = p.n_kept ? 1.0f / static_cast<float>(N) : p.inv_N;
          const unsigned misalign = stage_row<THREADS>(p, s_ptr, row, N);
          fast = __syncthreads_or(static_cast<int>(misalign)) == 0;
        }
        if (fast)
          vector_tile<THREADS, UPT, U, BF16, OPT, EMA, false>(p, s_ptr, N, inv_N, tile, n_units);
        else
          rows_scalar_range<BF16, OPT, EMA>(p, e0, e1, threadIdx.x, THREADS);
      }
    }
    if (tail0 < p.P && blockIdx.x == 0) rows_scalar_range<BF16, OPT, EMA>(p, tail0, p.P, threadIdx.x, THREADS);
  }
}

// ---- K3 ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) ema_kernel(float* __restrict__ ema, const float* __restrict__ theta, int64_t P,
                                                  float alpha, float one_minus_alpha, int aligned) {
  const int64_t gtid = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  const int64_t gthreads = static_cast<int64_t>(gridDim.x) * blockDim.x;
  const int64_t n4 = aligned ? P / 4 : 0;
  for (int64_t v = gtid; v < n4; v += gthreads) {
    float4 e = ld_state16(ema + 4 * v);
    const float4 t = ld_state16(theta + 4 * v);
    e.x = __fmaf_rn(alpha, e.x, __fmul_rn(one_minus_alpha, t.x));
    e.y = __fmaf_rn(alpha, e.y, __fmul_rn(one_minus_alpha, t.y));
    e.z = __fmaf_rn(alpha, e.z, __fmul_rn(one_minus_alpha, t.z));
    e.w = __fmaf_rn(alpha, e.w, __fmul_rn(one_minus_alpha, t.w));
    st_state16(ema + 4 * v, e);
  }
  for (int64_t i = n4 * 4 + gtid; i < P; i += gthreads) ema[i] = __fmaf_rn(alpha, ema[i], __fmul_rn(one_minus_alpha, theta[i]));  // same form as the fused kernel
}

// ---- variants and dispatch ---------------------------------------------------------------------
struct Variant {
  int threads, upt, unroll, minb;
};
// variant ids are 1-based in the ABI (0 = default for the dtype)
constexpr Variant kVariants[] = {
    {256, 1, 8, 4},   // 1
    {256, 2, 8, 2},   // 2
    {256, 1, 16, 3},  // 3
    {512, 1, 8, 2},   // 4
};
constexpr int kNumVariants = sizeof(kVariants) / sizeof(kVariants[0]);

using KernelFn = void (*)(const FusedParams);

// bf16 gradients with RMSProp hold 8 parameters x (acc, theta, ema, ms, mom) = 40 live values per thread:
// at 4 CTAs/SM (64 registers) that spills, so this one combination runs at 3 CTAs/SM (85 registers).
constexpr int minb_for(int v, bool bf16, int opt) {
  const int cap = 768 / kVariants[v].threads;  // resident threads per SM that leave 85 registers each
  return (bf16 && opt == OPT_RMSPROP_MOM && kVariants[v].minb > cap) ? cap : kVariants[v].minb;
}

template <int V, bool BF16, int OPT, int EMA, bool ROWS = false>
constexpr KernelFn kernel_for() {
  return fused_aggregate_update_ema<kVariants[V].threads, kVariants[V].upt, kVariants[V].unroll,
                                    minb_for(V, BF16, OPT), BF16, OPT, EMA, ROWS>;
}

// per-server rows: the default variant only (a forced variant > 1 is PSYNC_EUNSUPPORTED in the ABI)
template <bool BF16, int OPT>
KernelFn pick_rows_ema(int ema) {
  switch (ema) {
    case EMA_POST: return kernel_for<0, BF16, OPT, EMA_POST, true>();
    case EMA_PRE: return kernel_for<0, BF16, OPT, EMA_PRE, true>();
    default: return kernel_for<0, BF16, OPT, EMA_OFF, true>();
  }
}
template <bool BF16>
KernelFn pick_rows_opt(int opt, int ema) {
  switch (opt) {
    case OPT_SGD: return pick_rows_ema<BF16, OPT_SGD>(ema);
    case OPT_MOMENTUM: return pick_rows_ema<BF16, OPT_MOMENTUM>(ema);
    default: return pick_rows_ema<BF16, OPT_RMSPROP_MOM>(ema);
  }
}
KernelFn pick_rows_kernel(int dtype, int opt, int ema) {
  return dtype == 1 ? pick_rows_opt<true>(opt, ema) : pick_rows_opt<false>(opt, ema);
}

template <int V, bool BF16, int OPT>
KernelFn pick_ema(int ema) {
  switch (ema) {
    case EMA_POST: return kernel_for<V, BF16, OPT, EMA_POST>();
    case EMA_PRE: return kernel_for<V, BF16, OPT, EMA_PRE>();
    default: return kernel_for<V, BF16, OPT, EMA_OFF>();
  }
}
template <int V, bool BF16>
KernelFn pick_opt(int opt, int ema) {
  switch (opt) {
    case OPT_SGD: return pick_ema<V, BF16, OPT_SGD>(ema);
    case OPT_MOMENTUM: return pick_ema<V, BF16, OPT_MOMENTUM>(ema);
    default: return pick_ema<V, BF16, OPT_RMSPROP_MOM>(ema);
  }
}
template <int V>
KernelFn pick_dtype(int dtype, int opt, int ema) {
  return dtype == 1 ? pick_opt<V, true>(opt, ema) : pick_opt<V, false>(opt, ema);
}
KernelFn pick_kernel(int v, int dtype, int opt, int ema) {
  switch (v) {
    case 0: return pick_dtype<0>(dtype, opt, ema);
    case 1: return pick_dtype<1>(dtype, opt, ema);
    case 2: return pick_dtype<2>(dtype, opt, ema);
    default: return pick_dtype<3>(dtype, opt, ema);
  }
}

int resolve_variant(int dtype, int variant) {
  if (variant >= 1 && variant <= kNumVariants) return variant - 1;
  return dtype == 1 ? 0 : 0;  // default: variant 1 (tuned on B200, see DESIGN.md s.6)
}

}  // namespace

int fused_num_variants() { return kNumVariants; }

int sm_count() {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      sms <= 0) {
    cudaGetLastError();
    return 148;
  }
  return sms;
}

cudaError_t fused_geometry(int dtype, int opt, int ema, int variant, int grid_ctas, int64_t P, FusedGeometry* out) {
  const int v = resolve_variant(dtype, variant);
  const Variant& vr = kVariants[v];
  const int E = dtype == 1 ? 8 : 4;
  out->block = vr.threads;
  out->tile_elems = vr.threads * vr.upt * E;
  out->smem_bytes = static_cast<int>(sizeof(const char*)) * kMaxWorkers;
  // One tile per CTA, always: the hardware CTA scheduler balances the tiles dynamically over the SMs, which
  // measured 2-3 % faster on B200 than a persistent grid with static striding (DESIGN.md s.5), and a kernel
  // without a tile loop stays inside 64 registers without spilling.  grid_ctas is accepted and ignored.
  (void)opt;
  (void)ema;
  (void)grid_ctas;
  const int64_t n_tiles = (P / E + static_cast<int64_t>(vr.threads) * vr.upt - 1) / (static_cast<int64_t>(vr.threads) * vr.upt);
  int64_t grid = n_tiles;
  if (grid > 0x7FFFFFFF) return cudaErrorInvalidConfiguration;  // > 2^41 parameters: not addressable in HBM anyway
  if (grid < 1) grid = 1;
  out->grid = static_cast<int>(grid);
  return cudaSuccess;
}

cudaError_t launch_fused(const FusedParams& p, int dtype, int opt, int ema, int variant, int grid_ctas,
                         cudaStream_t stream) {
  FusedGeometry g;
  cudaError_t err = fused_geometry(dtype, opt, ema, variant, grid_ctas, p.P, &g);
  if (err != cudaSuccess) return err;
  const int v = resolve_variant(dtype, variant);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(static_cast<unsigned>(g.grid));
  cfg.blockDim = dim3(static_cast<unsigned>(g.block));
  cfg.dynamicSmemBytes = 0;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, (p.per_shard || p.n_kept != nullptr) ? pick_rows_kernel(dtype, opt, ema) : pick_kernel(v, dtype, opt, ema), p);
}

cudaError_t launch_ema(float* d_ema, const float* d_theta, int64_t P, float alpha, cudaStream_t stream) {
  const int aligned = ((reinterpret_cast<uintptr_t>(d_ema) | reinterpret_cast<uintptr_t>(d_theta)) & 15u) == 0;
  int64_t blocks = (P / 4 + 255) / 256;
  const int64_t cap = static_cast<int64_t>(sm_count()) * 8;
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  ema_kernel<<<static_cast<int>(blocks), 256, 0, stream>>>(d_ema, d_theta, P, alpha, 1.0f - alpha, aligned);
  return cudaGetLastError();
}

}  // namespace psync
