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
    if (N <= 0 || N > p.kept_stride) continue;  // a count nobody wrote: the row counts as failed
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

  // HOIST: with at most two fp32 state arrays (SGD, or momentum without EMA) the theta / ema loads fit in registers
  // next to the last batch of gradient loads, so they are issued WITH it instead of after it: one memory round trip
  // less per CTA.  Nothing for N = 100 (other CTAs cover it), but a CTA with N = 8 lives for four round trips
  // (kept -> pointers -> gradients -> theta) and the small sweep points are latency-bound: a small gain there (P = 1 Mi,
  // N = 8: 3072 -> 3283 GB/s; 4 Mi, N = 8: 6133 -> 6190; profiles/r2_small_points.md).  Same loads, same adds in the same
  // order: same bits.
  constexpr int kStateArrays = 1 + (EMA != EMA_OFF ? 1 : 0) + (OPT != OPT_SGD ? 1 : 0) + (OPT == OPT_RMSPROP_MOM ? 1 : 0);
  constexpr bool HOIST = !BF16 && UPT == 1 && kStateArrays <= 2;
  float4 th[UPT][Q], em[UPT][Q], a0[UPT][Q], a1[UPT][Q];
  auto load_state = [&]() {
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
  };

  int n = 0;
  const int n_loop = HOIST ? ((N - 1) / U) * U : (N / U) * U;  // HOIST keeps 1..U gradients for the final batch
  for (; n < n_loop; n += U) {  // full batches: U x UPT independent 16-byte loads in flight
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
  if (HOIST || n < N) {  // last batch (partial unless HOIST and U divides N): same shape, predicated
    uint4 r[U][UPT];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const bool on = (n + u) < N;
      const char* g = s_ptr[on ? (n + u) : (N - 1)];
#pragma unroll
      for (int j = 0; j < UPT; ++j) r[u][j] = on ? ldg_stream16(g + unit[j] * 16) : make_uint4(0u, 0u, 0u, 0u);
    }
    if (HOIST) load_state();
#pragma unroll
    for (int u = 0; u < U; ++u)
      if ((n + u) < N) {
#pragma unroll
        for (int j = 0; j < UPT; ++j) accumulate_unit<BF16>(acc[j], r[u][j]);
      }
  }

  // theta / state / ema: loaded once the gradient registers are dead; other resident warps hide the latency
  if (!HOIST) load_state();

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
        bool bad_count = false;  // a device-side count outside [1, kept_stride] (never written, stale): failed row
        if (fast) {
          N = p.n_kept ? p.n_kept[row] : p.N;
          bad_count = N <= 0 || N > p.kept_stride || N > kMaxWorkers;
          if (bad_count) N = 0;
          inv_N = p.n_kept ? 1.0f / static_cast<float>(N) : p.inv_N;
          const unsigned misalign = stage_row<THREADS>(p, s_ptr, row, N);
          fast = __syncthreads_or(static_cast<int>(misalign)) == 0;
        }
        if (bad_count) {
          // leave the slice untouched
        } else if (fast)
          vector_tile<THREADS, UPT, U, BF16, OPT, EMA, false>(p, s_ptr, N, inv_N, tile, n_units);
        else
          rows_scalar_range<BF16, OPT, EMA>(p, e0, e1, threadIdx.x, THREADS);
      }
    }
    if (tail0 < p.P && blockIdx.x == 0) rows_scalar_range<BF16, OPT, EMA>(p, tail0, p.P, threadIdx.x, THREADS);
  }
}


// ---- variant 6: 256-bit loads (sm_100: ld.global.v8, SASS LDG.E.256) with L2::evict_first ----------------------
// Same schedule as vector_tile with 32-byte units: E = 8 (fp32) or 16 (bf16) parameters per thread, one tile per
// CTA, U independent loads in flight, strictly ascending worker order per element -- the same bits as every other
// variant.  Kept selectable so that the A/B against the 128-bit default can be re-run (profiles/r2_variants.md).
struct alignas(32) U8 {
  uint32_t v[8];
};
__device__ __forceinline__ U8 ldg_stream32(const void* p) {
  U8 r;
  asm volatile("ld.global.nc.L1::no_allocate.L2::evict_first.v8.u32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(r.v[0]), "=r"(r.v[1]), "=r"(r.v[2]), "=r"(r.v[3]), "=r"(r.v[4]), "=r"(r.v[5]), "=r"(r.v[6]),
                 "=r"(r.v[7])
               : "l"(p));
  return r;
}

template <int THREADS, int U, int MINB, bool BF16, int OPT, int EMA>
__global__ void __launch_bounds__(THREADS, MINB) fused_aggregate_update_ema_v256(const FusedParams p) {
  constexpr int E = BF16 ? 16 : 8;  // parameters per 32-byte unit
  constexpr int Q = E / 4;
  __shared__ const char* s_ptr[kMaxWorkers];
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  if (p.status != nullptr && *p.status != 0) return;
  unsigned misalign = 0;
  for (int n = threadIdx.x; n < p.N; n += THREADS) {
    const char* g = static_cast<const char*>(p.grads[p.kept[n]]);
    s_ptr[n] = g;
    misalign |= static_cast<unsigned>(reinterpret_cast<uintptr_t>(g)) & 31u;
  }
  const bool vec_ok = (__syncthreads_or(static_cast<int>(misalign)) == 0) && (p.base_aligned != 0);
  if (!vec_ok) {
    scalar_range<BF16, OPT, EMA>(p, s_ptr, 0, p.P, static_cast<int64_t>(blockIdx.x) * THREADS + threadIdx.x,
                                 static_cast<int64_t>(gridDim.x) * THREADS);
    return;
  }
  const int64_t n_units = p.P / E;
  const int64_t tail0 = n_units * E;
  const int64_t u = static_cast<int64_t>(blockIdx.x) * THREADS + threadIdx.x;
  if (static_cast<int64_t>(blockIdx.x) * THREADS < n_units) {
    const bool live = u < n_units;
    const int64_t unit = live ? u : (n_units - 1);
    const int N = p.N;
    float acc[E];
#pragma unroll
    for (int e = 0; e < E; ++e) acc[e] = 0.f;
    auto add_unit = [&acc](const U8& r) {
      const uint4 lo = make_uint4(r.v[0], r.v[1], r.v[2], r.v[3]), hi = make_uint4(r.v[4], r.v[5], r.v[6], r.v[7]);
      accumulate_unit<BF16>(acc, lo);
      accumulate_unit<BF16>(acc + E / 2, hi);
    };
    int n = 0;
    for (; n + U <= N; n += U) {
      U8 r[U];
#pragma unroll
      for (int v = 0; v < U; ++v) r[v] = ldg_stream32(s_ptr[n + v] + unit * 32);
#pragma unroll
      for (int v = 0; v < U; ++v) add_unit(r[v]);
    }
    for (; n < N; ++n) add_unit(ldg_stream32(s_ptr[n] + unit * 32));

    float4 th[Q], em[Q], a0[Q], a1[Q];
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      const int64_t e = unit * E + 4 * q;
      th[q] = ld_state16(p.theta + e);
      if (EMA != EMA_OFF) em[q] = ld_state16(p.ema + e);
      if (OPT != OPT_SGD) a0[q] = ld_state16(p.s0 + e);
      if (OPT == OPT_RMSPROP_MOM) a1[q] = ld_state16(p.s1 + e);
    }
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      float* t4 = reinterpret_cast<float*>(&th[q]);
      float* e4 = reinterpret_cast<float*>(&em[q]);
      float* x4 = reinterpret_cast<float*>(&a0[q]);
      float* y4 = reinterpret_cast<float*>(&a1[q]);
#pragma unroll
      for (int l = 0; l < 4; ++l) update_element<OPT, EMA>(acc[4 * q + l], p.inv_N, t4[l], e4[l], x4[l], y4[l], p);
      if (live) {
        const int64_t e = unit * E + 4 * q;
        st_state16(p.theta + e, th[q]);
        if (EMA != EMA_OFF) st_state16(p.ema + e, em[q]);
        if (OPT != OPT_SGD) st_state16(p.s0 + e, a0[q]);
        if (OPT == OPT_RMSPROP_MOM) st_state16(p.s1 + e, a1[q]);
      }
    }
  }
  if (tail0 < p.P && blockIdx.x == 0) scalar_range<BF16, OPT, EMA>(p, s_ptr, tail0, p.P, threadIdx.x, THREADS);
}

// ---- variant 5: TMA bulk staging -- cp.async.bulk global -> shared through an mbarrier ring ----------------------
// One producer thread (warp CONSUMERS/32, lane 0) issues one cp.async.bulk per kept worker: that worker's 4 KB row
// of the CTA's tile (256 16-byte units) into stage n % STAGES, completion counted in bytes on full[stage].  The 256
// consumer threads wait for the stage, add their 16-byte unit from shared memory (ascending worker order, so the
// same bits as every other variant) and release it on empty[stage] (one arrival per consumer warp).  Bytes in
// flight no longer cost registers: STAGES x 4 KB per CTA.  Needs 16-byte aligned buffers (like the 128-bit path).
// Kept selectable so that the A/B against plain 128-bit loads can be re-run (profiles/r2_variants.md).
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  asm volatile(
      "{\n\t.reg .pred ok;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 ok, [%0], %1;\n\t"
      "@ok bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, uint64_t* bar, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}

template <int STAGES, int MINB, bool BF16, int OPT, int EMA>
__global__ void __launch_bounds__(256 + 32, MINB) fused_aggregate_update_ema_bulk(const FusedParams p) {
  constexpr int CONSUMERS = 256;
  constexpr int E = BF16 ? 8 : 4;
  constexpr int Q = E / 4;
  constexpr unsigned kRowBytes = CONSUMERS * 16;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint4* stage = reinterpret_cast<uint4*>(smem_raw);                                      // [STAGES][256] x 16 B
  const char** s_ptr = reinterpret_cast<const char**>(smem_raw + STAGES * kRowBytes);    // [kMaxWorkers]
  uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + STAGES * kRowBytes + sizeof(char*) * kMaxWorkers);
  uint64_t* empty = full + STAGES;

  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  if (p.status != nullptr && *p.status != 0) return;
  unsigned misalign = 0;
  for (int n = threadIdx.x; n < p.N; n += CONSUMERS + 32) {
    const char* g = static_cast<const char*>(p.grads[p.kept[n]]);
    s_ptr[n] = g;
    misalign |= static_cast<unsigned>(reinterpret_cast<uintptr_t>(g)) & 15u;
  }
  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(&full[s], 1);               // the producer's arrive.expect_tx; the copy completes the bytes
      mbar_init(&empty[s], CONSUMERS / 32);  // one arrival per consumer warp
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  const bool vec_ok = (__syncthreads_or(static_cast<int>(misalign)) == 0) && (p.base_aligned != 0);
  if (!vec_ok) {
    if (threadIdx.x < CONSUMERS)
      scalar_range<BF16, OPT, EMA>(p, s_ptr, 0, p.P, static_cast<int64_t>(blockIdx.x) * CONSUMERS + threadIdx.x,
                                   static_cast<int64_t>(gridDim.x) * CONSUMERS);
    return;
  }
  const int N = p.N;
  const int64_t n_units = p.P / E;
  const int64_t tail0 = n_units * E;
  const int64_t u0 = static_cast<int64_t>(blockIdx.x) * CONSUMERS;
  const bool has_tile = u0 < n_units;
  const int64_t live_units = has_tile ? ((n_units - u0 < CONSUMERS) ? (n_units - u0) : CONSUMERS) : 0;

  if (threadIdx.x >= CONSUMERS) {  // ---- producer warp
    if (threadIdx.x == CONSUMERS && has_tile) {
      uint64_t policy;
      asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
      const unsigned bytes = static_cast<unsigned>(live_units) * 16u;
      for (int n = 0; n < N; ++n) {
        const int s = n % STAGES;
        if (n >= STAGES) mbar_wait(&empty[s], ((n / STAGES) - 1) & 1);  // every consumer warp has read the slot
        mbar_expect_tx(&full[s], bytes);
        bulk_g2s(stage + s * CONSUMERS, s_ptr[n] + u0 * 16, bytes, &full[s], policy);
      }
    }
    return;
  }

  // ---- consumers
  if (has_tile) {
    const bool live = threadIdx.x < live_units;
    const int64_t unit = u0 + (live ? threadIdx.x : 0);
    float acc[E];
#pragma unroll
    for (int e = 0; e < E; ++e) acc[e] = 0.f;
    for (int n = 0; n < N; ++n) {
      const int s = n % STAGES;
      mbar_wait(&full[s], (n / STAGES) & 1);
      const uint4 r = live ? stage[s * CONSUMERS + threadIdx.x] : make_uint4(0u, 0u, 0u, 0u);
      __syncwarp();
      if ((threadIdx.x & 31) == 0) mbar_arrive(&empty[s]);
      accumulate_unit<BF16>(acc, r);
    }
    float4 th[Q], em[Q], a0[Q], a1[Q];
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      const int64_t e = unit * E + 4 * q;
      th[q] = ld_state16(p.theta + e);
      if (EMA != EMA_OFF) em[q] = ld_state16(p.ema + e);
      if (OPT != OPT_SGD) a0[q] = ld_state16(p.s0 + e);
      if (OPT == OPT_RMSPROP_MOM) a1[q] = ld_state16(p.s1 + e);
    }
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      float* t4 = reinterpret_cast<float*>(&th[q]);
      float* e4 = reinterpret_cast<float*>(&em[q]);
      float* x4 = reinterpret_cast<float*>(&a0[q]);
      float* y4 = reinterpret_cast<float*>(&a1[q]);
#pragma unroll
      for (int l = 0; l < 4; ++l) update_element<OPT, EMA>(acc[4 * q + l], p.inv_N, t4[l], e4[l], x4[l], y4[l], p);
      if (live) {
        const int64_t e = unit * E + 4 * q;
        st_state16(p.theta + e, th[q]);
        if (EMA != EMA_OFF) st_state16(p.ema + e, em[q]);
        if (OPT != OPT_SGD) st_state16(p.s0 + e, a0[q]);
        if (OPT == OPT_RMSPROP_MOM) st_state16(p.s1 + e, a1[q]);
      }
    }
  }
  if (tail0 < p.P && blockIdx.x == 0) scalar_range<BF16, OPT, EMA>(p, s_ptr, tail0, p.P, threadIdx.x, CONSUMERS);
}

// ---- variant 7: per-thread cp.async ring (the staging Alg. 2's kernels use, async_kernel.cu) --------------------
// Every thread copies the 16-byte units of its own column of the kept buffers into its own slots of a D-deep ring in
// shared memory (cp.async.cg, SASS LDGSTS.E.BYPASS.128; one commit group per buffer) and adds them in ascending worker
// order as they land (cp.async.wait_group): no barrier, no mbarrier, no producer warp, and no registers for loads in
// flight -- so theta / state / ema are requested right after the ring is filled, not after the gradient stream, for
// EVERY instance (one dependent round trip less per CTA).  Same adds in the same order: the same bits as variant 1.
template <int D, int MINB, bool BF16, int OPT, int EMA>
__global__ void __launch_bounds__(256, MINB) fused_aggregate_update_ema_tring(const FusedParams p) {
  constexpr int THREADS = 256;
  constexpr int E = BF16 ? 8 : 4;
  constexpr int Q = E / 4;
  __shared__ const char* s_ptr[kMaxWorkers];
  __shared__ __align__(16) uint4 s_ring[D][THREADS];

  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  const int64_t n_units = p.P / E;
  const int64_t n_tiles = (n_units + THREADS - 1) / THREADS;
  const int64_t tail0 = n_units * E;
  if (p.status != nullptr && *p.status != 0) return;
  const unsigned misalign = stage_row<THREADS>(p, s_ptr, 0, p.N);
  const bool vec_ok = (__syncthreads_or(static_cast<int>(misalign)) == 0) && (p.base_aligned != 0);
  if (!vec_ok) {
    scalar_range<BF16, OPT, EMA>(p, s_ptr, 0, p.P, static_cast<int64_t>(blockIdx.x) * THREADS + threadIdx.x,
                                 static_cast<int64_t>(gridDim.x) * THREADS);
    return;
  }
  if (blockIdx.x < n_tiles) {
    const int N = p.N;
    const int64_t u = static_cast<int64_t>(blockIdx.x) * THREADS + threadIdx.x;
    const bool live = u < n_units;
    const int64_t unit = live ? u : (n_units - 1);  // dead slots re-read a valid unit and store nothing
    const uint32_t slot0 = static_cast<uint32_t>(__cvta_generic_to_shared(&s_ring[0][threadIdx.x]));
#pragma unroll
    for (int i = 0; i < D; ++i) {
      if (i < N)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(slot0 + i * THREADS * 16), "l"(s_ptr[i] + unit * 16)
                     : "memory");
      asm volatile("cp.async.commit_group;" ::: "memory");
    }
    float4 th[Q], em[Q], a0[Q], a1[Q];
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      const int64_t e = unit * E + 4 * q;
      th[q] = ld_state16(p.theta + e);
      if (EMA != EMA_OFF) em[q] = ld_state16(p.ema + e);
      if (OPT != OPT_SGD) a0[q] = ld_state16(p.s0 + e);
      if (OPT == OPT_RMSPROP_MOM) a1[q] = ld_state16(p.s1 + e);
    }
    float acc[E];
#pragma unroll
    for (int e = 0; e < E; ++e) acc[e] = 0.f;
    auto one = [&](int i, int slot) {
      asm volatile("cp.async.wait_group %0;" ::"n"(D - 1) : "memory");  // buffer i has landed (groups retire in order)
      const uint4 r = s_ring[slot][threadIdx.x];
      accumulate_unit<BF16>(acc, r);  // strictly ascending worker order
      if (i + D < N)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(slot0 + slot * THREADS * 16),
                     "l"(s_ptr[i + D] + unit * 16)
                     : "memory");
      asm volatile("cp.async.commit_group;" ::: "memory");
    };
    int i0 = 0;
    for (; i0 + D <= N; i0 += D) {
#pragma unroll
      for (int v = 0; v < D; ++v) one(i0 + v, v);
    }
    for (int i = i0; i < N; ++i) one(i, i - i0);
    asm volatile("cp.async.wait_group 0;" ::: "memory");
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      float* t4 = reinterpret_cast<float*>(&th[q]);
      float* e4 = reinterpret_cast<float*>(&em[q]);
      float* x4 = reinterpret_cast<float*>(&a0[q]);
      float* y4 = reinterpret_cast<float*>(&a1[q]);
#pragma unroll
      for (int l = 0; l < 4; ++l) update_element<OPT, EMA>(acc[4 * q + l], p.inv_N, t4[l], e4[l], x4[l], y4[l], p);
      if (live) {
        const int64_t e = unit * E + 4 * q;
        st_state16(p.theta + e, th[q]);
        if (EMA != EMA_OFF) st_state16(p.ema + e, em[q]);
        if (OPT != OPT_SGD) st_state16(p.s0 + e, a0[q]);
        if (OPT == OPT_RMSPROP_MOM) st_state16(p.s1 + e, a1[q]);
      }
    }
  }
  if (tail0 < p.P && blockIdx.x == 0) scalar_range<BF16, OPT, EMA>(p, s_ptr, tail0, p.P, threadIdx.x, THREADS);
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
enum VariantKind { kPlain128 = 0, kBulkRing = 1, kPlain256 = 2, kThreadRing = 3, kRemoved = 4 };
struct Variant {
  int threads, upt, unroll, minb, kind;
};
// variant ids are 1-based in the ABI (0 = default)
constexpr Variant kVariants[] = {
    {256, 1, 8, 4, kPlain128},    // 1  the default: 128-bit loads, 8 in flight per thread, 4 CTAs/SM
    {256, 2, 8, 2, kRemoved},     // 2  } other tile shapes of the plain kernel (2 units per thread, 16 loads in flight,
    {256, 1, 16, 3, kRemoved},    // 3  } 512 threads): "no size at which one wins" (profiles/r2_variants.md), removed
    {512, 1, 8, 2, kRemoved},     // 4  } after round 2 -- the ids stay reserved and return PSYNC_EUNSUPPORTED
    {256, 1, 12, 3, kBulkRing},   // 5  cp.async.bulk -> 12-stage shared-memory ring (unroll = stages), 1 producer warp
    {256, 1, 8, 2, kPlain256},    // 6  256-bit loads with L2::evict_first, 8 in flight per thread
    {256, 1, 8, 4, kThreadRing},  // 7  per-thread cp.async ring in shared memory (unroll = depth), state requested up front
    {128, 1, 8, 8, kRemoved},     // 8  half-size tiles (128 threads, 8 CTAs/SM): no gain (profiles/r2_small_points.md), removed
};
constexpr int kNumVariants = sizeof(kVariants) / sizeof(kVariants[0]);
constexpr int kRingStages = kVariants[4].unroll;
constexpr int kRingSmemBytes = kRingStages * 256 * 16 + static_cast<int>(sizeof(const char*)) * kMaxWorkers + 2 * kRingStages * 8;

using KernelFn = void (*)(const FusedParams);

// bf16 gradients with RMSProp hold 8 parameters x (acc, theta, ema, ms, mom) = 40 live values per thread:
// at 4 CTAs/SM (64 registers) that spills, so this one combination runs at 3 CTAs/SM (85 registers).
constexpr int minb_for(int v, bool bf16, int opt) {
  const int cap = 768 / kVariants[v].threads;  // resident threads per SM that leave 85 registers each
  return (bf16 && opt == OPT_RMSPROP_MOM && kVariants[v].minb > cap) ? cap : kVariants[v].minb;
}

template <int V, bool BF16, int OPT, int EMA, bool ROWS = false>
constexpr KernelFn kernel_for() {
  if constexpr (kVariants[V].kind == kBulkRing)
    return fused_aggregate_update_ema_bulk<kVariants[V].unroll, kVariants[V].minb, BF16, OPT, EMA>;
  else if constexpr (kVariants[V].kind == kThreadRing)
    return fused_aggregate_update_ema_tring<kVariants[V].unroll, minb_for(V, BF16, OPT), BF16, OPT, EMA>;
  else if constexpr (kVariants[V].kind == kPlain256)
    return fused_aggregate_update_ema_v256<kVariants[V].threads, kVariants[V].unroll, (BF16 ? 1 : kVariants[V].minb),
                                           BF16, OPT, EMA>;
  else
    return fused_aggregate_update_ema<kVariants[V].threads, kVariants[V].upt, kVariants[V].unroll,
                                      minb_for(V, BF16, OPT), BF16, OPT, EMA, ROWS>;
}

// kept rows with a device-side count / one row per server in the flat index space: the default variant only
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
    case 4: return pick_dtype<4>(dtype, opt, ema);
    case 5: return pick_dtype<5>(dtype, opt, ema);
    case 6: return pick_dtype<6>(dtype, opt, ema);
    default: return nullptr;  // a removed variant (the ABI refuses it before it gets here)
  }
}

int resolve_variant(int variant) {
  if (variant >= 1 && variant <= kNumVariants) return variant - 1;
  return 0;  // default: variant 1 (tuned on B200, DESIGN.md s.5; the A/B of all six is profiles/r2_variants.md)
}

}  // namespace

int fused_num_variants() { return kNumVariants; }

bool fused_variant_exists(int variant) {
  return variant == 0 || (variant >= 1 && variant <= kNumVariants && kVariants[variant - 1].kind != kRemoved);
}

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
  const int v = resolve_variant(variant);
  const Variant& vr = kVariants[v];
  const int E = (dtype == 1 ? 8 : 4) * (vr.kind == kPlain256 ? 2 : 1);  // parameters per 16- or 32-byte unit
  out->block = vr.threads + (vr.kind == kBulkRing ? 32 : 0);           // + the producer warp
  out->tile_elems = vr.threads * vr.upt * E;
  out->smem_bytes = vr.kind == kBulkRing ? kRingSmemBytes
                    : static_cast<int>(sizeof(const char*)) * kMaxWorkers + (vr.kind == kThreadRing ? vr.unroll * 256 * 16 : 0);
  // One tile per CTA, always: the hardware CTA scheduler balances the tiles dynamically over the SMs, which
  // measured 2-3 % faster on B200 than a persistent grid with static striding (DESIGN.md s.5), and a kernel
  // without a tile loop stays inside 64 registers without spilling.  grid_ctas is accepted and ignored.
  (void)opt;
  (void)ema;
  (void)grid_ctas;
  const int64_t n_tiles = (P / E + static_cast<int64_t>(vr.threads) * vr.upt - 1) / (static_cast<int64_t>(vr.threads) * vr.upt);  // E: per unit of this variant
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
  const int v = resolve_variant(variant);
  const bool rows = p.per_shard || p.n_kept != nullptr;
  const KernelFn kernel = rows ? pick_rows_kernel(dtype, opt, ema) : pick_kernel(v, dtype, opt, ema);
  if (kernel == nullptr) return cudaErrorInvalidValue;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(static_cast<unsigned>(g.grid));
  cfg.blockDim = dim3(static_cast<unsigned>(g.block));
  cfg.dynamicSmemBytes = 0;
  if (!rows && kVariants[v].kind == kBulkRing) {  // the ring lives in dynamic shared memory (> 48 KB: opt in)
    cfg.dynamicSmemBytes = kRingSmemBytes;
    err = cudaFuncSetAttribute(reinterpret_cast<const void*>(kernel), cudaFuncAttributeMaxDynamicSharedMemorySize,
                               kRingSmemBytes);
    if (err != cudaSuccess) return err;
  }
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, p);
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
