// K2s: the SHARD-AWARE fused aggregate + update + EMA -- Alg. 4 l.8-9 as parameter server j
// runs it: server j owns theta[j] (L42), receives the slice G_k[j] of every worker's gradient (L152) and applies
//     theta(t+1)[j] <- theta(t)[j] - (gamma_t / n_j) sum_{k in kept_j} G_k[j];   ema[j] <- alpha ema[j] + (1-alpha) theta[j]
//
// Two gradient layouts (psync_step.grad_layout):
//   SLICES  d_grads is [W*M]: entry k*M + j -> the len_j elements of G_k[j], each its own allocation with its
//           own alignment (what a parameter server, or the landing buffer of a reduce-scatter, holds);
//   FLAT    d_grads is [W] flat P-element buffers; server j's slice of worker k starts at element off[j].
// and any kept-row mode (one shared row, one row per server, device-side counts).
//
// Work list (hard part 4): the grid is one CTA per (server, tile); tile_start[j] is the
// prefix sum of ceil(len_j / TILE) (psync_shard_worklist), a CTA finds its server by binary search.  A tile never
// straddles two servers, so every CTA stages ONE kept row and streams with 128-bit loads.
//
// Alignment (hard part 3): the 128-bit stream is aligned to the GRADIENT slices -- they are 96 % of the bytes.
// The first kept worker's slice base fixes a head peel h: the elements before its first 128-byte boundary
// (< 32 fp32 / < 64 bf16), so that every warp-level 512-byte request covers exactly four 128-byte lines (a tile that
// starts on a 16-byte but not a 128-byte boundary costs 12 % more L2 sector traffic and 1.5 % of the kernel: ncu,
// profiles/r2_sharded.md); units are [h + uE, h + (u+1)E) of the slice.  A kept worker whose base has another
// 16-byte phase is read with narrower loads (that worker only); the head/tail peel is done element by element by the
// server's first CTA.  theta / state / ema start at element off[j] + h of flat arrays, which for ragged cuts is NOT
// 16-byte aligned in general: then each WARP transposes its 32 sums through shared memory (no CTA barrier: a
// __syncthreads here cost 3 % -- every warp waited for the CTA's slowest gradient load) and theta / state / ema are
// read and written as coalesced 32-bit accesses (lane l <-> elements l, l + 32, ... of the warp's 128- or 256-element
// segment), so they still move every byte once.
// The arithmetic per element is exactly K2's (same fixed-order fp32 sum, same update_element): bit-identical.

#include "psync_device.cuh"

namespace psync {
namespace {

using namespace dev;

constexpr int kThreads = 256;  // = PSYNC_TILE_UNITS: one 16-byte unit per thread
constexpr int kU = 8;          // independent 128-bit loads in flight per thread

template <bool BF16, int OPT, int EMA, int MINB>
__global__ void __launch_bounds__(kThreads, MINB) sharded_aggregate_update_ema(const FusedParams p) {
  constexpr int E = BF16 ? 8 : 4;
  constexpr int ESZ = BF16 ? 2 : 4;
  constexpr int Q = E / 4;
  __shared__ const char* s_ptr[kMaxWorkers];
  __shared__ __align__(16) float s_acc[kThreads * E];

  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  // ---- which (server, tile) is this CTA; its kept row ---------------------------------------------------------
  // The prologue is a chain of dependent loads that every CTA pays before its first gradient byte moves, so it is kept
  // SHORT: the server by a warp-wide search (1-2 levels), then everything that only needs j in ONE level -- shard
  // bounds, tile origin, status, count, this thread's entry of the kept row and the row's first entry -- loaded before
  // any of it is checked (all of these addresses are valid whatever the values turn out to be), then the slice
  // pointers in one more level.
  const int64_t b = blockIdx.x;
  // The grid is the work list's total, computed by the host from the shard table; a table built for another gradient
  // dtype (another tile size) has another total: then nothing is touched, instead of a partial update.
  const int64_t total = p.tile_start[p.M];
  const int j = upper_slot_warp(p.tile_start, p.M, b);
  const int row = p.per_shard ? j : 0;
  const int32_t* kept = p.kept + static_cast<int64_t>(row) * p.kept_stride;
  const int64_t off_j = p.shard_off[j];
  const int64_t off_j1 = p.shard_off[j + 1];
  const int64_t tile0 = p.tile_start[j];
  const int st = p.status != nullptr ? p.status[row] : 0;
  const int N = p.n_kept != nullptr ? p.n_kept[row] : p.N;
  const int k_first = kept[0];
  const int i_mine = static_cast<int>(threadIdx.x) < p.kept_stride ? static_cast<int>(threadIdx.x) : p.kept_stride - 1;
  const int k_mine = kept[i_mine];
  if (total != static_cast<int64_t>(gridDim.x)) return;
  if (st != 0) return;  // this server did not collect its gradients
  if (N <= 0 || N > p.kept_stride || N > kMaxWorkers) return;  // a count nobody wrote: treat the row as failed
  const int64_t len_j = off_j1 - off_j;
  const int64_t tile = b - tile0;
  const float inv_N = p.n_kept ? 1.0f / static_cast<float>(N) : p.inv_N;

  // ---- stage server j's kept row as slice base pointers; the first one fixes the phase ---------------------
  // Every thread reads the row's first pointer itself (one address for the whole CTA: a broadcast), so the head peel
  // is known before the staging pass and one barrier is enough.
  auto slice_ptr = [&](int k) -> const char* {
    return p.slices ? static_cast<const char*>(p.grads[static_cast<int64_t>(k) * p.M + j])
                    : static_cast<const char*>(p.grads[k]) + off_j * ESZ;
  };
  const char* g_first = slice_ptr(k_first);
  const char* g_mine = static_cast<int>(threadIdx.x) < N ? slice_ptr(k_mine) : g_first;
  const unsigned ref = static_cast<unsigned>(reinterpret_cast<uintptr_t>(g_first)) & 127u;
  const int h = static_cast<int>(((128u - ref) & 127u) / ESZ);  // head peel: elements before the first 128-byte line
  unsigned mis = 0;
  for (int i = threadIdx.x; i < N; i += kThreads) {
    const char* g = i < kThreads ? g_mine : slice_ptr(kept[i]);
    mis |= ((static_cast<unsigned>(reinterpret_cast<uintptr_t>(g)) ^ ref) & 15u);  // another 16-byte phase
    s_ptr[i] = g + h * ESZ;  // unit u of this worker = s_ptr[i] + 16 u
  }
  const bool mixed = __syncthreads_or(static_cast<int>(mis)) != 0;  // some kept worker has another phase

  const int64_t nu = len_j > h ? (len_j - h) / E : 0;  // whole units of this server
  const int64_t u0 = tile * kThreads;
  const int64_t e0 = off_j + h;                        // parameter index of unit 0's first element

  if (u0 < nu) {
    const int64_t live_units = (nu - u0 < kThreads) ? (nu - u0) : kThreads;
    const bool live = threadIdx.x < live_units;
    const int64_t unit = live ? (u0 + threadIdx.x) : (nu - 1);  // dead slots re-read a valid unit, store nothing
    const bool theta_vec = p.base_aligned != 0 && (e0 & 3) == 0;  // CTA-uniform: theta co-aligned with the units
    // transposed epilogue: lane l of a warp owns elements l, l + 32, ... of the warp's segment of 32 units
    constexpr int SEG = 32 * E;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t seg_e0 = e0 + (u0 + warp * 32) * E;              // parameter index of the segment
    const int64_t live_in_seg = (live_units - warp * 32) * E;      // may be <= 0 (dead warp) or > SEG

    // theta / state / ema in registers: float4 per unit (co-aligned) or E scalars (transposed); both are E values
    float th[E], em[E], a0[E], a1[E];
    auto load_state = [&]() {
      if (theta_vec) {
#pragma unroll
        for (int q = 0; q < Q; ++q) {
          const int64_t e = e0 + unit * E + 4 * q;
          *reinterpret_cast<float4*>(&th[4 * q]) = ld_state16(p.theta + e);
          if (EMA != EMA_OFF) *reinterpret_cast<float4*>(&em[4 * q]) = ld_state16(p.ema + e);
          if (OPT != OPT_SGD) *reinterpret_cast<float4*>(&a0[4 * q]) = ld_state16(p.s0 + e);
          if (OPT == OPT_RMSPROP_MOM) *reinterpret_cast<float4*>(&a1[4 * q]) = ld_state16(p.s1 + e);
        }
      } else {
        const bool on = live_in_seg > 0;  // a dead warp must not touch memory
#pragma unroll
        for (int q = 0; q < E; ++q) {
          const int idx = q * 32 + lane;
          const int64_t e = seg_e0 + (idx < live_in_seg ? idx : 0);
          th[q] = on ? ld_state32(p.theta + e) : 0.f;
          if (EMA != EMA_OFF) em[q] = on ? ld_state32(p.ema + e) : 0.f;
          if (OPT != OPT_SGD) a0[q] = on ? ld_state32(p.s0 + e) : 1.f;
          if (OPT == OPT_RMSPROP_MOM) a1[q] = on ? ld_state32(p.s1 + e) : 0.f;
        }
      }
    };
    // HOIST (as in K2): with at most two fp32 state arrays their loads are issued WITH the last batch of gradient
    // loads -- one dependent memory round trip less per CTA, which is what small N is bound by.
    constexpr int kStateArrays = 1 + (EMA != EMA_OFF ? 1 : 0) + (OPT != OPT_SGD ? 1 : 0) + (OPT == OPT_RMSPROP_MOM ? 1 : 0);
    constexpr bool HOIST = !BF16 && kStateArrays <= 2;

    float acc[E];
#pragma unroll
    for (int e = 0; e < E; ++e) acc[e] = 0.f;

    if (!mixed) {
      int n = 0;
      const int n_loop = HOIST ? ((N - 1) / kU) * kU : (N / kU) * kU;  // HOIST keeps 1..kU gradients for the last batch
      for (; n < n_loop; n += kU) {
        uint4 r[kU];
#pragma unroll
        for (int u = 0; u < kU; ++u) r[u] = ldg_stream16(s_ptr[n + u] + unit * 16);
#pragma unroll
        for (int u = 0; u < kU; ++u) accumulate_unit<BF16>(acc, r[u]);  // strictly ascending worker order
      }
      if (HOIST || n < N) {
        uint4 r[kU];
#pragma unroll
        for (int u = 0; u < kU; ++u) {
          const bool on = (n + u) < N;
          r[u] = on ? ldg_stream16(s_ptr[on ? (n + u) : (N - 1)] + unit * 16) : make_uint4(0u, 0u, 0u, 0u);
        }
        if (HOIST) load_state();
#pragma unroll
        for (int u = 0; u < kU; ++u)
          if ((n + u) < N) accumulate_unit<BF16>(acc, r[u]);
      }
      if (!HOIST) load_state();
    } else {
#pragma unroll 4
      for (int n = 0; n < N; ++n) {
        const char* g = s_ptr[n];
        const uint4 r = load_unit_any<BF16>(g + unit * 16, (reinterpret_cast<uintptr_t>(g) & 15u) == 0);
        accumulate_unit<BF16>(acc, r);
      }
      load_state();
    }

    if (theta_vec) {
#pragma unroll
      for (int l = 0; l < E; ++l) update_element<OPT, EMA>(acc[l], inv_N, th[l], em[l], a0[l], a1[l], p);
      if (live) {
#pragma unroll
        for (int q = 0; q < Q; ++q) {
          const int64_t e = e0 + unit * E + 4 * q;
          st_state16(p.theta + e, *reinterpret_cast<float4*>(&th[4 * q]));
          if (EMA != EMA_OFF) st_state16(p.ema + e, *reinterpret_cast<float4*>(&em[4 * q]));
          if (OPT != OPT_SGD) st_state16(p.s0 + e, *reinterpret_cast<float4*>(&a0[4 * q]));
          if (OPT == OPT_RMSPROP_MOM) st_state16(p.s1 + e, *reinterpret_cast<float4*>(&a1[4 * q]));
        }
      }
    } else {
      // theta's slice is not co-aligned with the gradient units: every warp transposes its own 32 sums through
      // shared memory (__syncwarp only) and theta / state / ema move as coalesced 32-bit accesses.
      float* seg = s_acc + warp * SEG;
#pragma unroll
      for (int q = 0; q < Q; ++q)
        *reinterpret_cast<float4*>(&seg[(lane * Q + q) * 4]) =
            make_float4(acc[4 * q], acc[4 * q + 1], acc[4 * q + 2], acc[4 * q + 3]);
      __syncwarp();
#pragma unroll
      for (int q = 0; q < E; ++q) {
        const int idx = q * 32 + lane;
        update_element<OPT, EMA>(seg[idx], inv_N, th[q], em[q], a0[q], a1[q], p);
        if (idx < live_in_seg) {
          const int64_t e = seg_e0 + idx;
          st_state32(p.theta + e, th[q]);
          if (EMA != EMA_OFF) st_state32(p.ema + e, em[q]);
          if (OPT != OPT_SGD) st_state32(p.s0 + e, a0[q]);
          if (OPT == OPT_RMSPROP_MOM) st_state32(p.s1 + e, a1[q]);
        }
      }
    }
  }

  // ---- head and tail peel of server j (fewer than 2E elements), by its first CTA --------------------------
  if (tile == 0) {
    const int64_t tail0 = h + nu * E;  // first element after the whole units (h > len_j: everything is "head")
    const int64_t n_head = h < len_j ? h : len_j;
    const int64_t n_tail = len_j > tail0 ? len_j - tail0 : 0;
    if (threadIdx.x < n_head + n_tail) {
      const int64_t e = threadIdx.x < n_head ? threadIdx.x : tail0 + (threadIdx.x - n_head);
      float S = 0.f;
#pragma unroll 8
      for (int n = 0; n < N; ++n) S += load_grad_scalar<BF16>(s_ptr[n] - h * ESZ, e);
      update_in_memory<OPT, EMA>(p, S, inv_N, off_j + e);
    }
  }
}

// ---- work list: tile_start[j] = sum_{i<j} ceil(len_i / tile_elems), tile_start[M] = number of tiles ----------
__global__ void __launch_bounds__(1024) shard_worklist_kernel(const int64_t* shard_off, int32_t M, int32_t tile_elems,
                                                              int64_t* __restrict__ tile_start) {
  __shared__ int64_t s_warp[32];
  __shared__ int64_t s_carry;
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) {
    s_carry = 0;
    tile_start[0] = 0;
  }
  __syncthreads();
  for (int32_t base = 0; base < M; base += 1024) {  // 1024 servers per round, inclusive block scan
    const int32_t j = base + threadIdx.x;
    int64_t v = 0;
    if (j < M) {
      const int64_t len = shard_off[j + 1] - shard_off[j];
      v = (len + tile_elems - 1) / tile_elems;
    }
    int64_t incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int64_t up = __shfl_up_sync(0xFFFFFFFFu, incl, d);
      if (lane >= d) incl += up;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    if (warp == 0) {
      int64_t w = s_warp[lane];
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const int64_t up = __shfl_up_sync(0xFFFFFFFFu, w, d);
        if (lane >= d) w += up;
      }
      s_warp[lane] = w;
    }
    __syncthreads();
    const int64_t carry = s_carry;
    const int64_t before = warp > 0 ? s_warp[warp - 1] : 0;
    if (j < M) tile_start[j + 1] = carry + before + incl;
    __syncthreads();
    if (threadIdx.x == 1023) s_carry = carry + before + incl;
    __syncthreads();
  }
}

using KernelFn = void (*)(const FusedParams);

// bf16 gradients hold 8 parameters per thread: with RMSProp (40 live values) 3 CTAs/SM, like K2 (fused_kernel.cu)
template <bool BF16, int OPT>
KernelFn pick_ema(int ema) {
  constexpr int MINB = (BF16 && OPT == OPT_RMSPROP_MOM) ? 3 : 4;
  switch (ema) {
    case EMA_POST: return sharded_aggregate_update_ema<BF16, OPT, EMA_POST, MINB>;
    case EMA_PRE: return sharded_aggregate_update_ema<BF16, OPT, EMA_PRE, MINB>;
    default: return sharded_aggregate_update_ema<BF16, OPT, EMA_OFF, MINB>;
  }
}
template <bool BF16>
KernelFn pick_opt(int opt, int ema) {
  switch (opt) {
    case OPT_SGD: return pick_ema<BF16, OPT_SGD>(ema);
    case OPT_MOMENTUM: return pick_ema<BF16, OPT_MOMENTUM>(ema);
    default: return pick_ema<BF16, OPT_RMSPROP_MOM>(ema);
  }
}

}  // namespace

int sharded_tile_elems(int dtype) { return kThreads * (dtype == 1 ? 8 : 4); }

cudaError_t launch_shard_worklist_elems(const int64_t* d_shard_off, int32_t M, int32_t tile_elems, int64_t* d_tile_start,
                                        cudaStream_t stream) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(1);
  cfg.blockDim = dim3(1024);
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, shard_worklist_kernel, d_shard_off, M, tile_elems, d_tile_start);
}

cudaError_t launch_shard_worklist(const int64_t* d_shard_off, int32_t M, int dtype, int64_t* d_tile_start,
                                  cudaStream_t stream) {
  return launch_shard_worklist_elems(d_shard_off, M, static_cast<int32_t>(sharded_tile_elems(dtype)), d_tile_start, stream);
}

cudaError_t launch_sharded(const FusedParams& p, int dtype, int opt, int ema, int64_t n_tiles, cudaStream_t stream) {
  if (n_tiles <= 0) return cudaSuccess;
  if (n_tiles > 0x7FFFFFFF) return cudaErrorInvalidConfiguration;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(static_cast<unsigned>(n_tiles));
  cfg.blockDim = dim3(kThreads);
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, dtype == 1 ? pick_opt<true>(opt, ema) : pick_opt<false>(opt, ema), p);
}

}  // namespace psync
