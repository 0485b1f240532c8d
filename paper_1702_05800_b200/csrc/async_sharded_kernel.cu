// K4s: Alg. 2 run LITERALLY PER PARAMETER SERVER j -- "Async-SGD Parameter Server j":
//
//     for t = 0, 1, ...:  wait for gradient G from any worker                       (L85)
//                         theta(t+1)[j] <- theta(t)[j] - gamma_t G[j]               (L86)
//                         ema(t)[j] = alpha ema(t-1)[j] + (1-alpha) theta(t)[j]     (L87)
//
// Every server runs this loop on its own: the order in which the gradients reach server j, and how many have
// arrived, is server j's (the same remark as for Alg. 4), and what it receives is G[j] -- with
// PSYNC_GRADS_SLICES one buffer per (worker, server), each its own allocation with its own alignment; with flat
// buffers the range [off[j], off[j+1]) of each.  Row r(j) = per_shard ? j : 0 of the order table lists the workers
// in the order server j applies them, K_j = n_kept ? n_kept[r] : N of them; gammas[i] is the rate of the server's
// i-th iteration of this batch, gscales[k] worker k's clip factor (L313).
//
// Same CTA <-> data mapping as the synchronous shard-aware kernel K2s (sharded_kernel.cu): one CTA per (server,
// tile) of the work list, the 128-bit gradient stream aligned to the server's first slice (head peel to its first
// 128-byte line), narrower loads for a slice with another 16-byte phase, head / tail elements done one by one by the
// server's first CTA.  Same arithmetic per element as K4 (async_kernel.cu: K dependent optimizer steps + EMAs in
// registers, packed fp32x2, the gradient stream staged through a per-thread cp.async ring): bit-identical to it and to K launches of the
// synchronous step with N = 1 (tested).
// What differs from K2s: the state cannot wait for the end of the gradient stream -- every arriving gradient is
// applied to it -- so when theta's slice is not co-aligned with the gradient units (ragged cuts: off[j] + h is not a
// multiple of 4) each warp moves theta / state / ema as coalesced 32-bit accesses and transposes them through shared
// memory ONCE on the way in and once on the way out (K-independent; the gradient stream stays 128-bit).

#include "async_common.cuh"

namespace psync {
namespace {

using namespace dev;

constexpr int kThreads = 256;  // = PSYNC_TILE_UNITS: one 16-byte unit per thread

// Where this thread's unit and its warp's segment lie, derived from four CTA-uniform numbers.  The kernel derives it
// twice: before the gradient loop from registers, and after it from a copy of the four numbers in shared memory read
// through a volatile pointer -- so that none of these addresses stays live across the loop, which needs all of the 64
// registers that 4 CTAs/SM allow for the state, the update's temporaries and the stream's addresses.  (History: in
// the register-pipelined form of the loop ptxas, short of registers, merged the two gradient buffers into one and the
// warp waited for every batch -- 48 % of all stall samples; profiles/r2_async.md.)
template <int E>
struct Geom {
  int64_t nu, u0, e0, unit, seg_e0, live_in_seg;
  bool live, theta_vec;
  int lane;
  float* seg;
};
template <int E>
__device__ __forceinline__ Geom<E> make_geom(int64_t off_j, int64_t len_j, int h, int64_t tile, int base_aligned,
                                             float* s_seg) {
  Geom<E> g;
  g.nu = len_j > h ? (len_j - h) / E : 0;  // whole units of this server
  g.u0 = tile * kThreads;
  g.e0 = off_j + h;                        // parameter index of unit 0's first element
  const int64_t live_units = (g.nu - g.u0 < kThreads) ? (g.nu - g.u0) : kThreads;
  g.live = threadIdx.x < live_units;
  g.unit = g.live ? (g.u0 + threadIdx.x) : (g.nu - 1);  // dead slots re-read a valid unit, store nothing
  g.theta_vec = base_aligned != 0 && (g.e0 & 3) == 0;   // CTA-uniform: theta co-aligned with the units
  const int warp = threadIdx.x >> 5;
  g.lane = threadIdx.x & 31;
  g.seg_e0 = g.e0 + (g.u0 + warp * 32) * E;
  g.live_in_seg = (live_units - warp * 32) * E;  // <= 0 for a dead warp: it touches no memory
  g.seg = s_seg + warp * (32 * E);
  return g;
}

// one array's E values of this thread's unit: 128-bit when co-aligned, else coalesced 32-bit + warp transpose
template <int E>
__device__ __forceinline__ void load_arr(const Geom<E>& g, const float* arr, float4* dst, float fill) {
  constexpr int Q = E / 4;
  if (g.theta_vec) {
#pragma unroll
    for (int q = 0; q < Q; ++q) dst[q] = ld_state16(arr + g.e0 + g.unit * E + 4 * q);
  } else {
#pragma unroll
    for (int q = 0; q < E; ++q) {
      const int idx = q * 32 + g.lane;
      g.seg[idx] = idx < g.live_in_seg ? ld_state32(arr + g.seg_e0 + idx) : fill;
    }
    __syncwarp();
#pragma unroll
    for (int q = 0; q < Q; ++q) dst[q] = *reinterpret_cast<const float4*>(&g.seg[(g.lane * Q + q) * 4]);
    __syncwarp();
  }
}
template <int E>
__device__ __forceinline__ void store_arr(const Geom<E>& g, float* arr, const float4* src) {
  constexpr int Q = E / 4;
  if (g.theta_vec) {
    if (g.live) {
#pragma unroll
      for (int q = 0; q < Q; ++q) st_state16(arr + g.e0 + g.unit * E + 4 * q, src[q]);
    }
  } else {
#pragma unroll
    for (int q = 0; q < Q; ++q) *reinterpret_cast<float4*>(&g.seg[(g.lane * Q + q) * 4]) = src[q];
    __syncwarp();
#pragma unroll
    for (int q = 0; q < E; ++q) {
      const int idx = q * 32 + g.lane;
      if (idx < g.live_in_seg) st_state32(arr + g.seg_e0 + idx, g.seg[idx]);
    }
    __syncwarp();
  }
}
template <int E, int OPT, int EMA>
__device__ __forceinline__ void load_state(const Geom<E>& g, const FusedParams& p, float4* th4, float4* em4, float4* a04,
                                           float4* a14) {
  load_arr<E>(g, p.theta, th4, 0.f);
  if (EMA != EMA_OFF) load_arr<E>(g, p.ema, em4, 0.f);
  if (OPT != OPT_SGD) load_arr<E>(g, p.s0, a04, 1.f);
  if (OPT == OPT_RMSPROP_MOM) load_arr<E>(g, p.s1, a14, 0.f);
}

template <bool BF16, int OPT, int EMA, bool SCALED, int D, int MINB>
__global__ void __launch_bounds__(kThreads, MINB) async_sharded_kernel(const FusedParams p) {
  constexpr int E = BF16 ? 8 : 4;
  constexpr int ESZ = BF16 ? 2 : 4;
  constexpr int Q = E / 4;
  __shared__ const char* s_ptr[kMaxWorkers];
  __shared__ float s_gamma[kMaxWorkers];
  __shared__ float s_scale[kMaxWorkers];
  __shared__ __align__(16) float s_seg[kThreads * E];
  __shared__ int64_t s_meta[4];  // off_j, len_j, h, tile: what Geom is derived from, re-read after the gradient loop
  __shared__ __align__(16) uint4 s_ring[D][kThreads];  // per-thread cp.async ring of arrivals on their way (as K4's)

  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  int K;
  bool mixed;
  {
    // ---- which (server, tile) is this CTA; its row of the order table ---------------------------------------
    // The prologue is a chain of dependent loads that every CTA pays before its first gradient byte moves, so it is
    // kept SHORT: the server by a warp-wide search (1-2 levels), then everything that only needs j in ONE level --
    // shard bounds, tile origin, status, count, this thread's entry of the order row and the row's first entry --
    // loaded before any of it is checked (all of these addresses are valid whatever the values turn out to be),
    // then the slice pointers in one more level.
    const int64_t b = blockIdx.x;
    const int64_t total = p.tile_start[p.M];
    const int j = upper_slot_warp(p.tile_start, p.M, b);
    const int row = p.per_shard ? j : 0;
    const int32_t* order = p.kept + static_cast<int64_t>(row) * p.kept_stride;
    const int64_t off_j = p.shard_off[j];
    const int64_t off_j1 = p.shard_off[j + 1];
    const int64_t tile0 = p.tile_start[j];
    const int st = p.status != nullptr ? p.status[row] : 0;
    K = p.n_kept != nullptr ? p.n_kept[row] : p.N;  // gradients that have reached server j
    const int k_first = order[0];
    const int i_mine = static_cast<int>(threadIdx.x) < p.kept_stride ? static_cast<int>(threadIdx.x) : p.kept_stride - 1;
    const int k_mine = order[i_mine];
    if (total != static_cast<int64_t>(gridDim.x)) return;  // a work list of another layout: touch nothing
    if (st != 0) return;                                   // this server applies nothing
    if (K <= 0 || K > p.kept_stride || K > kMaxWorkers) return;  // nothing arrived, or a count nobody wrote
    const int64_t len_j = off_j1 - off_j;
    const int64_t tile = b - tile0;

    // ---- stage server j's arrivals: slice base pointers, rates, clip factors; the first slice fixes the phase -
    auto slice_ptr = [&](int k) -> const char* {
      return p.slices ? static_cast<const char*>(p.grads[static_cast<int64_t>(k) * p.M + j])
                      : static_cast<const char*>(p.grads[k]) + off_j * ESZ;
    };
    const char* g_first = slice_ptr(k_first);
    const char* g_mine = static_cast<int>(threadIdx.x) < K ? slice_ptr(k_mine) : g_first;
    const unsigned ref = static_cast<unsigned>(reinterpret_cast<uintptr_t>(g_first)) & 127u;
    const int h = static_cast<int>(((128u - ref) & 127u) / ESZ);  // head peel: elements before the first 128-byte line
    unsigned mis = 0;
    for (int i = threadIdx.x; i < K; i += kThreads) {
      const int k = i < kThreads ? k_mine : order[i];
      const char* g = i < kThreads ? g_mine : slice_ptr(k);
      mis |= ((static_cast<unsigned>(reinterpret_cast<uintptr_t>(g)) ^ ref) & 15u);
      s_ptr[i] = g + h * ESZ;  // unit u of this arrival = s_ptr[i] + 16 u
      s_scale[i] = p.gscales ? p.gscales[k] : 1.0f;   // indexed by WORKER
      s_gamma[i] = p.gammas ? p.gammas[i] : p.gamma;  // rate of the server's i-th iteration of this batch
    }
    if (threadIdx.x == 0) {
      s_meta[0] = off_j;
      s_meta[1] = len_j;
      s_meta[2] = h;
      s_meta[3] = tile;
    }
    mixed = __syncthreads_or(static_cast<int>(mis)) != 0;
  }
  const volatile int64_t* meta = s_meta;

  float4 th4[Q], em4[Q], a04[Q], a14[Q];
  int64_t goff;  // byte offset of this thread's unit in every arrival's slice
  const uint32_t slot0 = static_cast<uint32_t>(__cvta_generic_to_shared(&s_ring[0][threadIdx.x]));
  {
    const Geom<E> g = make_geom<E>(meta[0], meta[1], static_cast<int>(meta[2]), meta[3], p.base_aligned, s_seg);
    if (g.u0 >= g.nu) goto peel;  // CTA-uniform: this tile holds no whole unit (a server shorter than its head)
    goff = g.unit * 16;
    // the first D arrivals are requested BEFORE the state: when theta is not co-aligned its loads are followed by a
    // trip through shared memory, and the gradient stream should not wait for that (one commit group per arrival)
    if (!mixed) {
#pragma unroll
      for (int i = 0; i < D; ++i) {
        if (i < K)
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(slot0 + i * kThreads * 16), "l"(s_ptr[i] + goff)
                       : "memory");
        asm volatile("cp.async.commit_group;" ::: "memory");
      }
    }
    load_state<E, OPT, EMA>(g, p, th4, em4, a04, a14);
  }
  {
    float2* th = reinterpret_cast<float2*>(th4);
    float2* em = reinterpret_cast<float2*>(em4);
    float2* a0 = reinterpret_cast<float2*>(a04);
    float2* a1 = reinterpret_cast<float2*>(a14);
    const PairCoeffs pc = make_pair_coeffs(p);

    unsigned bad = 0;  // RMSProp: did any ms + eps leave the range of the unchecked packed rsqrt?
    if (!mixed) {
      // K4's loop: wait for arrival i (groups retire in order), take it from its slot, apply it, refill the slot with
      // arrival i + D.  Every thread copies and consumes only its own slots: no barrier.
      auto one = [&](int i, int slot) {
        asm volatile("cp.async.wait_group %0;" ::"n"(D - 1) : "memory");
        const uint4 r = s_ring[slot][threadIdx.x];
        apply_unit<BF16, OPT, EMA, SCALED>(r, s_scale[i], s_gamma[i], th, em, a0, a1, pc, bad);
        if (i + D < K)
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(slot0 + slot * kThreads * 16),
                       "l"(s_ptr[i + D] + goff)
                       : "memory");
        asm volatile("cp.async.commit_group;" ::: "memory");
      };
      int i0 = 0;
      for (; i0 + D <= K; i0 += D) {
#pragma unroll
        for (int v = 0; v < D; ++v) one(i0 + v, v);
      }
      for (int i = i0; i < K; ++i) one(i, i - i0);
      asm volatile("cp.async.wait_group 0;" ::: "memory");
    } else {
#pragma unroll 2
      for (int i = 0; i < K; ++i) {
        const char* g = s_ptr[i];
        const uint4 r = load_unit_any<BF16>(g + goff, (reinterpret_cast<uintptr_t>(g) & 15u) == 0);
        apply_unit<BF16, OPT, EMA, SCALED>(r, s_scale[i], s_gamma[i], th, em, a0, a1, pc, bad);
      }
    }

    // ---- epilogue: the addresses are derived again (Geom's comment) -----------------------------------------
    const Geom<E> g = make_geom<E>(meta[0], meta[1], static_cast<int>(meta[2]), meta[3], p.base_aligned, s_seg);
    if (OPT == OPT_RMSPROP_MOM && __any_sync(0xFFFFFFFFu, rsqrt_pair_left_range(bad))) {
      // Never on sane data: a non-finite or absurd second moment somewhere in this warp.  Nothing has been stored
      // yet: the whole warp (the transposed loads are warp-collective) redoes its units from memory with the checked
      // scalar update, which gives the same bits wherever the packed form was in range.
      load_state<E, OPT, EMA>(g, p, th4, em4, a04, a14);
      float* ths = reinterpret_cast<float*>(th4);
      float* ems = reinterpret_cast<float*>(em4);
      float* a0s = reinterpret_cast<float*>(a04);
      float* a1s = reinterpret_cast<float*>(a14);
      for (int n = 0; n < K; ++n) {
        const char* gp = s_ptr[n];
        const uint4 r = load_unit_any<BF16>(gp + g.unit * 16, (reinterpret_cast<uintptr_t>(gp) & 15u) == 0);
#pragma unroll
        for (int e = 0; e < E; ++e)
          update_element_g<OPT, EMA>(unit_element<BF16>(r, e), s_scale[n], s_gamma[n], ths[e], ems[e], a0s[e], a1s[e], p);
      }
    }
    store_arr<E>(g, p.theta, th4);
    if (EMA != EMA_OFF) store_arr<E>(g, p.ema, em4);
    if (OPT != OPT_SGD) store_arr<E>(g, p.s0, a04);
    if (OPT == OPT_RMSPROP_MOM) store_arr<E>(g, p.s1, a14);
  }

peel:
  // ---- head and tail peel of server j, by its first CTA: K dependent updates per element, in registers --------
  if (meta[3] == 0) {
    const int64_t off_j = meta[0], len_j = meta[1];
    const int h = static_cast<int>(meta[2]);
    const int64_t nu = len_j > h ? (len_j - h) / E : 0;
    const int64_t tail0 = h + nu * E;
    const int64_t n_head = h < len_j ? h : len_j;
    const int64_t n_tail = len_j > tail0 ? len_j - tail0 : 0;
    if (threadIdx.x < n_head + n_tail) {
      const int64_t e = threadIdx.x < n_head ? threadIdx.x : tail0 + (threadIdx.x - n_head);
      const int64_t i = off_j + e;
      float th = p.theta[i];
      float em = (EMA != EMA_OFF) ? p.ema[i] : 0.f;
      float a0 = (OPT != OPT_SGD) ? p.s0[i] : 0.f;
      float a1 = (OPT == OPT_RMSPROP_MOM) ? p.s1[i] : 0.f;
      for (int n = 0; n < K; ++n)
        update_element_g<OPT, EMA>(load_grad_scalar<BF16>(s_ptr[n] - h * ESZ, e), s_scale[n], s_gamma[n], th, em, a0, a1, p);
      p.theta[i] = th;
      if (EMA != EMA_OFF) p.ema[i] = em;
      if (OPT != OPT_SGD) p.s0[i] = a0;
      if (OPT == OPT_RMSPROP_MOM) p.s1[i] = a1;
    }
  }
}

// ring depth and CTAs per SM (K4's ring shapes; bf16 has a 8 KB transpose buffer, so a shallower ring keeps the CTA
// within 48 KB of static shared memory)
struct Shape {
  int depth, minb;
};
constexpr Shape shape_for(bool bf16, int opt) {
  return bf16 ? (opt == OPT_RMSPROP_MOM ? Shape{4, 3} : Shape{4, 3}) : Shape{6, 4};
}

using KernelFn = void (*)(const FusedParams);

template <bool BF16, int OPT, int EMA>
KernelFn pick_scaled(bool scaled) {
  constexpr Shape S = shape_for(BF16, OPT);
  return scaled ? async_sharded_kernel<BF16, OPT, EMA, true, S.depth, S.minb>
                : async_sharded_kernel<BF16, OPT, EMA, false, S.depth, S.minb>;
}
template <bool BF16, int OPT>
KernelFn pick_ema(int ema, bool scaled) {
  switch (ema) {
    case EMA_POST: return pick_scaled<BF16, OPT, EMA_POST>(scaled);
    case EMA_PRE: return pick_scaled<BF16, OPT, EMA_PRE>(scaled);
    default: return pick_scaled<BF16, OPT, EMA_OFF>(scaled);
  }
}
template <bool BF16>
KernelFn pick_opt(int opt, int ema, bool scaled) {
  switch (opt) {
    case OPT_SGD: return pick_ema<BF16, OPT_SGD>(ema, scaled);
    case OPT_MOMENTUM: return pick_ema<BF16, OPT_MOMENTUM>(ema, scaled);
    default: return pick_ema<BF16, OPT_RMSPROP_MOM>(ema, scaled);
  }
}

}  // namespace

int async_sharded_smem_bytes(int dtype) {
  return static_cast<int>((sizeof(const char*) + 2 * sizeof(float)) * kMaxWorkers) + 4 * kThreads * (dtype == 1 ? 8 : 4);
}

cudaError_t launch_async_sharded(const FusedParams& p, int dtype, int opt, int ema, int64_t n_tiles, cudaStream_t stream) {
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
  const bool scaled = p.gscales != nullptr;
  return cudaLaunchKernelEx(&cfg, dtype == 1 ? pick_opt<true>(opt, ema, scaled) : pick_opt<false>(opt, ema, scaled), p);
}

}  // namespace psync
