// K4: the Async-SGD parameter server -- PAPER.md Algorithm 2 (L78-89), the paper's comparison method:
//
//     for t = 0, 1, ...:  wait for gradient G from any worker                       (L85)
//                         theta(t+1)[j] <- theta(t)[j] - gamma_t G[j]               (L86)
//                         ema(t)[j] = alpha ema(t-1)[j] + (1-alpha) theta(t)[j]     (L87)
//
// Every arriving gradient is one iteration.  K gradients that have arrived (K1c gives their order)
// are applied ONE AT A TIME, in that order, but in ONE pass over HBM: a thread loads its 16-byte
// unit of theta / state / ema once, walks the K gradient buffers in arrival order applying the
// optimizer step and the EMA after each one in registers, and stores once.  Per element the
// arithmetic is exactly K launches of the synchronous step with N=1, b=0 (bit-identical; tested),
// but the traffic is K*sizeof(grad) + 8*(1 + n_state + [EMA]) bytes per parameter instead of
// K*(sizeof(grad) + 8*(...)): 8.4x less for K=106 with RMSProp + EMA.
// Unlike the synchronous step the chain of K dependent updates is real arithmetic -- one optimizer
// update per gradient LOAD.  With SGD / momentum the kernel streams at the HBM roofline; with RMSProp
// it is bound by the FMA pipe (19 fp32 operations per element update at 128 lanes per clock per SM)
// about as much as by HBM.  What keeps it near both limits on B200: the update runs on PAIRS of
// elements with the packed fp32x2 instructions (FFMA2 / FMUL2: half the issue slots, same bits), the
// step is (gamma G) * rsqrt(ms + eps) with the correctly rounded rsqrt computed by an 8-operation
// refinement of MUFU.RSQ whose range check is a sticky flag outside the inner loop (psync_device.cuh),
// and the gradients of the next arrivals are on their way while the current one is applied.
// Two launch shapes of the same arithmetic (psync_step.variant in psync_async_apply; bit-identical, tested):
//   async_apply_ring_kernel  (0, default) the stream staged through a per-thread cp.async ring in shared memory
//   async_apply_kernel       (1) two register buffers, software-pipelined batches
//   (a third shape, 8-byte units -- one pair of parameters per thread -- measured 3.5 % slower on cfg3's shape,
//    profiles/r2_async.md, and was removed after round 2)

#include "async_common.cuh"

namespace psync {
namespace {

using namespace dev;

// PIPE: software-pipelined batches (below); SCALED: per-worker clip factors are applied (else they are all 1)
template <int THREADS, int U, int MINB, bool PIPE, bool BF16, int OPT, int EMA, bool SCALED>
__global__ void __launch_bounds__(THREADS, MINB) async_apply_kernel(const FusedParams p) {
  constexpr int E = BF16 ? 8 : 4;
  constexpr int Q = E / 4;
  __shared__ const char* s_ptr[kMaxWorkers];
  __shared__ float s_gamma[kMaxWorkers];
  __shared__ float s_scale[kMaxWorkers];  // global-norm clip factor of the i-th gradient (1 without clipping)

  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  if (p.status != nullptr && *p.status != 0) return;
  const int K = p.n_kept ? *p.n_kept : p.N;  // gradients that arrived
  if (K <= 0 || K > kMaxWorkers) return;  // nothing arrived, or a count nobody wrote

  unsigned misalign = 0;
  for (int i = threadIdx.x; i < K; i += THREADS) {
    const int k = p.kept[i];  // kept[] holds the arrival order
    const char* g = static_cast<const char*>(p.grads[k]);
    s_ptr[i] = g;
    s_scale[i] = p.gscales ? p.gscales[k] : 1.0f;  // indexed by WORKER (L313: each worker clips its own gradient)
    s_gamma[i] = p.gammas ? p.gammas[i] : p.gamma;  // gamma_t of iteration t+i
    misalign |= static_cast<unsigned>(reinterpret_cast<uintptr_t>(g)) & 15u;
  }
  const bool vec_ok = (__syncthreads_or(static_cast<int>(misalign)) == 0) && (p.base_aligned != 0);

  const PairCoeffs pc = make_pair_coeffs(p);
  const int64_t n_units = vec_ok ? p.P / E : 0;
  for (int64_t u = static_cast<int64_t>(blockIdx.x) * THREADS + threadIdx.x; u < n_units;
       u += static_cast<int64_t>(gridDim.x) * THREADS) {
    float4 th4[Q], em4[Q], a04[Q], a14[Q];
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      const int64_t e = u * E + 4 * q;
      th4[q] = ld_state16(p.theta + e);
      if (EMA != EMA_OFF) em4[q] = ld_state16(p.ema + e);
      if (OPT != OPT_SGD) a04[q] = ld_state16(p.s0 + e);
      if (OPT == OPT_RMSPROP_MOM) a14[q] = ld_state16(p.s1 + e);
    }
    float2* th = reinterpret_cast<float2*>(th4);
    float2* em = reinterpret_cast<float2*>(em4);
    float2* a0 = reinterpret_cast<float2*>(a04);
    float2* a1 = reinterpret_cast<float2*>(a14);

    unsigned bad = 0;  // RMSProp: did any ms + eps leave the range of the unchecked packed rsqrt?
    if (PIPE) {
      // Software-pipelined over batches of U gradients: the loads of batch b+1 are in flight while the U dependent
      // updates of batch b run (the updates are real arithmetic here -- with RMSProp the FMA pipe, not HBM, is the
      // limit -- so a warp that only started its next loads after its updates left both idle in turn).
      const int n_batches = K / U;
      uint4 cur[U], nxt[U];
      if (n_batches > 0) {
#pragma unroll
        for (int v = 0; v < U; ++v) cur[v] = ldg_stream16(s_ptr[v] + u * 16);
      }
      for (int b = 0; b < n_batches; ++b) {
        const int i = b * U;
        if (b + 1 < n_batches) {
#pragma unroll
          for (int v = 0; v < U; ++v) nxt[v] = ldg_stream16(s_ptr[i + U + v] + u * 16);
        }
#pragma unroll
        for (int v = 0; v < U; ++v)
          apply_unit<BF16, OPT, EMA, SCALED>(cur[v], s_scale[i + v], s_gamma[i + v], th, em, a0, a1, pc, bad);
#pragma unroll
        for (int v = 0; v < U; ++v) cur[v] = nxt[v];
      }
      for (int i = n_batches * U; i < K; ++i) {
        const uint4 r = ldg_stream16(s_ptr[i] + u * 16);
        apply_unit<BF16, OPT, EMA, SCALED>(r, s_scale[i], s_gamma[i], th, em, a0, a1, pc, bad);
      }
    } else {
      int i = 0;
      for (; i + U <= K; i += U) {  // U independent 16-byte loads in flight, then U dependent updates
        uint4 r[U];
#pragma unroll
        for (int v = 0; v < U; ++v) r[v] = ldg_stream16(s_ptr[i + v] + u * 16);
#pragma unroll
        for (int v = 0; v < U; ++v)
          apply_unit<BF16, OPT, EMA, SCALED>(r[v], s_scale[i + v], s_gamma[i + v], th, em, a0, a1, pc, bad);
      }
      for (; i < K; ++i) {
        const uint4 r = ldg_stream16(s_ptr[i] + u * 16);
        apply_unit<BF16, OPT, EMA, SCALED>(r, s_scale[i], s_gamma[i], th, em, a0, a1, pc, bad);
      }
    }
    if (OPT == OPT_RMSPROP_MOM && rsqrt_pair_left_range(bad)) {
      // Never on sane data: a non-finite or absurd second moment.  Nothing has been stored yet, so redo this unit from
      // memory with the checked scalar update (IEEE special values propagate as the definition says).
#pragma unroll
      for (int q = 0; q < Q; ++q) {
        const int64_t e = u * E + 4 * q;
        th4[q] = ld_state16(p.theta + e);
        if (EMA != EMA_OFF) em4[q] = ld_state16(p.ema + e);
        a04[q] = ld_state16(p.s0 + e);
        a14[q] = ld_state16(p.s1 + e);
      }
      float* ths = reinterpret_cast<float*>(th4);
      float* ems = reinterpret_cast<float*>(em4);
      float* a0s = reinterpret_cast<float*>(a04);
      float* a1s = reinterpret_cast<float*>(a14);
      for (int n = 0; n < K; ++n) {
        const uint4 r = ldg_stream16(s_ptr[n] + u * 16);
#pragma unroll
        for (int e = 0; e < E; ++e)
          update_element_g<OPT, EMA>(unit_element<BF16>(r, e), s_scale[n], s_gamma[n], ths[e], ems[e], a0s[e], a1s[e], p);
      }
    }

#pragma unroll
    for (int q = 0; q < Q; ++q) {
      const int64_t e = u * E + 4 * q;
      st_state16(p.theta + e, th4[q]);
      if (EMA != EMA_OFF) st_state16(p.ema + e, em4[q]);
      if (OPT != OPT_SGD) st_state16(p.s0 + e, a04[q]);
      if (OPT == OPT_RMSPROP_MOM) st_state16(p.s1 + e, a14[q]);
    }
  }

  // scalar path: the < E trailing parameters, or everything when a buffer is not 16-byte aligned
  const int64_t tail0 = n_units * E;
  const bool mine = vec_ok ? (blockIdx.x == 0) : true;
  if (tail0 < p.P && mine) {
    const int64_t first = vec_ok ? threadIdx.x : static_cast<int64_t>(blockIdx.x) * THREADS + threadIdx.x;
    const int64_t stride = vec_ok ? THREADS : static_cast<int64_t>(gridDim.x) * THREADS;
    for (int64_t e = tail0 + first; e < p.P; e += stride) {
      float th = p.theta[e];
      float em = (EMA != EMA_OFF) ? p.ema[e] : 0.f;
      float a0 = (OPT != OPT_SGD) ? p.s0[e] : 0.f;
      float a1 = (OPT == OPT_RMSPROP_MOM) ? p.s1[e] : 0.f;
      for (int i = 0; i < K; ++i)
        update_element_g<OPT, EMA>(load_grad_scalar<BF16>(s_ptr[i], e), s_scale[i], s_gamma[i], th, em, a0, a1, p);
      p.theta[e] = th;
      if (EMA != EMA_OFF) p.ema[e] = em;
      if (OPT != OPT_SGD) p.s0[e] = a0;
      if (OPT == OPT_RMSPROP_MOM) p.s1[e] = a1;
    }
  }
}

// K4 with the gradient stream staged through a per-thread ring in SHARED memory (cp.async, LDGSTS): the loads in flight
// live in shared memory instead of registers, so D arrivals per thread are on their way while one is applied, without the
// second register buffer of the pipelined form.  Every thread copies and consumes only its own 16-byte slots, so the only
// synchronisation is cp.async.wait_group -- no barrier.  The default of psync_async_apply (flat buffers,
// one order); bit-identical to the register-pipelined form.
template <int D, int MINB, bool BF16, int OPT, int EMA, bool SCALED>
__global__ void __launch_bounds__(256, MINB) async_apply_ring_kernel(const FusedParams p) {
  constexpr int THREADS = 256;
  constexpr int E = BF16 ? 8 : 4;
  constexpr int Q = E / 4;
  __shared__ const char* s_ptr[kMaxWorkers];
  __shared__ float s_gamma[kMaxWorkers];
  __shared__ float s_scale[kMaxWorkers];
  __shared__ __align__(16) uint4 s_ring[D][THREADS];

  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  if (p.status != nullptr && *p.status != 0) return;
  const int K = p.n_kept ? *p.n_kept : p.N;
  if (K <= 0 || K > kMaxWorkers) return;

  unsigned misalign = 0;
  for (int i = threadIdx.x; i < K; i += THREADS) {
    const int k = p.kept[i];
    const char* g = static_cast<const char*>(p.grads[k]);
    s_ptr[i] = g;
    s_scale[i] = p.gscales ? p.gscales[k] : 1.0f;
    s_gamma[i] = p.gammas ? p.gammas[i] : p.gamma;
    misalign |= static_cast<unsigned>(reinterpret_cast<uintptr_t>(g)) & 15u;
  }
  const bool vec_ok = (__syncthreads_or(static_cast<int>(misalign)) == 0) && (p.base_aligned != 0);

  const PairCoeffs pc = make_pair_coeffs(p);
  const int64_t n_units = vec_ok ? p.P / E : 0;
  const uint32_t slot0 = static_cast<uint32_t>(__cvta_generic_to_shared(&s_ring[0][threadIdx.x]));
  for (int64_t u = static_cast<int64_t>(blockIdx.x) * THREADS + threadIdx.x; u < n_units;
       u += static_cast<int64_t>(gridDim.x) * THREADS) {
    // D arrivals on their way before anything else (one commit group per arrival, empty past K)
#pragma unroll
    for (int i = 0; i < D; ++i) {
      if (i < K)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(slot0 + i * THREADS * 16), "l"(s_ptr[i] + u * 16)
                     : "memory");
      asm volatile("cp.async.commit_group;" ::: "memory");
    }
    float4 th4[Q], em4[Q], a04[Q], a14[Q];
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      const int64_t e = u * E + 4 * q;
      th4[q] = ld_state16(p.theta + e);
      if (EMA != EMA_OFF) em4[q] = ld_state16(p.ema + e);
      if (OPT != OPT_SGD) a04[q] = ld_state16(p.s0 + e);
      if (OPT == OPT_RMSPROP_MOM) a14[q] = ld_state16(p.s1 + e);
    }
    float2* th = reinterpret_cast<float2*>(th4);
    float2* em = reinterpret_cast<float2*>(em4);
    float2* a0 = reinterpret_cast<float2*>(a04);
    float2* a1 = reinterpret_cast<float2*>(a14);
    unsigned bad = 0;
    // one arrival: wait for it (groups retire in order), take it from its slot, apply it, refill the slot with
    // arrival i + D (the slot is free once its value has been consumed by the update)
    auto one = [&](int i, int slot) {
      asm volatile("cp.async.wait_group %0;" ::"n"(D - 1) : "memory");
      const uint4 r = s_ring[slot][threadIdx.x];
      apply_unit<BF16, OPT, EMA, SCALED>(r, s_scale[i], s_gamma[i], th, em, a0, a1, pc, bad);
      if (i + D < K)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(slot0 + slot * THREADS * 16),
                     "l"(s_ptr[i + D] + u * 16)
                     : "memory");
      asm volatile("cp.async.commit_group;" ::: "memory");
    };
    int i0 = 0;
    for (; i0 + D <= K; i0 += D) {  // unrolled over the ring: static slots
#pragma unroll
      for (int v = 0; v < D; ++v) one(i0 + v, v);
    }
    for (int i = i0; i < K; ++i) one(i, i - i0);
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    if (OPT == OPT_RMSPROP_MOM && rsqrt_pair_left_range(bad)) {  // redo from memory with the checked scalar update
#pragma unroll
      for (int q = 0; q < Q; ++q) {
        const int64_t e = u * E + 4 * q;
        th4[q] = ld_state16(p.theta + e);
        if (EMA != EMA_OFF) em4[q] = ld_state16(p.ema + e);
        a04[q] = ld_state16(p.s0 + e);
        a14[q] = ld_state16(p.s1 + e);
      }
      float* ths = reinterpret_cast<float*>(th4);
      float* ems = reinterpret_cast<float*>(em4);
      float* a0s = reinterpret_cast<float*>(a04);
      float* a1s = reinterpret_cast<float*>(a14);
      for (int n = 0; n < K; ++n) {
        const uint4 r = ldg_stream16(s_ptr[n] + u * 16);
#pragma unroll
        for (int e = 0; e < E; ++e)
          update_element_g<OPT, EMA>(unit_element<BF16>(r, e), s_scale[n], s_gamma[n], ths[e], ems[e], a0s[e], a1s[e], p);
      }
    }
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      const int64_t e = u * E + 4 * q;
      st_state16(p.theta + e, th4[q]);
      if (EMA != EMA_OFF) st_state16(p.ema + e, em4[q]);
      if (OPT != OPT_SGD) st_state16(p.s0 + e, a04[q]);
      if (OPT == OPT_RMSPROP_MOM) st_state16(p.s1 + e, a14[q]);
    }
  }

  const int64_t tail0 = n_units * E;
  const bool mine = vec_ok ? (blockIdx.x == 0) : true;
  if (tail0 < p.P && mine) {
    const int64_t first = vec_ok ? threadIdx.x : static_cast<int64_t>(blockIdx.x) * THREADS + threadIdx.x;
    const int64_t stride = vec_ok ? THREADS : static_cast<int64_t>(gridDim.x) * THREADS;
    for (int64_t e = tail0 + first; e < p.P; e += stride) {
      float th = p.theta[e];
      float em = (EMA != EMA_OFF) ? p.ema[e] : 0.f;
      float a0 = (OPT != OPT_SGD) ? p.s0[e] : 0.f;
      float a1 = (OPT == OPT_RMSPROP_MOM) ? p.s1[e] : 0.f;
      for (int i = 0; i < K; ++i)
        update_element_g<OPT, EMA>(load_grad_scalar<BF16>(s_ptr[i], e), s_scale[i], s_gamma[i], th, em, a0, a1, p);
      p.theta[e] = th;
      if (EMA != EMA_OFF) p.ema[e] = em;
      if (OPT != OPT_SGD) p.s0[e] = a0;
      if (OPT == OPT_RMSPROP_MOM) p.s1[e] = a1;
    }
  }
}

// K1c: rank sort of <= 1024 keys in one CTA.  Thread i owns worker i: its rank is the number of eligible
// workers that come before it in (arrival, index) order; -0.0 == +0.0; non-finite = never arrived.
// One CTA per row: row r of arrival [rows][W] is what parameter server r saw (Alg. 2 is the program of one server j).
__global__ void __launch_bounds__(1024) order_by_arrival_kernel(const float* arrival_rows, int32_t W,  // plain: written by a predecessor under PDL
                                                                int32_t* __restrict__ order_rows,
                                                                int32_t* __restrict__ n_arrived_rows) {
  __shared__ uint32_t s_key[kMaxWorkers];
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const float* arrival = arrival_rows + static_cast<int64_t>(blockIdx.x) * W;
  int32_t* order = order_rows + static_cast<int64_t>(blockIdx.x) * W;
  int32_t* n_arrived = n_arrived_rows + blockIdx.x;
  const int i = threadIdx.x;
  uint32_t key = 0xFFFFFFFFu;
  if (i < W) {
    uint32_t u = __float_as_uint(arrival[i]);
    if ((u & 0x7F800000u) != 0x7F800000u) {
      if (u == 0x80000000u) u = 0u;
      key = (u & 0x80000000u) ? ~u : (u | 0x80000000u);  // order-preserving; never 0xFFFFFFFF for finite input
    }
    s_key[i] = key;
  }
  const int n = __syncthreads_count(key != 0xFFFFFFFFu);
  if (key != 0xFFFFFFFFu) {
    int rank = 0;
    for (int j = 0; j < W; ++j) {
      const uint32_t kj = s_key[j];
      rank += (kj < key || (kj == key && j < i)) ? 1 : 0;
    }
    order[rank] = i;
  }
  if (i == 0) *n_arrived = n;
}

struct AsyncShape {
  int threads, unroll, minb;
  bool pipe;
};
// {threads, gradients per batch, CTAs per SM, software-pipelined}, measured on B200 (profiles/r2_async.md).  fp32: two
// batches live (one applied, one in flight), 64 registers, 4 CTAs/SM; for RMSProp (FMA-pipe-bound) batches of 3 were the
// best of nine shapes (cfg3 shape: 1.83 ms; batches of 2: 1.95, 4 at 3 CTAs/SM: 2.13, 8 unpipelined: 2.23).  bf16 holds
// 8 parameters per thread: one batch of 8 loads, 3 CTAs/SM (RMSProp: pipelined short batches, 2 CTAs/SM).
constexpr AsyncShape shape_for(bool bf16, int opt) {
  return bf16 ? (opt == OPT_RMSPROP_MOM ? AsyncShape{256, 2, 2, true} : AsyncShape{256, 8, 3, false})
              : (opt == OPT_RMSPROP_MOM ? AsyncShape{256, 3, 4, true} : AsyncShape{256, 4, 4, true});
}

using KernelFn = void (*)(const FusedParams);

template <bool BF16, int OPT, int EMA>
KernelFn pick_scaled(bool scaled) {
  constexpr AsyncShape S = shape_for(BF16, OPT);
  return scaled ? async_apply_kernel<S.threads, S.unroll, S.minb, S.pipe, BF16, OPT, EMA, true>
                : async_apply_kernel<S.threads, S.unroll, S.minb, S.pipe, BF16, OPT, EMA, false>;
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

cudaError_t async_geometry(int dtype, int grid_ctas, int64_t P, FusedGeometry* out) {
  const AsyncShape s = shape_for(dtype == 1, OPT_SGD);  // every shape has 256 threads: the grid does not depend on opt
  const int E = dtype == 1 ? 8 : 4;
  out->block = s.threads;
  out->tile_elems = s.threads * E;
  out->smem_bytes = static_cast<int>((sizeof(const char*) + 2 * sizeof(float)) * kMaxWorkers);
  int64_t grid = grid_ctas > 0 ? grid_ctas : (P / E + s.threads - 1) / s.threads;  // one unit per thread
  if (grid > 0x7FFFFFFF) grid = 0x7FFFFFFF;
  if (grid < 1) grid = 1;
  out->grid = static_cast<int>(grid);
  return cudaSuccess;
}

// the shared-memory ring (cp.async): {ring depth, CTAs per SM}.  Depth 4 / 6 / 8 are within 1 % of one another on
// every shape (cfg3's: 1.769 / 1.753 / 1.759 ms), 5 or 6 CTAs/SM are slower (profiles/r2_async.md).
struct RingShape {
  int depth, minb;
};
#ifndef PSYNC_RING_BF16_MINB
#define PSYNC_RING_BF16_MINB 3
#endif
constexpr RingShape ring_shape_for(bool bf16, int opt) {
  return bf16 ? (opt == OPT_RMSPROP_MOM ? RingShape{6, 3} : RingShape{6, PSYNC_RING_BF16_MINB}) : RingShape{6, 4};
}
template <bool BF16, int OPT, int EMA>
KernelFn pick_ring_scaled(bool scaled) {
  constexpr RingShape S = ring_shape_for(BF16, OPT);
  return scaled ? async_apply_ring_kernel<S.depth, S.minb, BF16, OPT, EMA, true>
                : async_apply_ring_kernel<S.depth, S.minb, BF16, OPT, EMA, false>;
}
template <bool BF16, int OPT>
KernelFn pick_ring_ema(int ema, bool scaled) {
  switch (ema) {
    case EMA_POST: return pick_ring_scaled<BF16, OPT, EMA_POST>(scaled);
    case EMA_PRE: return pick_ring_scaled<BF16, OPT, EMA_PRE>(scaled);
    default: return pick_ring_scaled<BF16, OPT, EMA_OFF>(scaled);
  }
}
template <bool BF16>
KernelFn pick_ring(int opt, int ema, bool scaled) {
  switch (opt) {
    case OPT_SGD: return pick_ring_ema<BF16, OPT_SGD>(ema, scaled);
    case OPT_MOMENTUM: return pick_ring_ema<BF16, OPT_MOMENTUM>(ema, scaled);
    default: return pick_ring_ema<BF16, OPT_RMSPROP_MOM>(ema, scaled);
  }
}

cudaError_t launch_async_apply_ring(const FusedParams& p, int dtype, int opt, int ema, int grid_ctas, cudaStream_t stream) {
  FusedGeometry g;
  async_geometry(dtype, grid_ctas, p.P, &g);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(static_cast<unsigned>(g.grid));
  cfg.blockDim = dim3(256);
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  const bool scaled = p.gscales != nullptr;
  return cudaLaunchKernelEx(&cfg, dtype == 1 ? pick_ring<true>(opt, ema, scaled) : pick_ring<false>(opt, ema, scaled), p);
}

cudaError_t launch_async_apply(const FusedParams& p, int dtype, int opt, int ema, int grid_ctas, cudaStream_t stream) {
  FusedGeometry g;
  async_geometry(dtype, grid_ctas, p.P, &g);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(static_cast<unsigned>(g.grid));
  cfg.blockDim = dim3(static_cast<unsigned>(g.block));
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  const bool scaled = p.gscales != nullptr;
  return cudaLaunchKernelEx(&cfg, dtype == 1 ? pick_opt<true>(opt, ema, scaled) : pick_opt<false>(opt, ema, scaled), p);
}

cudaError_t launch_order_by_arrival(const float* d_arrival, int32_t W, int32_t rows, int32_t* d_order,
                                    int32_t* d_n_arrived, cudaStream_t stream) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(static_cast<unsigned>(rows));
  cfg.blockDim = dim3(static_cast<unsigned>((W + 31) / 32 * 32));
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, order_by_arrival_kernel, d_arrival, W, d_order, d_n_arrived);
}

}  // namespace psync
