// The C ABI of include/psync.h: argument checks, dispatch to the sm_100a kernels, and the
// host-buffer step (chunked, double-buffered H2D of the kept workers only).  No torch types, no
// CPU arithmetic path: every step of Alg. 4 runs in the kernels of this directory.

#include <cstring>
#include <vector>

#include "../../include/psync.h"
#include "psync_kernels.cuh"

namespace {

using psync::FusedParams;

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

int check_step(const psync_step* s, bool need_device_tables) {
  if (s == nullptr) return PSYNC_EINVAL;
  if (s->P < 0 || s->M < 1 || s->h_shard_off == nullptr) return PSYNC_EINVAL;
  if (s->h_shard_off[0] != 0 || s->h_shard_off[s->M] != s->P) return PSYNC_EINVAL;
  for (int32_t j = 0; j < s->M; ++j)
    if (s->h_shard_off[j + 1] < s->h_shard_off[j]) return PSYNC_EINVAL;
  if (s->N < 1 || s->W < s->N || s->W > PSYNC_MAX_WORKERS) return PSYNC_EINVAL;
  if (s->grad_dtype != PSYNC_F32 && s->grad_dtype != PSYNC_BF16) return PSYNC_EINVAL;
  if (s->opt < PSYNC_SGD || s->opt > PSYNC_RMSPROP_MOM) return PSYNC_EINVAL;
  if (s->ema_mode < PSYNC_EMA_POST || s->ema_mode > PSYNC_EMA_OFF) return PSYNC_EINVAL;
  if (s->P > 0) {  // an empty parameter vector needs no buffers
    if (s->d_theta == nullptr) return PSYNC_EINVAL;
    if (s->ema_mode != PSYNC_EMA_OFF && s->d_ema == nullptr) return PSYNC_EINVAL;
    if (s->opt != PSYNC_SGD && s->d_state0 == nullptr) return PSYNC_EINVAL;
    if (s->opt == PSYNC_RMSPROP_MOM && s->d_state1 == nullptr) return PSYNC_EINVAL;
  }
  if (need_device_tables && (s->d_grads == nullptr || s->d_kept == nullptr)) return PSYNC_EINVAL;
  if (s->grid_ctas < 0 || s->variant < 0 || s->variant > psync::fused_num_variants()) return PSYNC_EINVAL;
  if (s->per_shard != 0 && s->per_shard != 1) return PSYNC_EINVAL;
  if (s->kept_stride < 0 || (s->kept_stride != 0 && s->kept_stride < s->N && s->d_n_kept == nullptr)) return PSYNC_EINVAL;
  if (s->kept_stride > PSYNC_MAX_WORKERS) return PSYNC_EINVAL;
  if (need_device_tables && s->per_shard && s->d_shard_off == nullptr) return PSYNC_EINVAL;
  if (s->grad_layout != PSYNC_GRADS_FLAT && s->grad_layout != PSYNC_GRADS_SLICES) return PSYNC_EINVAL;
  if (need_device_tables && s->grad_layout == PSYNC_GRADS_SLICES && (s->d_shard_off == nullptr || s->d_tile_start == nullptr))
    return PSYNC_EINVAL;
  if ((s->per_shard || s->d_n_kept != nullptr || s->grad_layout == PSYNC_GRADS_SLICES) && s->variant > 1)
    return PSYNC_EUNSUPPORTED;  // rows / shard-aware kernels: default launch shape only
  if (!psync::fused_variant_exists(s->variant)) return PSYNC_EUNSUPPORTED;  // an id whose kernel was removed (2, 3, 4, 8)
  return PSYNC_OK;
}

// Coefficients formed in fp32 (reading R8); element range [first, first + count).
FusedParams make_params(const psync_step* s, int64_t first, int64_t count, const void* const* d_grads,
                        const int32_t* d_kept, const int32_t* d_status) {
  FusedParams p;
  p.P = count;
  p.N = s->N;
  p.grads = d_grads;
  p.kept = d_kept;
  p.status = d_status;
  p.theta = s->d_theta + first;
  p.ema = (s->ema_mode != PSYNC_EMA_OFF) ? s->d_ema + first : nullptr;
  p.s0 = (s->opt != PSYNC_SGD) ? s->d_state0 + first : nullptr;
  p.s1 = (s->opt == PSYNC_RMSPROP_MOM) ? s->d_state1 + first : nullptr;
  p.gamma = s->gamma_t;
  p.alpha = s->alpha;
  p.one_minus_alpha = 1.0f - s->alpha;
  p.mu = s->mu;
  p.rho = s->rho;
  p.one_minus_rho = 1.0f - s->rho;
  p.eps = s->eps;
  p.inv_N = 1.0f / static_cast<float>(s->N);
  p.per_shard = s->per_shard;
  p.kept_stride = s->kept_stride > 0 ? s->kept_stride : (s->d_n_kept != nullptr ? s->W : s->N);
  p.M = s->M;
  p.shard_off = s->d_shard_off;
  p.n_kept = s->d_n_kept;
  p.slices = s->grad_layout == PSYNC_GRADS_SLICES ? 1 : 0;
  p.tile_start = s->d_tile_start;
  p.gammas = nullptr;
  p.gscales = nullptr;
  p.base_aligned = aligned16(p.theta) && (p.ema == nullptr || aligned16(p.ema)) && (p.s0 == nullptr || aligned16(p.s0)) &&
                   (p.s1 == nullptr || aligned16(p.s1));
  return p;
}

// The shard-aware kernel (work list, one CTA per (server, tile)) serves the slices layout, and flat buffers with one
// kept row per server when the caller supplies the work list; everything else is the flat stream.
bool wants_sharded(const psync_step* s) {
  return s->grad_layout == PSYNC_GRADS_SLICES || (s->per_shard != 0 && s->d_tile_start != nullptr);
}

int64_t sharded_tiles(const psync_step* s) {
  const int64_t T = psync::sharded_tile_elems(s->grad_dtype);
  int64_t n = 0;
  for (int32_t j = 0; j < s->M; ++j) n += (s->h_shard_off[j + 1] - s->h_shard_off[j] + T - 1) / T;
  return n;
}

cudaError_t launch_step_kernel(const psync_step* s, const FusedParams& p, cudaStream_t stream) {
  if (wants_sharded(s)) return psync::launch_sharded(p, s->grad_dtype, s->opt, s->ema_mode, sharded_tiles(s), stream);
  return psync::launch_fused(p, s->grad_dtype, s->opt, s->ema_mode, s->variant, s->grid_ctas, stream);
}

constexpr int64_t kDefaultChunkElems = int64_t{1} << 20;

// The copy stream and the four events psync_step_host needs; created per call, or once by psync_host_ctx_create.
struct HostCtx {
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t copied[2] = {nullptr, nullptr};
  cudaEvent_t consumed[2] = {nullptr, nullptr};
};

void host_ctx_release(HostCtx* c) {
  if (c->copy_stream != nullptr) {
    cudaStreamSynchronize(c->copy_stream);
    cudaStreamDestroy(c->copy_stream);
    c->copy_stream = nullptr;
  }
  for (int i = 0; i < 2; ++i) {
    if (c->copied[i] != nullptr) cudaEventDestroy(c->copied[i]);
    if (c->consumed[i] != nullptr) cudaEventDestroy(c->consumed[i]);
    c->copied[i] = c->consumed[i] = nullptr;
  }
}

bool host_ctx_init(HostCtx* c) {
  if (cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess) return false;
  for (int i = 0; i < 2; ++i) {
    if (cudaEventCreateWithFlags(&c->copied[i], cudaEventDisableTiming) != cudaSuccess) return false;
    if (cudaEventCreateWithFlags(&c->consumed[i], cudaEventDisableTiming) != cudaSuccess) return false;
  }
  return true;
}

int64_t round_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

struct HostLayout {
  int64_t chunk, stride_bytes;
  size_t off_stage[2], off_ptrs[2], off_ident, off_arrival, off_tags, off_kept, off_tnth, off_status, total;
};

bool host_layout(int32_t N, int32_t W, int32_t dtype, int64_t chunk_elems, HostLayout* L) {
  if (N < 1 || W < N || W > PSYNC_MAX_WORKERS) return false;
  if (dtype != PSYNC_F32 && dtype != PSYNC_BF16) return false;
  if (chunk_elems == 0) chunk_elems = kDefaultChunkElems;
  if (chunk_elems < 64 || chunk_elems % 64 != 0) return false;
  const int64_t esz = dtype == PSYNC_BF16 ? 2 : 4;
  L->chunk = chunk_elems;
  L->stride_bytes = round_up(chunk_elems * esz, 256);
  size_t off = 0;
  for (int i = 0; i < 2; ++i) {
    L->off_stage[i] = off;
    off += static_cast<size_t>(L->stride_bytes) * N;
  }
  for (int i = 0; i < 2; ++i) {
    L->off_ptrs[i] = off;
    off += static_cast<size_t>(round_up(int64_t{8} * N, 256));
  }
  L->off_ident = off;
  off += static_cast<size_t>(round_up(int64_t{4} * N, 256));
  L->off_arrival = off;
  off += static_cast<size_t>(round_up(int64_t{4} * W, 256));
  L->off_tags = off;
  off += static_cast<size_t>(round_up(int64_t{4} * W, 256));
  L->off_kept = off;
  off += static_cast<size_t>(round_up(int64_t{4} * N, 256));
  L->off_tnth = off;
  off += 256;
  L->off_status = off;
  off += 256;
  L->total = off;
  return true;
}

}  // namespace

extern "C" {

PSYNC_API int psync_version(void) { return PSYNC_VERSION; }

PSYNC_API const char* psync_status_string(int status) {
  switch (status) {
    case PSYNC_OK: return "PSYNC_OK";
    case PSYNC_EINVAL: return "PSYNC_EINVAL: invalid argument";
    case PSYNC_ETOOFEW: return "PSYNC_ETOOFEW: fewer than N eligible workers";
    case PSYNC_EUNSUPPORTED: return "PSYNC_EUNSUPPORTED";
    case PSYNC_ECUDA: return "PSYNC_ECUDA: CUDA runtime error";
    default: return "PSYNC: unknown status";
  }
}

PSYNC_API int psync_select_first_n(const float* d_arrival, const int32_t* d_step_tag, int32_t t, int32_t N, int32_t b,
                         int32_t* d_kept, float* d_t_nth, int32_t* d_status, void* stream) {
  if (d_arrival == nullptr || d_kept == nullptr || d_status == nullptr) return PSYNC_EINVAL;
  if (N < 1 || b < 0 || static_cast<int64_t>(N) + b > PSYNC_MAX_WORKERS) return PSYNC_EINVAL;
  const cudaError_t err = psync::launch_select_first_n(d_arrival, d_step_tag, t, N, N + b, 1, d_kept, d_t_nth, d_status,
                                                       static_cast<cudaStream_t>(stream));
  return err == cudaSuccess ? PSYNC_OK : PSYNC_ECUDA;
}

PSYNC_API int psync_select_first_n_sharded(const float* d_arrival, const int32_t* d_step_tag, int32_t t, int32_t N,
                                 int32_t b, int32_t M, int32_t* d_kept, float* d_t_nth, int32_t* d_status,
                                 void* stream) {
  if (d_arrival == nullptr || d_kept == nullptr || d_status == nullptr) return PSYNC_EINVAL;
  if (N < 1 || b < 0 || M < 1 || static_cast<int64_t>(N) + b > PSYNC_MAX_WORKERS) return PSYNC_EINVAL;
  const cudaError_t err = psync::launch_select_first_n(d_arrival, d_step_tag, t, N, N + b, M, d_kept, d_t_nth, d_status,
                                                       static_cast<cudaStream_t>(stream));
  return err == cudaSuccess ? PSYNC_OK : PSYNC_ECUDA;
}

PSYNC_API int psync_select_timeout(const float* d_arrival, const int32_t* d_step_tag, int32_t t, int32_t W,
                         int32_t rows, float timeout, int32_t min_keep, int32_t* d_kept, int32_t* d_n_kept,
                         int32_t* d_status, void* stream) {
  if (d_arrival == nullptr || d_kept == nullptr || d_n_kept == nullptr || d_status == nullptr) return PSYNC_EINVAL;
  if (W < 1 || W > PSYNC_MAX_WORKERS || rows < 1 || min_keep < 1 || timeout != timeout) return PSYNC_EINVAL;
  const cudaError_t err = psync::launch_select_timeout(d_arrival, d_step_tag, t, W, rows, timeout, min_keep, d_kept,
                                                       d_n_kept, d_status, static_cast<cudaStream_t>(stream));
  return err == cudaSuccess ? PSYNC_OK : PSYNC_ECUDA;
}

PSYNC_API int psync_aggregate_update(const psync_step* step, void* stream) {
  const int st = check_step(step, true);
  if (st != PSYNC_OK) return st;
  if (step->P == 0) return PSYNC_OK;
  const FusedParams p = make_params(step, 0, step->P, step->d_grads, step->d_kept, step->d_status);
  const cudaError_t err = launch_step_kernel(step, p, static_cast<cudaStream_t>(stream));
  return err == cudaSuccess ? PSYNC_OK : PSYNC_ECUDA;
}

PSYNC_API int psync_shard_worklist(const int64_t* d_shard_off, int32_t M, int32_t grad_dtype, int64_t* d_tile_start,
                         void* stream) {
  if (d_shard_off == nullptr || d_tile_start == nullptr || M < 1) return PSYNC_EINVAL;
  if (grad_dtype != PSYNC_F32 && grad_dtype != PSYNC_BF16) return PSYNC_EINVAL;
  return psync::launch_shard_worklist(d_shard_off, M, grad_dtype, d_tile_start, static_cast<cudaStream_t>(stream)) ==
                 cudaSuccess
             ? PSYNC_OK
             : PSYNC_ECUDA;
}

PSYNC_API int psync_step_device(const psync_step* step, const float* d_arrival, const int32_t* d_step_tag, int32_t t,
                      float* d_t_nth, void* stream) {
  const int st = check_step(step, true);
  if (st != PSYNC_OK) return st;
  if (d_arrival == nullptr || step->d_status == nullptr || step->d_n_kept != nullptr) return PSYNC_EINVAL;
  if (step->kept_stride != 0 && step->kept_stride != step->N) return PSYNC_EINVAL;  // the selection writes rows of N
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int32_t rows = step->per_shard ? step->M : 1;
  if (psync::launch_select_first_n(d_arrival, d_step_tag, t, step->N, step->W, rows, const_cast<int32_t*>(step->d_kept),
                                   d_t_nth, const_cast<int32_t*>(step->d_status), s) != cudaSuccess)
    return PSYNC_ECUDA;
  if (step->P == 0) return PSYNC_OK;
  const FusedParams p = make_params(step, 0, step->P, step->d_grads, step->d_kept, step->d_status);
  return launch_step_kernel(step, p, s) == cudaSuccess ? PSYNC_OK : PSYNC_ECUDA;
}

PSYNC_API int psync_order_by_arrival(const float* d_arrival, int32_t W, int32_t* d_order, int32_t* d_n_arrived,
                           void* stream) {
  if (d_arrival == nullptr || d_order == nullptr || d_n_arrived == nullptr) return PSYNC_EINVAL;
  if (W < 1 || W > PSYNC_MAX_WORKERS) return PSYNC_EINVAL;
  return psync::launch_order_by_arrival(d_arrival, W, 1, d_order, d_n_arrived, static_cast<cudaStream_t>(stream)) ==
                 cudaSuccess
             ? PSYNC_OK
             : PSYNC_ECUDA;
}

PSYNC_API int psync_order_by_arrival_sharded(const float* d_arrival, int32_t W, int32_t M, int32_t* d_order,
                                   int32_t* d_n_arrived, void* stream) {
  if (d_arrival == nullptr || d_order == nullptr || d_n_arrived == nullptr) return PSYNC_EINVAL;
  if (W < 1 || W > PSYNC_MAX_WORKERS || M < 1) return PSYNC_EINVAL;
  return psync::launch_order_by_arrival(d_arrival, W, M, d_order, d_n_arrived, static_cast<cudaStream_t>(stream)) ==
                 cudaSuccess
             ? PSYNC_OK
             : PSYNC_ECUDA;
}

PSYNC_API int psync_async_apply(const psync_step* step, const float* d_gamma, const float* d_gscale, void* stream) {
  if (step == nullptr) return PSYNC_EINVAL;
  psync_step s = *step;
  // launch shapes of the flat single-order kernel: 0 the shared-memory ring (default), 1 the register-pipelined form.
  // Everything else is refused: the work-list kernel (per server / slices) has one shape, the 8-byte-unit shape (2)
  // was removed after round 2 (measured slower, profiles/r2_async.md).
  const bool flat_one_order = step->per_shard == 0 && step->grad_layout == PSYNC_GRADS_FLAT;
  if (step->variant < 0) return PSYNC_EINVAL;
  if (step->variant > (flat_one_order ? 1 : 0)) return PSYNC_EUNSUPPORTED;
  const bool ring_shape = step->variant == 0 && flat_one_order;
  s.variant = 0;
  const int st = check_step(&s, true);
  if (st != PSYNC_OK) return st;
  // Alg. 2 per server (one order row per server) walks the (server, tile) work list like the slices layout does
  if (s.per_shard != 0 && s.d_tile_start == nullptr) return PSYNC_EUNSUPPORTED;  // no flat-index rows form of Alg. 2
  if (s.P == 0) return PSYNC_OK;
  FusedParams p = make_params(&s, 0, s.P, s.d_grads, s.d_kept, s.d_status);
  p.gammas = d_gamma;
  p.gscales = d_gscale;
  const cudaError_t err =
      ring_shape ? psync::launch_async_apply_ring(p, s.grad_dtype, s.opt, s.ema_mode, s.grid_ctas, static_cast<cudaStream_t>(stream)) :
      wants_sharded(&s) ? psync::launch_async_sharded(p, s.grad_dtype, s.opt, s.ema_mode, sharded_tiles(&s),
                                                      static_cast<cudaStream_t>(stream))
                        : psync::launch_async_apply(p, s.grad_dtype, s.opt, s.ema_mode, s.grid_ctas,
                                                    static_cast<cudaStream_t>(stream));
  return err == cudaSuccess ? PSYNC_OK : PSYNC_ECUDA;
}

PSYNC_API int psync_async_step_device(const psync_step* step, const float* d_arrival, const float* d_gamma,
                            const float* d_gscale, void* stream) {
  if (step == nullptr || d_arrival == nullptr) return PSYNC_EINVAL;
  if (step->d_kept == nullptr || step->d_n_kept == nullptr) return PSYNC_EINVAL;  // the order kernel's outputs
  if (step->W < 1 || step->W > PSYNC_MAX_WORKERS || step->M < 1) return PSYNC_EINVAL;
  if (step->kept_stride != 0 && step->kept_stride != step->W) return PSYNC_EINVAL;  // the order kernel writes rows of W
  psync_step s = *step;
  s.kept_stride = s.W;
  s.N = s.W;  // the count comes from the device (d_n_kept); N only has to satisfy 1 <= N <= W
  const int32_t rows = s.per_shard ? s.M : 1;
  if (psync::launch_order_by_arrival(d_arrival, s.W, rows, const_cast<int32_t*>(s.d_kept),
                                     const_cast<int32_t*>(s.d_n_kept), static_cast<cudaStream_t>(stream)) != cudaSuccess)
    return PSYNC_ECUDA;
  return psync_async_apply(&s, d_gamma, d_gscale, stream);
}

PSYNC_API size_t psync_clip_workspace_bytes(int32_t W, int64_t P, int32_t grad_dtype) {
  if (W < 1 || W > PSYNC_MAX_WORKERS || P < 0 || (grad_dtype != PSYNC_F32 && grad_dtype != PSYNC_BF16)) return 0;
  return psync::clip_workspace_bytes(W, P, grad_dtype);
}

PSYNC_API int psync_clip_scales(const void* const* d_grads, int32_t W, int64_t P, int32_t grad_dtype, float clip,
                      float* d_scales, void* d_work, size_t work_bytes, void* stream) {
  if (d_grads == nullptr || d_scales == nullptr || d_work == nullptr) return PSYNC_EINVAL;
  if (W < 1 || W > PSYNC_MAX_WORKERS || P < 0 || !(clip > 0.0f)) return PSYNC_EINVAL;
  if (grad_dtype != PSYNC_F32 && grad_dtype != PSYNC_BF16) return PSYNC_EINVAL;
  if (work_bytes < psync::clip_workspace_bytes(W, P, grad_dtype) || (reinterpret_cast<uintptr_t>(d_work) & 7u) != 0)
    return PSYNC_EINVAL;
  return psync::launch_clip_scales(d_grads, W, P, grad_dtype, clip, d_scales, d_work, static_cast<cudaStream_t>(stream)) ==
                 cudaSuccess
             ? PSYNC_OK
             : PSYNC_ECUDA;
}

namespace {
// sum_j ceil(len_j / chunk) for a valid host shard table, -1 otherwise
int64_t clip_slice_chunks(int32_t M, const int64_t* h_shard_off, int32_t grad_dtype) {
  if (M < 1 || h_shard_off == nullptr || h_shard_off[0] != 0) return -1;
  if (grad_dtype != PSYNC_F32 && grad_dtype != PSYNC_BF16) return -1;
  const int64_t ce = psync::clip_chunk_elems(grad_dtype);
  int64_t n = 0;
  for (int32_t j = 0; j < M; ++j) {
    const int64_t len = h_shard_off[j + 1] - h_shard_off[j];
    if (len < 0) return -1;
    n += (len + ce - 1) / ce;
  }
  return n;
}
}  // namespace

PSYNC_API size_t psync_clip_slices_workspace_bytes(int32_t W, int32_t M, const int64_t* h_shard_off, int32_t grad_dtype) {
  const int64_t n = clip_slice_chunks(M, h_shard_off, grad_dtype);
  if (W < 1 || W > PSYNC_MAX_WORKERS || n < 0) return 0;
  return psync::clip_slices_workspace_bytes(W, M, n);
}

PSYNC_API int psync_clip_scales_slices(const void* const* d_grads, int32_t W, int32_t M, const int64_t* h_shard_off,
                             const int64_t* d_shard_off, int32_t grad_dtype, float clip, float* d_scales, void* d_work,
                             size_t work_bytes, void* stream) {
  if (d_grads == nullptr || d_shard_off == nullptr || d_scales == nullptr || d_work == nullptr) return PSYNC_EINVAL;
  if (W < 1 || W > PSYNC_MAX_WORKERS || !(clip > 0.0f)) return PSYNC_EINVAL;
  const int64_t n = clip_slice_chunks(M, h_shard_off, grad_dtype);
  if (n < 0) return PSYNC_EINVAL;
  if (work_bytes < psync::clip_slices_workspace_bytes(W, M, n) || (reinterpret_cast<uintptr_t>(d_work) & 7u) != 0)
    return PSYNC_EINVAL;
  return psync::launch_clip_scales_slices(d_grads, W, M, d_shard_off, n, grad_dtype, clip, d_scales, d_work,
                                          static_cast<cudaStream_t>(stream)) == cudaSuccess
             ? PSYNC_OK
             : PSYNC_ECUDA;
}

PSYNC_API int psync_kth_arrival_stats(const float* d_arrival, int32_t T, int32_t W, float* d_sorted, int32_t* d_count,
                            double* d_mean, double* d_median, const double* d_iters, double* d_est_time, void* stream) {
  if (d_arrival == nullptr || d_sorted == nullptr || d_count == nullptr || d_mean == nullptr || d_median == nullptr)
    return PSYNC_EINVAL;
  if (T < 1 || W < 1 || W > PSYNC_MAX_WORKERS || (d_iters == nullptr) != (d_est_time == nullptr)) return PSYNC_EINVAL;
  return psync::launch_kth_arrival_stats(d_arrival, T, W, d_sorted, d_count, d_mean, d_median, d_iters, d_est_time,
                                         static_cast<cudaStream_t>(stream)) == cudaSuccess
             ? PSYNC_OK
             : PSYNC_ECUDA;
}

PSYNC_API int psync_interp_iterations(const int32_t* h_N, const double* h_iters, int32_t n_pts, int32_t W,
                            double* d_iters, void* stream) {
  if (h_N == nullptr || h_iters == nullptr || d_iters == nullptr) return PSYNC_EINVAL;
  if (n_pts < 1 || n_pts > psync::kMaxInterpPoints || W < 1 || W > PSYNC_MAX_WORKERS) return PSYNC_EINVAL;
  psync::InterpPoints pts;
  pts.n = n_pts;
  for (int32_t p = 0; p < psync::kMaxInterpPoints; ++p) {
    pts.N[p] = p < n_pts ? h_N[p] : 0;
    pts.iters[p] = p < n_pts ? h_iters[p] : 0.0;
    if (p > 0 && p < n_pts && h_N[p] <= h_N[p - 1]) return PSYNC_EINVAL;
  }
  return psync::launch_interp_iterations(pts, W, d_iters, static_cast<cudaStream_t>(stream)) == cudaSuccess ? PSYNC_OK
                                                                                                          : PSYNC_ECUDA;
}

PSYNC_API int psync_staleness(int64_t* d_read_iter, int32_t W, const int32_t* d_order, const int32_t* d_n_arrived,
                    int32_t K, int64_t* d_t, int32_t lag, int64_t* d_staleness, double* d_stats, int32_t* d_status,
                    void* stream) {
  if (d_read_iter == nullptr || d_order == nullptr || d_t == nullptr || d_staleness == nullptr || d_stats == nullptr ||
      d_status == nullptr)
    return PSYNC_EINVAL;
  if (W < 1 || W > PSYNC_MAX_WORKERS || K < 0 || K > W || lag < 0) return PSYNC_EINVAL;
  return psync::launch_staleness(d_read_iter, W, 1, d_order, d_n_arrived, K, d_t, lag, d_staleness, d_stats, d_status,
                                 static_cast<cudaStream_t>(stream)) == cudaSuccess
             ? PSYNC_OK
             : PSYNC_ECUDA;
}

PSYNC_API int psync_staleness_sharded(int64_t* d_read_iter, int32_t W, int32_t M, const int32_t* d_order,
                            const int32_t* d_n_arrived, int32_t K, int64_t* d_t, int32_t lag, int64_t* d_staleness,
                            double* d_stats, int32_t* d_status, void* stream) {
  if (d_read_iter == nullptr || d_order == nullptr || d_t == nullptr || d_staleness == nullptr || d_stats == nullptr ||
      d_status == nullptr)
    return PSYNC_EINVAL;
  if (W < 1 || W > PSYNC_MAX_WORKERS || M < 1 || K < 0 || K > W || lag < 0) return PSYNC_EINVAL;
  return psync::launch_staleness(d_read_iter, W, M, d_order, d_n_arrived, K, d_t, lag, d_staleness, d_stats, d_status,
                                 static_cast<cudaStream_t>(stream)) == cudaSuccess
             ? PSYNC_OK
             : PSYNC_ECUDA;
}

PSYNC_API int psync_lr_schedule(float gamma0, float beta, int64_t t0, int32_t K, double s, float* d_gamma, void* stream) {
  if (K < 0 || t0 < 0 || !(beta > 0.0f) || (K > 0 && d_gamma == nullptr)) return PSYNC_EINVAL;
  if (K == 0) return PSYNC_OK;
  return psync::launch_lr_schedule(gamma0, beta, t0, K, s, d_gamma, static_cast<cudaStream_t>(stream)) == cudaSuccess
             ? PSYNC_OK
             : PSYNC_ECUDA;
}

PSYNC_API int psync_lr_schedule_counted(float gamma0, float beta, int64_t* d_t, int64_t t_set, const int32_t* d_n_add,
                                        int32_t rows, int32_t K, double s, float* d_gamma, void* stream) {
  if (d_t == nullptr || K < 0 || K > PSYNC_MAX_WORKERS || !(beta > 0.0f) || (K > 0 && d_gamma == nullptr)) return PSYNC_EINVAL;
  if (t_set < 0 && d_n_add != nullptr && rows < 1) return PSYNC_EINVAL;
  return psync::launch_lr_schedule_counted(gamma0, beta, d_t, t_set, d_n_add, rows, K, s, d_gamma,
                                           static_cast<cudaStream_t>(stream)) == cudaSuccess
             ? PSYNC_OK
             : PSYNC_ECUDA;
}

PSYNC_API int psync_ema(float* d_ema, const float* d_theta, int64_t P, float alpha, void* stream) {
  if (d_ema == nullptr || d_theta == nullptr || P < 0) return PSYNC_EINVAL;
  if (P == 0) return PSYNC_OK;
  const cudaError_t err = psync::launch_ema(d_ema, d_theta, P, alpha, static_cast<cudaStream_t>(stream));
  return err == cudaSuccess ? PSYNC_OK : PSYNC_ECUDA;
}

PSYNC_API int psync_launch_geometry(const psync_step* step, int32_t* grid, int32_t* block, int32_t* tile_elems,
                          int32_t* smem_bytes) {
  const int st = check_step(step, false);
  if (st != PSYNC_OK) return st;
  psync::FusedGeometry g;
  if (wants_sharded(step)) {
    const int64_t tiles = sharded_tiles(step);
    if (tiles > 0x7FFFFFFF) return PSYNC_ECUDA;
    g.grid = static_cast<int>(tiles);
    g.block = PSYNC_TILE_UNITS;
    g.tile_elems = psync::sharded_tile_elems(step->grad_dtype);
    g.smem_bytes = 8 * PSYNC_MAX_WORKERS + 4 * g.tile_elems + 4;
  } else if (psync::fused_geometry(step->grad_dtype, step->opt, step->ema_mode, step->variant, step->grid_ctas, step->P,
                                   &g) != cudaSuccess) {
    return PSYNC_ECUDA;
  }
  if (grid) *grid = g.grid;
  if (block) *block = g.block;
  if (tile_elems) *tile_elems = g.tile_elems;
  if (smem_bytes) *smem_bytes = g.smem_bytes;
  return PSYNC_OK;
}

PSYNC_API int psync_probe_read(const void* d_src, int64_t n_vec16, float* d_sink, void* stream) {
  if (d_src == nullptr || d_sink == nullptr || n_vec16 < 0 || !aligned16(d_src)) return PSYNC_EINVAL;
  return psync::launch_probe_read(d_src, n_vec16, d_sink, static_cast<cudaStream_t>(stream)) == cudaSuccess ? PSYNC_OK
                                                                                                             : PSYNC_ECUDA;
}

PSYNC_API int psync_probe_copy(void* d_dst, const void* d_src, int64_t n_vec16, void* stream) {
  if (d_src == nullptr || d_dst == nullptr || n_vec16 < 0 || !aligned16(d_src) || !aligned16(d_dst)) return PSYNC_EINVAL;
  return psync::launch_probe_copy(d_dst, d_src, n_vec16, static_cast<cudaStream_t>(stream)) == cudaSuccess ? PSYNC_OK
                                                                                                            : PSYNC_ECUDA;
}

PSYNC_API int psync_probe_pipe(int32_t mode, int64_t iters, float* d_sink, int64_t* h_lane_ops, void* stream) {
  if (mode < 0 || mode > 2 || iters < 1 || d_sink == nullptr) return PSYNC_EINVAL;
  int ctas = 0;
  if (psync::launch_probe_pipe(mode, iters, d_sink, &ctas, static_cast<cudaStream_t>(stream)) != cudaSuccess)
    return PSYNC_ECUDA;
  if (h_lane_ops != nullptr) *h_lane_ops = static_cast<int64_t>(ctas) * 256 * 8 * iters * (mode == 1 ? 2 : 1);
  return PSYNC_OK;
}

PSYNC_API int psync_selftest_rsqrt(const float* d_x, uint32_t first_bits, int64_t n, float* d_y,
                         unsigned long long* d_mismatch, void* stream) {
  if (n < 0 || d_mismatch == nullptr) return PSYNC_EINVAL;
  return psync::launch_selftest_rsqrt(d_x, first_bits, n, d_y, d_mismatch, static_cast<cudaStream_t>(stream)) ==
                 cudaSuccess
             ? PSYNC_OK
             : PSYNC_ECUDA;
}

PSYNC_API size_t psync_step_host_workspace_bytes(int32_t N, int32_t W, int32_t grad_dtype, int64_t chunk_elems) {
  HostLayout L;
  if (!host_layout(N, W, grad_dtype, chunk_elems, &L)) return 0;
  return L.total;
}

PSYNC_API int psync_host_ctx_create(void** ctx) {
  if (ctx == nullptr) return PSYNC_EINVAL;
  HostCtx* c = new HostCtx();
  if (!host_ctx_init(c)) {
    host_ctx_release(c);
    delete c;
    cudaGetLastError();
    *ctx = nullptr;
    return PSYNC_ECUDA;
  }
  *ctx = c;
  return PSYNC_OK;
}

PSYNC_API int psync_host_ctx_destroy(void* ctx) {
  if (ctx == nullptr) return PSYNC_EINVAL;
  HostCtx* c = static_cast<HostCtx*>(ctx);
  host_ctx_release(c);
  delete c;
  return PSYNC_OK;
}

PSYNC_API int psync_step_host(const psync_step* st, const float* h_arrival, const int32_t* h_step_tag, int32_t t,
                    const void* const* h_grads, float* h_theta_out, int32_t* h_kept, float* h_t_nth, void* d_work,
                    size_t work_bytes, int64_t chunk_elems, void* stream) {
  return psync_step_host_ctx(nullptr, st, h_arrival, h_step_tag, t, h_grads, h_theta_out, h_kept, h_t_nth, d_work,
                             work_bytes, chunk_elems, stream);
}

}  // extern "C"

namespace {
// The host-buffer pipeline behind psync_step_host_ctx (Alg. 4: selection, then the N kept buffers) and
// psync_async_step_host (async_mode, Alg. 2: arrival order, then every buffer that arrived, applied one at a time by K4 on
// each staged chunk; h_kept receives the order, *h_n_arrived the count, h_gamma optional per-iteration rates).
int host_step_impl(void* ctx, const psync_step* st, const float* h_arrival, const int32_t* h_step_tag, int32_t t,
                   const void* const* h_grads, float* h_theta_out, int32_t* h_kept, float* h_t_nth, void* d_work,
                   size_t work_bytes, int64_t chunk_elems, void* stream, bool async_mode, const float* h_gamma,
                   int32_t* h_n_arrived) {
  if (st == nullptr) return PSYNC_EINVAL;
  psync_step flat = *st;  // the device side of this path is always the flat stream (see SLICES below)
  flat.grad_layout = PSYNC_GRADS_FLAT;
  flat.d_shard_off = nullptr;
  flat.d_tile_start = nullptr;
  const int chk = check_step(&flat, false);
  if (chk != PSYNC_OK) return chk;
  if (st->grad_layout != PSYNC_GRADS_FLAT && st->grad_layout != PSYNC_GRADS_SLICES) return PSYNC_EINVAL;
  if (h_arrival == nullptr || h_grads == nullptr || d_work == nullptr) return PSYNC_EINVAL;
  if (st->per_shard != 0 || st->d_n_kept != nullptr) return PSYNC_EUNSUPPORTED;
  // SLICES: h_grads is [W*M] HOST pointers, entry k*M + j -> the len_j elements of G_k[j] as server j received them.  The
  // kept workers' slices are gathered chunk by chunk into the same flat staging buffers (one copy per (worker, server)
  // range that intersects the chunk), so the device side is the flat pipeline unchanged.
  const bool h_slices = st->grad_layout == PSYNC_GRADS_SLICES;
  HostLayout L;
  if (!host_layout(async_mode ? st->W : st->N, st->W, st->grad_dtype, chunk_elems, &L)) return PSYNC_EINVAL;
  if (work_bytes < L.total || (reinterpret_cast<uintptr_t>(d_work) & 255u) != 0) return PSYNC_EINVAL;
  if (!h_slices)
    for (int32_t k = 0; k < st->W; ++k)
      if (h_grads[k] == nullptr) return PSYNC_EINVAL;

  const int32_t W = st->W;
  int32_t N = async_mode ? W : st->N;  // async: replaced by the number of gradients that arrived
  const int64_t esz = st->grad_dtype == PSYNC_BF16 ? 2 : 4;
  char* work = static_cast<char*>(d_work);
  float* d_arrival = reinterpret_cast<float*>(work + L.off_arrival);
  int32_t* d_tags = reinterpret_cast<int32_t*>(work + L.off_tags);
  int32_t* d_kept = reinterpret_cast<int32_t*>(work + L.off_kept);
  float* d_tnth = reinterpret_cast<float*>(work + L.off_tnth);
  int32_t* d_status = reinterpret_cast<int32_t*>(work + L.off_status);
  int32_t* d_ident = reinterpret_cast<int32_t*>(work + L.off_ident);
  cudaStream_t s = static_cast<cudaStream_t>(stream);

  HostCtx local;                                   // used when the caller brought no context
  HostCtx* hc = ctx != nullptr ? static_cast<HostCtx*>(ctx) : &local;
  int result = PSYNC_OK;
  std::vector<int32_t> kept(N);  // N = W in async mode
  int32_t status = PSYNC_ECUDA;
  float t_nth = 0.f;

#define PSYNC_CU(call)              \
  do {                              \
    if ((call) != cudaSuccess) {    \
      result = PSYNC_ECUDA;         \
      goto cleanup;                 \
    }                               \
  } while (0)

  // 1. selection on the device (Alg. 4 l.3-6): the only thing the host learns is kept[] / status;
  //    async: the arrival order (Alg. 2, L85) and how many gradients arrived
  PSYNC_CU(cudaMemcpyAsync(d_arrival, h_arrival, sizeof(float) * W, cudaMemcpyHostToDevice, s));
  if (async_mode) {
    PSYNC_CU(psync::launch_order_by_arrival(d_arrival, W, 1, d_kept, d_status, s));  // d_status holds the count here
    PSYNC_CU(cudaMemcpyAsync(&status, d_status, sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    PSYNC_CU(cudaStreamSynchronize(s));
    N = status;
    if (h_n_arrived != nullptr) *h_n_arrived = N;
    if (N < 0 || N > W) {
      result = PSYNC_ECUDA;
      goto cleanup;
    }
    if (h_gamma != nullptr && N > 0)  // the tag area of the workspace is free in this mode: the rates of this batch
      PSYNC_CU(cudaMemcpyAsync(d_tags, h_gamma, sizeof(float) * N, cudaMemcpyHostToDevice, s));
    flat.N = N > 0 ? N : 1;
  } else {
    if (h_step_tag != nullptr)
      PSYNC_CU(cudaMemcpyAsync(d_tags, h_step_tag, sizeof(int32_t) * W, cudaMemcpyHostToDevice, s));
    PSYNC_CU(psync::launch_select_first_n(d_arrival, h_step_tag ? d_tags : nullptr, t, N, W, 1, d_kept, d_tnth, d_status, s));
    PSYNC_CU(cudaMemcpyAsync(&status, d_status, sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    PSYNC_CU(cudaStreamSynchronize(s));
    if (status != PSYNC_OK) {
      result = status;
      goto cleanup;
    }
    PSYNC_CU(cudaMemcpyAsync(&t_nth, d_tnth, sizeof(float), cudaMemcpyDeviceToHost, s));
  }
  if (N > 0) PSYNC_CU(cudaMemcpyAsync(kept.data(), d_kept, sizeof(int32_t) * N, cudaMemcpyDeviceToHost, s));
  for (int i = 0; i < 2; ++i)
    PSYNC_CU(psync::launch_fill_stage_table(reinterpret_cast<const void**>(work + L.off_ptrs[i]), d_ident,
                                            work + L.off_stage[i], L.stride_bytes, N > 0 ? N : 1, s));
  PSYNC_CU(cudaStreamSynchronize(s));
  if (h_slices)  // every slice of a KEPT worker must be there (dropped workers' slices are never looked at)
    for (int32_t n = 0; n < N; ++n)
      for (int32_t j = 0; j < st->M; ++j)
        if (st->h_shard_off[j + 1] > st->h_shard_off[j] && h_grads[static_cast<int64_t>(kept[n]) * st->M + j] == nullptr) {
          result = PSYNC_EINVAL;  // nothing has been updated yet
          goto cleanup;
        }
  if (h_kept != nullptr && N > 0) std::memcpy(h_kept, kept.data(), sizeof(int32_t) * N);
  if (h_t_nth != nullptr) *h_t_nth = t_nth;
  if (async_mode && N == 0) {  // nothing arrived: theta is unchanged (and still goes back to the host if asked for)
    if (h_theta_out != nullptr && st->P > 0) {
      PSYNC_CU(cudaMemcpyAsync(h_theta_out, st->d_theta, sizeof(float) * static_cast<size_t>(st->P), cudaMemcpyDeviceToHost, s));
      PSYNC_CU(cudaStreamSynchronize(s));
    }
    goto cleanup;
  }

  // 2./3. stream the kept buffers chunk by chunk; copy stream runs one chunk ahead of the kernel
  if (ctx == nullptr && !host_ctx_init(&local)) {
    result = PSYNC_ECUDA;
    goto cleanup;
  }
  {
    cudaStream_t copy_stream = hc->copy_stream;
    cudaEvent_t* copied = hc->copied;
    cudaEvent_t* consumed = hc->consumed;
    // both streams are idle here: `s` was synchronised above and every call ends with both streams drained
    int64_t c = 0;
    int32_t j_first = 0;
    for (int64_t first = 0; first < st->P; first += L.chunk, ++c) {
      const int buf = static_cast<int>(c & 1);
      const int64_t count = (st->P - first < L.chunk) ? (st->P - first) : L.chunk;
      while (h_slices && j_first + 1 < st->M && st->h_shard_off[j_first + 1] <= first) ++j_first;  // first server in chunk
      if (c >= 2) PSYNC_CU(cudaStreamWaitEvent(copy_stream, consumed[buf], 0));
      for (int32_t n = 0; n < N; ++n) {
        char* dst = work + L.off_stage[buf] + static_cast<int64_t>(n) * L.stride_bytes;
        if (!h_slices) {
          const char* src = static_cast<const char*>(h_grads[kept[n]]) + first * esz;
          PSYNC_CU(cudaMemcpyAsync(dst, src, static_cast<size_t>(count * esz), cudaMemcpyHostToDevice, copy_stream));
        } else {
          for (int32_t j = j_first; j < st->M && st->h_shard_off[j] < first + count; ++j) {  // servers in this chunk
            const int64_t lo = st->h_shard_off[j] > first ? st->h_shard_off[j] : first;
            const int64_t hi = st->h_shard_off[j + 1] < first + count ? st->h_shard_off[j + 1] : first + count;
            if (hi <= lo) continue;
            const char* slice = static_cast<const char*>(h_grads[static_cast<int64_t>(kept[n]) * st->M + j]);
            if (slice == nullptr) {  // a kept worker's slice is missing
              result = PSYNC_EINVAL;
              goto cleanup;
            }
            PSYNC_CU(cudaMemcpyAsync(dst + (lo - first) * esz, slice + (lo - st->h_shard_off[j]) * esz,
                                     static_cast<size_t>((hi - lo) * esz), cudaMemcpyHostToDevice, copy_stream));
          }
        }
      }
      PSYNC_CU(cudaEventRecord(copied[buf], copy_stream));
      PSYNC_CU(cudaStreamWaitEvent(s, copied[buf], 0));
      FusedParams p = make_params(&flat, first, count, reinterpret_cast<const void* const*>(work + L.off_ptrs[buf]),
                                  d_ident, nullptr);
      if (async_mode) {  // K4 on the staged chunk: slot i holds the i-th arrival
        p.gammas = h_gamma != nullptr ? reinterpret_cast<const float*>(d_tags) : nullptr;
        PSYNC_CU(psync::launch_async_apply_ring(p, st->grad_dtype, st->opt, st->ema_mode, st->grid_ctas, s));
      } else {
        PSYNC_CU(psync::launch_fused(p, st->grad_dtype, st->opt, st->ema_mode, st->variant, st->grid_ctas, s));
      }
      PSYNC_CU(cudaEventRecord(consumed[buf], s));
      if (h_theta_out != nullptr)
        PSYNC_CU(cudaMemcpyAsync(h_theta_out + first, st->d_theta + first, sizeof(float) * static_cast<size_t>(count),
                                 cudaMemcpyDeviceToHost, s));
    }
  }
  PSYNC_CU(cudaStreamSynchronize(hc->copy_stream));
  PSYNC_CU(cudaStreamSynchronize(s));

cleanup:
#undef PSYNC_CU
  if (result == PSYNC_ECUDA) cudaGetLastError();
  if (hc->copy_stream != nullptr) cudaStreamSynchronize(hc->copy_stream);
  if (ctx == nullptr) host_ctx_release(&local);
  return result;
}
}  // namespace

extern "C" {

PSYNC_API int psync_step_host_ctx(void* ctx, const psync_step* st, const float* h_arrival, const int32_t* h_step_tag,
                        int32_t t, const void* const* h_grads, float* h_theta_out, int32_t* h_kept, float* h_t_nth,
                        void* d_work, size_t work_bytes, int64_t chunk_elems, void* stream) {
  return host_step_impl(ctx, st, h_arrival, h_step_tag, t, h_grads, h_theta_out, h_kept, h_t_nth, d_work, work_bytes,
                        chunk_elems, stream, false, nullptr, nullptr);
}

PSYNC_API int psync_async_step_host(void* ctx, const psync_step* st, const float* h_arrival, const void* const* h_grads,
                          const float* h_gamma, float* h_theta_out, int32_t* h_order, int32_t* h_n_arrived, void* d_work,
                          size_t work_bytes, int64_t chunk_elems, void* stream) {
  return host_step_impl(ctx, st, h_arrival, nullptr, 0, h_grads, h_theta_out, h_order, nullptr, d_work, work_bytes,
                        chunk_elems, stream, true, h_gamma, h_n_arrived);
}

}  // extern "C"
