/* Plain-C client of include/psync.h: no Python, no torch.  Links libpsync.so and the CUDA runtime, runs one
 * parameter-server step (Alg. 4) on hand-checkable inputs and verifies the exact results.
 *
 *   W = 5 workers, N = 4, b = 1; arrival = {0.5, 2.0, 1.0, 0.125, 3.0}  ->  worker 4 is the straggler: kept = {0,1,2,3},
 *   t_Nth = 2.0.  Worker k's gradient is the constant (k+1)/4 (worker 4 holds NaN: it must never be read).
 *   mean = (0.25+0.5+0.75+1.0)/4 = 0.625; SGD gamma = 0.5, theta = 1  ->  theta' = 0.6875;
 *   EMA alpha = 0.5, ema = 0  ->  ema' = 0.34375.  All dyadic: exact in fp32.
 * Exit code 0 = all checks passed. */
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>

#include "psync.h"

#define CHECK(cond)                                                  \
  do {                                                               \
    if (!(cond)) {                                                   \
      fprintf(stderr, "FAILED line %d: %s\n", __LINE__, #cond);      \
      return 1;                                                      \
    }                                                                \
  } while (0)

int main(void) {
  enum { P = 4099, W = 5, N = 4 };
  const float arrival[W] = {0.5f, 2.0f, 1.0f, 0.125f, 3.0f};
  const int64_t shard_off[3] = {0, 1000, P};
  float *h = (float*)malloc(sizeof(float) * P), *d_theta, *d_ema, *d_arrival, *d_tnth, *d_grad[W];
  int32_t *d_kept, *d_status, kept[N], status = -99;
  const void** d_table;
  float tnth = 0.f;
  CHECK(psync_version() >= 200);
  CHECK(cudaMalloc((void**)&d_theta, sizeof(float) * P) == cudaSuccess);
  CHECK(cudaMalloc((void**)&d_ema, sizeof(float) * P) == cudaSuccess);
  CHECK(cudaMalloc((void**)&d_arrival, sizeof(arrival)) == cudaSuccess);
  CHECK(cudaMalloc((void**)&d_tnth, sizeof(float)) == cudaSuccess);
  CHECK(cudaMalloc((void**)&d_kept, sizeof(kept)) == cudaSuccess);
  CHECK(cudaMalloc((void**)&d_status, sizeof(int32_t)) == cudaSuccess);
  CHECK(cudaMalloc((void**)&d_table, sizeof(void*) * W) == cudaSuccess);
  for (int k = 0; k < W; ++k) {
    CHECK(cudaMalloc((void**)&d_grad[k], sizeof(float) * P) == cudaSuccess);
    for (int i = 0; i < P; ++i) h[i] = (k == 4) ? NAN : 0.25f * (float)(k + 1);
    CHECK(cudaMemcpy(d_grad[k], h, sizeof(float) * P, cudaMemcpyHostToDevice) == cudaSuccess);
  }
  CHECK(cudaMemcpy(d_table, d_grad, sizeof(void*) * W, cudaMemcpyHostToDevice) == cudaSuccess);
  for (int i = 0; i < P; ++i) h[i] = 1.0f;
  CHECK(cudaMemcpy(d_theta, h, sizeof(float) * P, cudaMemcpyHostToDevice) == cudaSuccess);
  CHECK(cudaMemset(d_ema, 0, sizeof(float) * P) == cudaSuccess);
  CHECK(cudaMemcpy(d_arrival, arrival, sizeof(arrival), cudaMemcpyHostToDevice) == cudaSuccess);

  psync_step st = {0};
  st.P = P; st.M = 2; st.h_shard_off = shard_off; st.N = N; st.W = W;
  st.d_grads = (const void* const*)d_table; st.grad_dtype = PSYNC_F32;
  st.d_kept = d_kept; st.d_status = d_status; st.d_theta = d_theta; st.d_ema = d_ema;
  st.opt = PSYNC_SGD; st.ema_mode = PSYNC_EMA_POST; st.gamma_t = 0.5f; st.alpha = 0.5f;

  /* argument errors are reported synchronously and enqueue nothing */
  st.N = 0;
  CHECK(psync_step_device(&st, d_arrival, NULL, 0, d_tnth, NULL) == PSYNC_EINVAL);
  st.N = N;
  CHECK(psync_select_first_n(NULL, NULL, 0, N, W - N, d_kept, NULL, d_status, NULL) == PSYNC_EINVAL);

  /* the step: selection + fused aggregate/update/EMA, one call, default stream */
  CHECK(psync_step_device(&st, d_arrival, NULL, 0, d_tnth, NULL) == PSYNC_OK);
  CHECK(cudaDeviceSynchronize() == cudaSuccess);
  CHECK(cudaMemcpy(kept, d_kept, sizeof(kept), cudaMemcpyDeviceToHost) == cudaSuccess);
  CHECK(cudaMemcpy(&status, d_status, sizeof(status), cudaMemcpyDeviceToHost) == cudaSuccess);
  CHECK(cudaMemcpy(&tnth, d_tnth, sizeof(tnth), cudaMemcpyDeviceToHost) == cudaSuccess);
  CHECK(status == PSYNC_OK && tnth == 2.0f);
  for (int n = 0; n < N; ++n) CHECK(kept[n] == n);
  CHECK(cudaMemcpy(h, d_theta, sizeof(float) * P, cudaMemcpyDeviceToHost) == cudaSuccess);
  for (int i = 0; i < P; ++i) CHECK(h[i] == 0.6875f);
  CHECK(cudaMemcpy(h, d_ema, sizeof(float) * P, cudaMemcpyDeviceToHost) == cudaSuccess);
  for (int i = 0; i < P; ++i) CHECK(h[i] == 0.34375f);

  /* the two-call form and the standalone EMA: theta'' = 0.6875 - 0.3125 = 0.375; ema'' = 0.5*0.34375 + 0.5*0.375 */
  st.ema_mode = PSYNC_EMA_OFF;
  CHECK(psync_select_first_n(d_arrival, NULL, 0, N, W - N, d_kept, d_tnth, d_status, NULL) == PSYNC_OK);
  CHECK(psync_aggregate_update(&st, NULL) == PSYNC_OK);
  CHECK(psync_ema(d_ema, d_theta, P, 0.5f, NULL) == PSYNC_OK);
  CHECK(cudaDeviceSynchronize() == cudaSuccess);
  CHECK(cudaMemcpy(h, d_theta, sizeof(float) * P, cudaMemcpyDeviceToHost) == cudaSuccess);
  for (int i = 0; i < P; ++i) CHECK(h[i] == 0.375f);
  CHECK(cudaMemcpy(h, d_ema, sizeof(float) * P, cudaMemcpyDeviceToHost) == cudaSuccess);
  for (int i = 0; i < P; ++i) CHECK(h[i] == 0.359375f);

  /* fewer than N arrivals: status says so on the device and nothing is touched */
  {
    const float late[W] = {0.5f, INFINITY, NAN, 0.125f, 3.0f};
    CHECK(cudaMemcpy(d_arrival, late, sizeof(late), cudaMemcpyHostToDevice) == cudaSuccess);
    CHECK(psync_step_device(&st, d_arrival, NULL, 0, d_tnth, NULL) == PSYNC_OK);
    CHECK(cudaDeviceSynchronize() == cudaSuccess);
    CHECK(cudaMemcpy(&status, d_status, sizeof(status), cudaMemcpyDeviceToHost) == cudaSuccess);
    CHECK(status == PSYNC_ETOOFEW);
    CHECK(cudaMemcpy(h, d_theta, sizeof(float) * P, cudaMemcpyDeviceToHost) == cudaSuccess);
    for (int i = 0; i < P; ++i) CHECK(h[i] == 0.375f);
  }
  /* the slices layout: what each server RECEIVES -- one cudaMalloc per (worker, server) slice, the slices of worker 1 placed
   * 4 bytes after the allocation boundary; theta = 1 again; same kept set {0,1,2,3} => theta' = 0.6875, ema' = 0.5*ema + 0.34375 */
  {
    enum { M = 2 };
    float* slice[W][M];
    const void* h_table[W * M];
    const void** d_slices;
    int64_t *d_off, *d_tiles, tiles[M + 1];
    for (int k = 0; k < W; ++k)
      for (int j = 0; j < M; ++j) {
        const int64_t len = shard_off[j + 1] - shard_off[j];
        float* base;
        CHECK(cudaMalloc((void**)&base, sizeof(float) * (size_t)(len + 1)) == cudaSuccess);
        slice[k][j] = base + (k == 1 ? 1 : 0);
        for (int64_t i = 0; i < len; ++i) h[i] = (k == 4) ? NAN : 0.25f * (float)(k + 1);
        CHECK(cudaMemcpy(slice[k][j], h, sizeof(float) * (size_t)len, cudaMemcpyHostToDevice) == cudaSuccess);
        h_table[k * M + j] = (k == 4) ? NULL : slice[k][j];          /* the straggler's slices are not even there */
      }
    CHECK(cudaMalloc((void**)&d_slices, sizeof(h_table)) == cudaSuccess);
    CHECK(cudaMemcpy(d_slices, h_table, sizeof(h_table), cudaMemcpyHostToDevice) == cudaSuccess);
    CHECK(cudaMalloc((void**)&d_off, sizeof(shard_off)) == cudaSuccess);
    CHECK(cudaMalloc((void**)&d_tiles, sizeof(tiles)) == cudaSuccess);
    CHECK(cudaMemcpy(d_off, shard_off, sizeof(shard_off), cudaMemcpyHostToDevice) == cudaSuccess);
    CHECK(psync_shard_worklist(d_off, M, PSYNC_F32, d_tiles, NULL) == PSYNC_OK);
    CHECK(cudaMemcpy(tiles, d_tiles, sizeof(tiles), cudaMemcpyDeviceToHost) == cudaSuccess);
    CHECK(tiles[0] == 0 && tiles[1] == 1 && tiles[2] == 1 + 4);      /* ceil(1000/1024), ceil(3099/1024) */
    for (int i = 0; i < P; ++i) h[i] = 1.0f;
    CHECK(cudaMemcpy(d_theta, h, sizeof(float) * P, cudaMemcpyHostToDevice) == cudaSuccess);
    CHECK(cudaMemcpy(d_arrival, arrival, sizeof(arrival), cudaMemcpyHostToDevice) == cudaSuccess);
    st.d_grads = (const void* const*)d_slices; st.grad_layout = PSYNC_GRADS_SLICES;
    st.d_shard_off = d_off; st.d_tile_start = d_tiles; st.ema_mode = PSYNC_EMA_POST;
    st.d_tile_start = NULL;
    CHECK(psync_step_device(&st, d_arrival, NULL, 0, d_tnth, NULL) == PSYNC_EINVAL);   /* slices need the work list */
    st.d_tile_start = d_tiles;
    CHECK(psync_step_device(&st, d_arrival, NULL, 0, d_tnth, NULL) == PSYNC_OK);
    CHECK(cudaDeviceSynchronize() == cudaSuccess);
    CHECK(cudaMemcpy(&status, d_status, sizeof(status), cudaMemcpyDeviceToHost) == cudaSuccess);
    CHECK(status == PSYNC_OK);
    CHECK(cudaMemcpy(h, d_theta, sizeof(float) * P, cudaMemcpyDeviceToHost) == cudaSuccess);
    for (int i = 0; i < P; ++i) CHECK(h[i] == 0.6875f);
    CHECK(cudaMemcpy(h, d_ema, sizeof(float) * P, cudaMemcpyDeviceToHost) == cudaSuccess);
    for (int i = 0; i < P; ++i) CHECK(h[i] == 0.5f * 0.359375f + 0.34375f);
    /* Alg. 2 per parameter server on the same slices: every arriving gradient is one iteration, each
     * server in ITS arrival order; worker 4 never arrives (its slices are NULL).  theta = 1, ema = 0, gamma = 0.5,
     * alpha = 0.5, EMA_PRE (the literal L87), gradients 0.25 (k+1):
     *   server 0: order {3,0,2,1}: theta 1 -> .5 -> .375 -> 0 -> -.25;   ema .5 -> .5 -> .4375 -> .21875
     *   server 1: order {1,0,3,2}: theta 1 -> .75 -> .625 -> .125 -> -.25; ema .5 -> .625 -> .625 -> .375
     * Clip factors of the sliced gradients with a bound no norm reaches: exactly 1. */
    {
      const float arr2[M][W] = {{0.5f, 2.0f, 1.0f, 0.125f, INFINITY}, {1.0f, 0.25f, 4.0f, 2.0f, NAN}};
      const int32_t want_order[M][4] = {{3, 0, 2, 1}, {1, 0, 3, 2}};
      float *d_arr2, *d_scales, scales[W];
      int32_t *d_order, *d_n, order[M][W], n_arr[M];
      void* d_work;
      const size_t work_bytes = psync_clip_slices_workspace_bytes(4, M, shard_off, PSYNC_F32);
      CHECK(work_bytes > 0);
      CHECK(cudaMalloc((void**)&d_arr2, sizeof(arr2)) == cudaSuccess);
      CHECK(cudaMalloc((void**)&d_scales, sizeof(scales)) == cudaSuccess);
      CHECK(cudaMalloc((void**)&d_order, sizeof(order)) == cudaSuccess);
      CHECK(cudaMalloc((void**)&d_n, sizeof(n_arr)) == cudaSuccess);
      CHECK(cudaMalloc(&d_work, work_bytes) == cudaSuccess);
      CHECK(cudaMemcpy(d_arr2, arr2, sizeof(arr2), cudaMemcpyHostToDevice) == cudaSuccess);
      CHECK(cudaMemset(d_scales, 0xFF, sizeof(scales)) == cudaSuccess);
      CHECK(psync_clip_scales_slices((const void* const*)d_slices, 4, M, shard_off, d_off, PSYNC_F32, 1.0e6f, d_scales,
                                     d_work, work_bytes, NULL) == PSYNC_OK);       /* workers 0..3: the first 4 rows */
      CHECK(psync_clip_scales_slices((const void* const*)d_slices, 4, M, shard_off, d_off, PSYNC_F32, 0.0f, d_scales,
                                     d_work, work_bytes, NULL) == PSYNC_EINVAL);
      CHECK(psync_order_by_arrival_sharded(d_arr2, W, M, d_order, d_n, NULL) == PSYNC_OK);
      for (int i = 0; i < P; ++i) h[i] = 1.0f;
      CHECK(cudaMemcpy(d_theta, h, sizeof(float) * P, cudaMemcpyHostToDevice) == cudaSuccess);
      CHECK(cudaMemset(d_ema, 0, sizeof(float) * P) == cudaSuccess);
      st.N = W; st.d_kept = d_order; st.d_status = NULL; st.d_n_kept = d_n; st.kept_stride = W; st.per_shard = 1;
      st.ema_mode = PSYNC_EMA_PRE;
      CHECK(psync_async_apply(&st, NULL, d_scales, NULL) == PSYNC_OK);
      CHECK(cudaDeviceSynchronize() == cudaSuccess);
      CHECK(cudaMemcpy(scales, d_scales, sizeof(scales), cudaMemcpyDeviceToHost) == cudaSuccess);
      for (int k = 0; k < 4; ++k) CHECK(scales[k] == 1.0f);
      CHECK(cudaMemcpy(order, d_order, sizeof(order), cudaMemcpyDeviceToHost) == cudaSuccess);
      CHECK(cudaMemcpy(n_arr, d_n, sizeof(n_arr), cudaMemcpyDeviceToHost) == cudaSuccess);
      for (int j = 0; j < M; ++j) {
        CHECK(n_arr[j] == 4);
        for (int i = 0; i < 4; ++i) CHECK(order[j][i] == want_order[j][i]);
      }
      CHECK(cudaMemcpy(h, d_theta, sizeof(float) * P, cudaMemcpyDeviceToHost) == cudaSuccess);
      for (int i = 0; i < P; ++i) CHECK(h[i] == -0.25f);
      CHECK(cudaMemcpy(h, d_ema, sizeof(float) * P, cudaMemcpyDeviceToHost) == cudaSuccess);
      for (int i = 0; i < P; ++i) CHECK(h[i] == (i < shard_off[1] ? 0.21875f : 0.375f));
    }
  }
  printf("abi_smoke ok: %s\n", psync_status_string(PSYNC_OK));
  return 0;
}
