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
  CHECK(psync_version() >= 130);
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
  printf("abi_smoke ok: %s\n", psync_status_string(PSYNC_OK));
  return 0;
}
