// Pieces shared by Alg. 2's two kernels (K4 async_kernel.cu: flat buffers, one arrival order; K4s
// async_sharded_kernel.cu: Alg. 2 per parameter server j over the (server, tile) work list): how one arriving
// gradient -- its 16-byte unit -- is applied to the parameters a thread holds.
#pragma once

#include "psync_device.cuh"

namespace psync {
namespace dev {

template <bool BF16>
__device__ __forceinline__ float unit_element(const uint4& r, int e) {
  const uint32_t w = (&r.x)[BF16 ? (e >> 1) : e];
  if (BF16) return __uint_as_float((e & 1) ? (w & 0xFFFF0000u) : (w << 16));
  return __uint_as_float(w);
}

// elements 2i and 2i+1 of a 16-byte unit as one fp32x2 operand
template <bool BF16>
__device__ __forceinline__ float2 unit_pair(const uint4& r, int i) {
  if (BF16) {
    const uint32_t w = (&r.x)[i];
    return make_float2(__uint_as_float(w << 16), __uint_as_float(w & 0xFFFF0000u));
  }
  return make_float2(__uint_as_float((&r.x)[2 * i]), __uint_as_float((&r.x)[2 * i + 1]));
}

// one arriving gradient (its 16-byte unit r) applied to the E parameters a thread holds, two at a time
template <bool BF16, int OPT, int EMA, bool SCALED>
__device__ __forceinline__ void apply_unit(const uint4& r, float scale, float gamma, float2* th, float2* em, float2* a0,
                                           float2* a1, const PairCoeffs& c, unsigned& bad) {
  constexpr int E = BF16 ? 8 : 4;
  const float2 scale2 = dup2(scale), gamma2 = dup2(gamma);
#pragma unroll
  for (int i = 0; i < E / 2; ++i)
    update_pair_g<OPT, EMA, SCALED>(unit_pair<BF16>(r, i), scale2, gamma2, th[i], em[i], a0[i], a1[i], c, bad);
}

}  // namespace dev
}  // namespace psync
