// Evaluation of one 2D Gabor primitive at one pixel (Eq.12) -- shared by the forward and the
// backward blend kernels so that both take bit-identical skip / clamp decisions: every operation is an
// explicit round-to-nearest intrinsic (no compiler-chosen contraction).
#pragma once

#include "common.cuh"

namespace gabsplat {

constexpr float kTwoPi = 6.28318530717958647692f;

template <int K>
struct PairEval {
  float dx, dy, u, v, G, M, raw, alpha;
  float cs[K > 0 ? K : 1], sn[K > 0 ? K : 1];
};

// Quadratic form of the envelope from the packed Cholesky factor: q = -(u^2 + v^2) <= 0  (Eq.3 :101).
__device__ __forceinline__ float envelope_q(float L11, float L21, float L22, float dx, float dy, float& u, float& v) {
  u = __fmaf_rn(L21, dy, __fmul_rn(L11, dx));
  v = __fmul_rn(L22, dy);
  return -__fmaf_rn(u, u, __fmul_rn(v, v));
}

// cos / sin of 2 pi * phase with the phase in cycles: reduce to [-1/2, 1/2] turns first, then MUFU.
__device__ __forceinline__ float cos_turns(float ph) {
  const float r = __fsub_rn(ph, rintf(ph));
  return __cosf(__fmul_rn(kTwoPi, r));
}
__device__ __forceinline__ float sin_turns(float ph) {
  const float r = __fsub_rn(ph, rintf(ph));
  return __sinf(__fmul_rn(kTwoPi, r));
}

// Modulation M = (1 - sum w) + sum w cos(2 pi f2D . d) = 1 + sum w (cos - 1)   (Eq.12 bracket)
// rec points at the staged record of the primitive (floats).  WANT_SIN also fills e.sn.
template <int K, bool WANT_SIN>
__device__ __forceinline__ void modulation(const float* __restrict__ rec, PairEval<K>& e) {
  float M = 1.0f;
  constexpr int wo = weight_offset(K);
#pragma unroll
  for (int k = 0; k < K; ++k) {
    const float ph = __fmaf_rn(rec[12 + 2 * k + 1], e.dy, __fmul_rn(rec[12 + 2 * k], e.dx));
    const float r = __fsub_rn(ph, rintf(ph));
    const float a = __fmul_rn(kTwoPi, r);
    e.cs[k] = __cosf(a);
    if (WANT_SIN) e.sn[k] = __sinf(a);
    M = __fmaf_rn(rec[wo + k], __fsub_rn(e.cs[k], 1.0f), M);
  }
  e.M = M;
}

}  // namespace gabsplat
