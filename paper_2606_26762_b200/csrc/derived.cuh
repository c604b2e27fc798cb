// Per-prototype DERIVED data (kept next to the state of record so the scoring / attention kernels stream compact
// operands): the Eq. 1 record, the bf16 shadows of the normalised key centre.  Shared by every
// kernel that rewrites a prototype (slot fill, update, import, maintenance) so that they all produce the same bits.
#pragma once
#include "common.cuh"

namespace pkv {

// 1 / sqrt(x) in fp64 from the fp32 hardware estimate and two Newton steps (2^-22 -> 2^-44 -> below fp64 rounding): the
// library rsqrt(double) costs ~40 instructions and three of them per touched prototype were 8 % of the update kernel
// (profiles/r02_experiments.md).  Every writer of derived data goes through these helpers, so they agree bit for bit.
__device__ __forceinline__ double rsqrt_nr(double x) {
  double y = (double)rsqrtf((float)x);
  y = y * fma(-0.5 * x * y, y, 1.5);
  y = y * fma(-0.5 * x * y, y, 1.5);
  return y;
}
__device__ __forceinline__ float inv_norm(float cc) { return cc > 0.f ? (float)rsqrt_nr((double)cc) : 0.f; }
// log n_k of Eq. 4 (bias of the pseudo-tokens; consumed in bf16 attention: 1e-6 relative is ample)
__device__ __forceinline__ float log_mass(int n) { return n >= 1 ? __logf((float)n) : 0.f; }

// Token-independent part of Eq. 1 for one prototype.  Sigma + eps I = R R^T (Cholesky),
// d_Mah^2 = |R^-1 delta|^2 = (dx/r11)^2 + ((dy - r21 dx/r11)/r22)^2.  Evaluated in fp64 from the fp32 state.
__device__ __forceinline__ ScoreRec make_rec(float cc, float mux, float muy, float sxx, float sxy, float syy, int tau,
                                             const Hyper& H) {
  ScoreRec r;
  r.invc = inv_norm(cc);
  r.mux = mux; r.muy = muy;
  const double a = (double)sxx + (double)H.sigma_eps, b = (double)sxy, e = (double)syy + (double)H.sigma_eps;
  const double i11 = rsqrt_nr(a);              // 1 / r11
  const double r21 = b * i11;
  const double t = e - r21 * r21;              // r22^2
  const double i22 = t > 0.0 ? rsqrt_nr(t) : (double)INFINITY;
  // lambda_sp * d_Mah = sqrt(q) with factors scaled by lambda_sp; for MAH_SQUARED scale by sqrt(lambda_sp).
  const double lam = (H.flags & PROTOKV_MAH_SQUARED) ? sqrt((double)H.lambda_sp) : (double)H.lambda_sp;
  r.u = (float)(lam * i11);
  r.v = (float)(lam * i22);
  r.w = (float)(lam * r21 * i11 * i22);
  r.tau = tau;
  r.tauf = (float)tau;
  return r;
}

__device__ __forceinline__ void split_bf16(float x, __nv_bfloat16& hi, __nv_bfloat16& lo) {
  hi = __float2bfloat16_rn(x);
  lo = __float2bfloat16_rn(x - __bfloat162float(hi));
}

// bf16 shadows of the NORMALISED key centre c / |c| = hi + lo (+ O(2^-17)): the tcgen05 assignment contracts the
// evicted keys with these, so its accumulator is |K_j| cos(K_j, c_k) and Eq. 1 needs no per-column scale.
template <int VEC>
__device__ __forceinline__ void store_shadows(const Dev& V, size_t off, const float (&c)[VEC], float invc) {
  if (!V.c_hi) return;
  __nv_bfloat16 hi[VEC], lo[VEC];
#pragma unroll
  for (int v = 0; v < VEC; ++v) split_bf16(c[v] * invc, hi[v], lo[v]);
  if (VEC == 4) {
    *reinterpret_cast<uint2*>(V.c_hi + off) = *reinterpret_cast<const uint2*>(hi);
    *reinterpret_cast<uint2*>(V.c_lo + off) = *reinterpret_cast<const uint2*>(lo);
  } else {
#pragma unroll
    for (int v = 0; v < VEC; ++v) { V.c_hi[off + v] = hi[v]; V.c_lo[off + v] = lo[v]; }
  }
}

// bf16 copies of a centre (key or value side) for the decode-style attention: dst = c_bf or p_bf
template <int VEC>
__device__ __forceinline__ void store_bf16_copy(__nv_bfloat16* dst, size_t off, const float (&x)[VEC]) {
  if (!dst) return;
  __nv_bfloat16 h[VEC];
#pragma unroll
  for (int v = 0; v < VEC; ++v) h[v] = __float2bfloat16_rn(x[v]);
  if (VEC == 4) *reinterpret_cast<uint2*>(dst + off) = *reinterpret_cast<const uint2*>(h);
  else {
#pragma unroll
    for (int v = 0; v < VEC; ++v) dst[off + v] = h[v];
  }
}

}  // namespace pkv
