// aev_common.cuh -- small device helpers shared by the AEV forward (K3) and backward (K7) kernels.
// One warp owns one centre atom (BASELINE.json north_star: "one warp per centre atom, coalesced float4
// coordinate loads, triplet loop in registers/smem").  Formulas: SURVEY.md Appendix A.
#pragma once
#include "nnp_internal.h"

namespace nnp {

constexpr int AEV_WARPS = 4;      // warps (centres) per block of the backward kernel (measured, 80 registers: 8 -> 86.6 us, 4 -> 84.2 us, 2 -> 85.5 us)
constexpr int AEV_FWD_WARPS = 2;  // ... of the forward kernel (measured, 48 registers: 8 -> 73.6 us, 4 -> 67.3 us, 2 -> 66.5 us)

__device__ __forceinline__ float ex2f(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__device__ __forceinline__ float lg2f(float x) {
  float y;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// f_C(R;Rc) = 0.5 cos(pi R / Rc) + 0.5 and its derivative (App. A "Cut-off"); R <= Rc is guaranteed by the list.
__device__ __forceinline__ void cutoff(float R, float inv_Rc, float& f, float& df) {
  const float x = 3.14159265358979f * R * inv_Rc;      // in [0, pi]: sin.approx / cos.approx err < 2^-21 absolute
  const float s = __sinf(x), c = __cosf(x);
  f = 0.5f * c + 0.5f;
  df = -0.5f * 3.14159265358979f * inv_Rc * s;
}

// zeta-th power of B (zeta = 32 by five squarings, App. A "Trig-free evaluation"); also B^(zeta-1).
__device__ __forceinline__ void bpow(const AevConst& c, float B, float& Bz, float& Bzm1) {
  if (c.zeta_is_32) {
    const float B2 = B * B, B4 = B2 * B2, B8 = B4 * B4, B16 = B8 * B8;
    Bzm1 = B16 * B8 * (B4 * B2 * B);
    Bz = B16 * B16;
  } else {
    Bzm1 = (B > 0.f) ? __powf(B, c.zeta - 1.0f) : 0.f;
    Bz = Bzm1 * B;
  }
}

}  // namespace nnp
