// aev_common.cuh -- per-warp neighbour staging shared by the AEV forward (K3) and backward (K7) kernels.
// One warp owns one centre atom (BASELINE.json north_star: "one warp per centre atom, coalesced float4
// coordinate loads, triplet loop in registers/smem").  Formulas: SURVEY.md Appendix A.
#pragma once
#include "nnp_internal.h"

namespace nnp {

constexpr int AEV_WARPS = 8;      // warps (centres) per block of the backward kernel
constexpr int AEV_FWD_WARPS = 4;  // ... of the forward kernel (measured: 4 -> 71.8 us, 8 -> 73.6 us; backward 8 -> 96 us, 4 -> 99 us)

// Per-warp shared staging of one centre's environment.
struct WarpEnv {
  float4 u[RCAP_MAX];      // radial neighbours: unit vector (x,y,z) and R
  float wR[RCAP_MAX];      // c_R * f_C(R; Rcr)
  float4 ua[ACAP_MAX];     // angular neighbours (subset, same order): unit vector and R
  float fA[ACAP_MAX];      // f_C(R; Rca)
  float dfA[ACAP_MAX];     // f_C'(R; Rca)
  uint8_t posA[ACAP_MAX];  // position of the angular neighbour in the radial row
  uint8_t slotR[RCAP_MAX];
  uint8_t slotA[ACAP_MAX];
  int segR[MAX_S + 1];     // radial row is sorted by species slot: segment starts
  int segA[MAX_S + 1];
};

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

// Loads the centre's rows into `e` (all lanes participate).  Returns nR, nA through references.
__device__ __forceinline__ void load_env(const AevConst& c, const GridInfo* __restrict__ g,
                                         const float4* __restrict__ spos, const uint32_t* __restrict__ rowR,
                                         const uint8_t* __restrict__ rowA, int nR, int nA, float4 ci, int lane,
                                         WarpEnv& e) {
  float ev[9];   // cell edge vectors (orthorhombic: diagonal)
#pragma unroll
  for (int k = 0; k < 9; ++k) ev[k] = g->ev[k];
  int seg[MAX_S];
#pragma unroll
  for (int s = 0; s < MAX_S; ++s) seg[s] = 0;
  for (int q0 = 0; q0 < nR; q0 += 32) {
    const int q = q0 + lane;
    int slot = -1;
    if (q < nR) {
      const uint32_t ent = rowR[q];
      const int jp = (int)(ent & JMASK);
      const int oc = (int)(ent >> JBITS);
      const float4 pj = spos[jp];
      float sx, sy, sz;
      cell_shift(ev, (oc & 3) - 1, ((oc >> 2) & 3) - 1, ((oc >> 4) & 3) - 1, sx, sy, sz);
      const float dx = (pj.x - ci.x) + sx, dy = (pj.y - ci.y) + sy, dz = (pj.z - ci.z) + sz;
      const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
      const float rinv = rsqrtf(d2);
      const float R = d2 * rinv;
      slot = (__float_as_int(pj.w) >> 28) & 7;
      float f, df;
      cutoff(fminf(R, c.Rcr), c.inv_Rcr, f, df);
      e.u[q] = make_float4(dx * rinv, dy * rinv, dz * rinv, R);
      e.wR[q] = c.cR * f;
      e.slotR[q] = (uint8_t)slot;
    }
#pragma unroll
    for (int s = 0; s < MAX_S; ++s) seg[s] += __popc(__ballot_sync(0xffffffffu, slot == s));
  }
  if (lane == 0) {
    int run = 0;
#pragma unroll
    for (int s = 0; s < MAX_S; ++s) { e.segR[s] = run; run += seg[s]; }
    e.segR[MAX_S] = run;
  }
  __syncwarp();
#pragma unroll
  for (int s = 0; s < MAX_S; ++s) seg[s] = 0;
  for (int a0 = 0; a0 < nA; a0 += 32) {
    const int a = a0 + lane;
    int slot = -1;
    if (a < nA) {
      const int p = rowA[a];
      const float4 v = e.u[p];
      float f, df;
      cutoff(fminf(v.w, c.Rca), c.inv_Rca, f, df);
      slot = e.slotR[p];
      e.ua[a] = v; e.fA[a] = f; e.dfA[a] = df; e.posA[a] = (uint8_t)p; e.slotA[a] = (uint8_t)slot;
    }
#pragma unroll
    for (int s = 0; s < MAX_S; ++s) seg[s] += __popc(__ballot_sync(0xffffffffu, slot == s));
  }
  if (lane == 0) {
    int run = 0;
#pragma unroll
    for (int s = 0; s < MAX_S; ++s) { e.segA[s] = run; run += seg[s]; }
    e.segA[MAX_S] = run;
  }
  __syncwarp();
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
