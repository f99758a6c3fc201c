// aev_backward.cuh -- the per-centre AEV backward pass (K7), shared by k_aev_backward (force.cu) and the single-kernel
// evaluation of small systems (small.cu).  One warp per centre; formulas: SURVEY.md Appendix A "Forces".
#pragma once
#include "aev_common.cuh"

namespace nnp {

__device__ __forceinline__ long long to_fix(float v) { return __float2ll_rn(v * 1099511627776.0f); }  // 2^40
__device__ __forceinline__ long long shfl_xor_ll(long long v, int o) {
  int lo = __shfl_xor_sync(0xffffffffu, (int)(v & 0xffffffffll), o);
  int hi = __shfl_xor_sync(0xffffffffu, (int)(v >> 32), o);
  return ((long long)hi << 32) | (unsigned int)lo;
}

// Both shares of one unordered angular pair {j,k} of centre i: oj = dE_i/dr_j and ok = dE_i/dr_k contributions of the
// 32 sub-features of the pair's species block (SURVEY.md Appendix A "Forces"; gb = this centre's dE/dAEV pieces).
// Per-warp staging of one centre's environment for the backward pass.
struct BwdEnv {
  float4 u[RCAP_MAX];      // radial neighbours: unit vector (x,y,z) and R
  float4 ua[ACAP_MAX];     // angular neighbours (subset, same order): unit vector and R
  float fA[ACAP_MAX];      // f_C(R; Rca)
  float dfA[ACAP_MAX];     // f_C'(R; Rca)
  uint8_t slotR[RCAP_MAX];
  uint8_t slotA[ACAP_MAX];
  uint8_t ainv[RCAP_MAX];  // position in the radial row -> index among the angular neighbours, 255 = not one
};

__device__ __forceinline__ void bwd_load_env(const AevConst& c, const GridInfo* __restrict__ g,
                                             const float4* __restrict__ spos, const uint32_t* __restrict__ rowR,
                                             const uint8_t* __restrict__ rowA, int nR, int nA, float4 ci, int lane,
                                             BwdEnv& e) {
  float ev[9];   // cell edge vectors (orthorhombic: diagonal)
#pragma unroll
  for (int k = 0; k < 9; ++k) ev[k] = g->ev[k];
  for (int q0 = 0; q0 < nR; q0 += 32) {
    const int q = q0 + lane;
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
      e.u[q] = make_float4(dx * rinv, dy * rinv, dz * rinv, d2 * rinv);
      e.slotR[q] = (uint8_t)((__float_as_int(pj.w) >> 28) & 7);
      e.ainv[q] = 255;
    }
  }
  __syncwarp();
  for (int a0 = 0; a0 < nA; a0 += 32) {
    const int a = a0 + lane;
    if (a < nA) {
      const int p = rowA[a];
      const float4 v = e.u[p];
      float f, df;
      cutoff(fminf(v.w, c.Rca), c.inv_Rca, f, df);
      e.ua[a] = v; e.fA[a] = f; e.dfA[a] = df; e.slotA[a] = e.slotR[p]; e.ainv[p] = (uint8_t)a;
    }
  }
  __syncwarp();
}

struct PairShares { float jx, jy, jz, kx, ky, kz; };
// Packed fp32 arithmetic (fma.rn.f32x2, sm_100): the theta shifts are handled two per instruction, and the dot products
// over z of the 4 x 8 dE/dAEV block accumulate two partial sums per instruction -- the kernel is bound by issue slots.
__device__ __forceinline__ PairShares pair_shares(const AevConst& c, float zm1, const float4* gb, int gs, float4 uj,
                                                  float fj, float dfj, float4 uk, float fk, float dfk) {
  const float u = fmaf(uj.x, uk.x, fmaf(uj.y, uk.y, uj.z * uk.z));
  const float cc = c.cTheta * u;
  const float ss = sqrtf(fmaxf(1.0f - cc * cc, 1e-12f));
  const float kd = 0.5f * c.zeta * c.cTheta / ss;            // -0.5 zeta dtheta/du
  const float2 cc2 = make_float2(cc, cc), ss2 = make_float2(ss, ss), ncc2 = make_float2(-cc, -cc);
  const float2 h2 = make_float2(0.5f, 0.5f), kd2 = make_float2(kd, kd);
  float2 F1[NSHFZ / 2], dF1[NSHFZ / 2];                       // pairs over z: (z, z + 1)
#pragma unroll
  for (int zp = 0; zp < NSHFZ / 2; ++zp) {
    const float2 cz = make_float2(c.cosZ[2 * zp], c.cosZ[2 * zp + 1]), sz = make_float2(c.sinZ[2 * zp], c.sinZ[2 * zp + 1]);
    const float2 cosd = __ffma2_rn(cc2, cz, __fmul2_rn(ss2, sz));
    const float2 sind = __ffma2_rn(ss2, cz, __fmul2_rn(ncc2, sz));
    float2 B = __ffma2_rn(h2, cosd, h2);
    B.x = fmaxf(B.x, 1e-30f); B.y = fmaxf(B.y, 1e-30f);       // floor keeps lg2 finite (B^(zeta-1) -> 0 or 1)
    const float2 Bm = make_float2(ex2f(zm1 * lg2f(B.x)), ex2f(zm1 * lg2f(B.y)));   // B^(zeta-1): two MUFU ops each
    F1[zp] = __fmul2_rn(Bm, B);
    dF1[zp] = __fmul2_rn(__fmul2_rn(kd2, Bm), sind);          // dF1/du
  }
  const float Rbar = 0.5f * (uj.w + uk.w);
  float S0 = 0.f, S1 = 0.f, sV = 0.f;
#pragma unroll
  for (int a = 0; a < NSHFA; ++a) {
    const float4 g0 = gb[(2 * a) * gs], g1 = gb[(2 * a + 1) * gs];
    float2 W2 = __fmul2_rn(make_float2(g0.x, g0.y), F1[0]), V2 = __fmul2_rn(make_float2(g0.x, g0.y), dF1[0]);
    W2 = __ffma2_rn(make_float2(g0.z, g0.w), F1[1], W2); V2 = __ffma2_rn(make_float2(g0.z, g0.w), dF1[1], V2);
    W2 = __ffma2_rn(make_float2(g1.x, g1.y), F1[2], W2); V2 = __ffma2_rn(make_float2(g1.x, g1.y), dF1[2], V2);
    W2 = __ffma2_rn(make_float2(g1.z, g1.w), F1[3], W2); V2 = __ffma2_rn(make_float2(g1.z, g1.w), dF1[3], V2);
    const float Wv = W2.x + W2.y, V = V2.x + V2.y;
    const float x = Rbar - c.ShfA[a];
    const float F2 = ex2f(-c.etaA_l2e * x * x);
    const float WF = Wv * F2;
    S0 += WF; S1 = fmaf(WF, x, S1);
    sV = fmaf(V, F2, sV);
  }
  // dt/dR_ij and dt/dR_ik (through Rbar and the cut-offs), dt/du
  const float Aj = 2.0f * fk * fmaf(-c.etaA * fj, S1, dfj * S0);
  const float Ak = 2.0f * fj * fmaf(-c.etaA * fk, S1, dfk * S0);
  const float Au = 2.0f * fj * fk * sV;
  const float qj = Au / uj.w, qk = Au / uk.w;
  const float rj = Aj - qj * u, rk = Ak - qk * u;
  PairShares o;
  o.jx = fmaf(rj, uj.x, qj * uk.x); o.jy = fmaf(rj, uj.y, qj * uk.y); o.jz = fmaf(rj, uj.z, qj * uk.z);
  o.kx = fmaf(rk, uk.x, qk * uj.x); o.ky = fmaf(rk, uk.y, qk * uj.y); o.kz = fmaf(rk, uk.z, qk * uj.z);
  return o;
}

// Pair partials p_ij = dE_i/dr_j of centre ip from its dE/dAEV row (float4 piece q at gb[q * gs]) and their fixed-point
// scatter: -p_ij to every neighbour j, +sum_j p_ij to the centre itself (facc, sorted index; 64-bit integer atomics).
// All 32 lanes of the warp call this with the warp's staging (e, Pacc) and the block's pairoff table.
template <bool VIRIAL>
__device__ __forceinline__ void aev_backward_centre(const AevConst& c, const GridInfo* __restrict__ g,
                                                    const GroupInfo* __restrict__ grp, const float4* __restrict__ spos,
                                                    const uint32_t* __restrict__ rowR, const uint8_t* __restrict__ rowA, int nR,
                                                    int nA, int ip, const float4* gb, int gs,
                                                    unsigned long long* __restrict__ facc, long long* __restrict__ wcentre,
                                                    int lane, BwdEnv& e, float (*Pacc)[3], const int* pairoff) {
  const float4 ci = spos[ip];
  bwd_load_env(c, g, spos, rowR, rowA, nR, nA, ci, lane, e);

  // ---- angular: p_ij for the angular neighbours, staged in Pacc
  if (nA <= 32) {
    // Every unordered pair {j,k} is evaluated ONCE and yields both p_ij and p_ik.
    //  * within a subset of <= 16 neighbours: lanes hold neighbours; in round m lane j pairs with k = (j + m) mod n,
    //    keeps its own share and hands k's share to lane k by shuffle (j -> k is a permutation, so every lane receives
    //    exactly one share per round); the 32 / W lane groups take alternate rounds;
    //  * 17..32 neighbours: A = the first 16, B = the rest: pairs within A, pairs within B, and the cross pairs
    //    A x B with both 16-lane groups holding A and each taking every other k in B (k's share = a 16-lane butterfly).
    // All orders are fixed by (round, lane): results are bitwise reproducible.  Pacc accumulates over the passes.
    const int n = nA;
    const float zm1 = c.zeta - 1.0f;
    for (int j = lane; j < n; j += 32) { Pacc[j][0] = 0.f; Pacc[j][1] = 0.f; Pacc[j][2] = 0.f; }
    __syncwarp();
    auto rr_pass = [&](int base, int ns) {
      const int W = (ns <= 8) ? 8 : 16;
      const int NG = 32 / W, grp_id = lane / W, jl = lane & (W - 1);
      const bool act = jl < ns;
      const int nrounds = ns >> 1;
      float px = 0.f, py = 0.f, pz = 0.f;
      float4 uj = make_float4(0.f, 0.f, 1.f, 1.f);
      float fj = 0.f, dfj = 0.f;
      int sj = 0;
      if (act) { uj = e.ua[base + jl]; fj = e.fA[base + jl]; dfj = e.dfA[base + jl]; sj = e.slotA[base + jl]; }
      for (int m0 = 1; m0 <= nrounds; m0 += NG) {
        const int m = m0 + grp_id;
        const bool last_half = ((ns & 1) == 0) && (m == nrounds);   // even ns: the round m = ns/2 holds each pair twice
        const bool on = act && m <= nrounds && (!last_half || jl < nrounds);
        float qx = 0.f, qy = 0.f, qz = 0.f;
        if (on) {
          int k = jl + m;
          if (k >= ns) k -= ns;
          k += base;
          const PairShares o = pair_shares(c, zm1, gb + pairoff[sj * MAX_S + e.slotA[k]] * gs, gs, uj, fj, dfj, e.ua[k], e.fA[k],
                                           e.dfA[k]);
          px += o.jx; py += o.jy; pz += o.jz;
          qx = o.kx; qy = o.ky; qz = o.kz;
        }
        int src = jl - m;
        if (src < 0) src += ns;
        const int srcl = (grp_id * W + src) & 31;
        const float rx = __shfl_sync(0xffffffffu, qx, srcl);
        const float ry = __shfl_sync(0xffffffffu, qy, srcl);
        const float rz = __shfl_sync(0xffffffffu, qz, srcl);
        if (act && m <= nrounds && (!last_half || jl >= nrounds)) { px += rx; py += ry; pz += rz; }
      }
      for (int o = W; o < 32; o <<= 1) {
        px += __shfl_xor_sync(0xffffffffu, px, o);
        py += __shfl_xor_sync(0xffffffffu, py, o);
        pz += __shfl_xor_sync(0xffffffffu, pz, o);
      }
      if (act && grp_id == 0) { Pacc[base + jl][0] += px; Pacc[base + jl][1] += py; Pacc[base + jl][2] += pz; }
      __syncwarp();
    };
    if (n <= 16) {
      rr_pass(0, n);
    } else {
      rr_pass(0, 16);
      rr_pass(16, n - 16);
      // cross pairs A x B
      const int g2 = lane >> 4, jl = lane & 15, nb = n - 16;
      const float4 uj = e.ua[jl];
      const float fj = e.fA[jl], dfj = e.dfA[jl];
      const int sj = e.slotA[jl];
      float px = 0.f, py = 0.f, pz = 0.f;
      for (int r0 = 0; r0 < nb; r0 += 2) {
        const int r = r0 + g2, k = 16 + r;
        float qx = 0.f, qy = 0.f, qz = 0.f;
        if (r < nb) {
          const PairShares o = pair_shares(c, zm1, gb + pairoff[sj * MAX_S + e.slotA[k]] * gs, gs, uj, fj, dfj, e.ua[k], e.fA[k],
                                           e.dfA[k]);
          px += o.jx; py += o.jy; pz += o.jz;
          qx = o.kx; qy = o.ky; qz = o.kz;
        }
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) {   // k's share: sum over the 16 lanes of the group
          qx += __shfl_xor_sync(0xffffffffu, qx, o);
          qy += __shfl_xor_sync(0xffffffffu, qy, o);
          qz += __shfl_xor_sync(0xffffffffu, qz, o);
        }
        if (jl == 0 && r < nb) { Pacc[k][0] += qx; Pacc[k][1] += qy; Pacc[k][2] += qz; }
      }
      px += __shfl_xor_sync(0xffffffffu, px, 16);
      py += __shfl_xor_sync(0xffffffffu, py, 16);
      pz += __shfl_xor_sync(0xffffffffu, pz, 16);
      __syncwarp();
      if (g2 == 0) { Pacc[jl][0] += px; Pacc[jl][1] += py; Pacc[jl][2] += pz; }
    }
  } else {
  // more than 32 angular neighbours (beyond liquid-water densities): lanes x partner loop, every pair from both ends
  const int P = (nA <= 8) ? 4 : (nA <= 16) ? 2 : 1;   // lanes per neighbour
  const int JW = 32 / P;                               // neighbours per pass
  const int h = lane % P;
  for (int j0 = 0; j0 < nA; j0 += JW) {
    const int j = j0 + lane / P;
    float px = 0.f, py = 0.f, pz = 0.f;
    if (j < nA) {
      const float4 uj = e.ua[j];
      const float fj = e.fA[j], dfj = e.dfA[j];
      const int sj = e.slotA[j];
      for (int k = h; k < nA; k += P) {
        if (k == j) continue;
        const float4 uk = e.ua[k];
        const float fk = e.fA[k];
        const int sk = e.slotA[k];
        const int s1 = min(sj, sk), s2 = max(sj, sk);
        const int pidx = s1 * c.S - (s1 * (s1 - 1)) / 2 + (s2 - s1);
        const float4* gbp = gb + (size_t)grp->cpos[c.nRB + pidx] * (BLK / 4) * gs;
        const float u = fmaf(uj.x, uk.x, fmaf(uj.y, uk.y, uj.z * uk.z));
        const float cc = c.cTheta * u;
        const float ss = sqrtf(fmaxf(1.0f - cc * cc, 1e-12f));
        const float dth_du = -c.cTheta / ss;
        float F1[NSHFZ], dF1[NSHFZ];
#pragma unroll
        for (int z = 0; z < NSHFZ; ++z) {
          const float cosd = fmaf(cc, c.cosZ[z], ss * c.sinZ[z]);
          const float sind = fmaf(ss, c.cosZ[z], -cc * c.sinZ[z]);
          const float B = fmaxf(fmaf(0.5f, cosd, 0.5f), 0.f);
          float Bz, Bm;
          bpow(c, B, Bz, Bm);
          F1[z] = Bz;
          dF1[z] = (-0.5f * c.zeta * dth_du) * Bm * sind;   // dF1/du
        }
        const float Rbar = 0.5f * (uj.w + uk.w);
        float sW = 0.f, sV = 0.f;
#pragma unroll
        for (int a = 0; a < NSHFA; ++a) {
          const float4 g0 = gbp[(2 * a) * gs], g1 = gbp[(2 * a + 1) * gs];
          float W = g0.x * F1[0], V = g0.x * dF1[0];
          W = fmaf(g0.y, F1[1], W); V = fmaf(g0.y, dF1[1], V);
          W = fmaf(g0.z, F1[2], W); V = fmaf(g0.z, dF1[2], V);
          W = fmaf(g0.w, F1[3], W); V = fmaf(g0.w, dF1[3], V);
          W = fmaf(g1.x, F1[4], W); V = fmaf(g1.x, dF1[4], V);
          W = fmaf(g1.y, F1[5], W); V = fmaf(g1.y, dF1[5], V);
          W = fmaf(g1.z, F1[6], W); V = fmaf(g1.z, dF1[6], V);
          W = fmaf(g1.w, F1[7], W); V = fmaf(g1.w, dF1[7], V);
          const float x = Rbar - c.ShfA[a];
          const float F2 = ex2f(-c.etaA_l2e * x * x);
          sW = fmaf(W * F2, fmaf(-c.etaA * x, fj, dfj), sW);   // dt/dR_ij / (2 F1 fk)
          sV = fmaf(V, F2, sV);
        }
        const float Aj = 2.0f * fk * sW;
        const float Au = 2.0f * fj * fk * sV;
        const float q = Au / uj.w;
        const float r = Aj - q * u;
        px = fmaf(r, uj.x, fmaf(q, uk.x, px));
        py = fmaf(r, uj.y, fmaf(q, uk.y, py));
        pz = fmaf(r, uj.z, fmaf(q, uk.z, pz));
      }
    }
    for (int o = 1; o < P; o <<= 1) {
      px += __shfl_xor_sync(0xffffffffu, px, o);
      py += __shfl_xor_sync(0xffffffffu, py, o);
      pz += __shfl_xor_sync(0xffffffffu, pz, o);
    }
    if (j < nA && h == 0) { Pacc[j][0] = px; Pacc[j][1] = py; Pacc[j][2] = pz; }
  }
  }
  __syncwarp();

  // ---- radial + assembly: lane <-> radial neighbour
  long long ox = 0, oy = 0, oz = 0;   // sum_j p_ij in fixed point
  long long wv[9];                    // VIRIAL: sum_j p_ij (x) d_ij of this centre, 2^-32 fixed point
#pragma unroll
  for (int k = 0; k < 9; ++k) wv[k] = 0;
  for (int q0 = 0; q0 < nR; q0 += 32) {
    const int q = q0 + lane;
    if (q < nR) {
      const float4 uq = e.u[q];
      const int s = e.slotR[q];
      const float4* gr = gb + (size_t)(grp->cpos[s >> 1] * (BLK / 4) + (s & 1) * 4) * gs;
      float fc, dfc;
      cutoff(fminf(uq.w, c.Rcr), c.inv_Rcr, fc, dfc);
      const float f = c.cR * fc, df = c.cR * dfc;
      // sum over the 16 shifts of g_m d/dR [c_R exp(-eta (R - Shf_m)^2) f_C(R)], two shifts per packed instruction
      const float2 R2 = make_float2(uq.w, uq.w), hf2 = make_float2(-2.0f * c.etaR * f, -2.0f * c.etaR * f), df2 = make_float2(df, df);
      float2 coef2 = make_float2(0.f, 0.f);
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        const float4 gv = gr[v * gs];
#pragma unroll
        for (int t = 0; t < 4; t += 2) {
          const float2 x = __fadd2_rn(R2, make_float2(-c.ShfR[4 * v + t], -c.ShfR[4 * v + t + 1]));
          const float2 y = __fmul2_rn(x, x);
          const float2 ex = make_float2(ex2f(-c.etaR_l2e * y.x), ex2f(-c.etaR_l2e * y.y));
          const float2 gg = (t == 0) ? make_float2(gv.x, gv.y) : make_float2(gv.z, gv.w);
          coef2 = __ffma2_rn(__fmul2_rn(gg, ex), __ffma2_rn(x, hf2, df2), coef2);
        }
      }
      const float coef = coef2.x + coef2.y;
      float px = coef * uq.x, py = coef * uq.y, pz = coef * uq.z;
      // angular share of this neighbour, if it is one
      const int ia = e.ainv[q];
      if (ia != 255) { px += Pacc[ia][0]; py += Pacc[ia][1]; pz += Pacc[ia][2]; }
      const long long fx = to_fix(px), fy = to_fix(py), fz = to_fix(pz);
      ox += fx; oy += fy; oz += fz;
      if (VIRIAL) {   // strain derivative dE/d eps_ab = sum p_ij[a] d_ij[b], d_ij = R u
        const float pp[3] = {px, py, pz}, dd[3] = {uq.w * uq.x, uq.w * uq.y, uq.w * uq.z};
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
          for (int b = 0; b < 3; ++b) wv[3 * a + b] += __float2ll_rn(pp[a] * dd[b] * 4294967296.0f);
      }
      const int jp = (int)(rowR[q] & JMASK);
      atomicAdd(&facc[3 * (size_t)jp + 0], (unsigned long long)(-fx));
      atomicAdd(&facc[3 * (size_t)jp + 1], (unsigned long long)(-fy));
      atomicAdd(&facc[3 * (size_t)jp + 2], (unsigned long long)(-fz));
    }
  }
  for (int o = 16; o > 0; o >>= 1) { ox += shfl_xor_ll(ox, o); oy += shfl_xor_ll(oy, o); oz += shfl_xor_ll(oz, o); }
  if (lane == 0) {
    atomicAdd(&facc[3 * (size_t)ip + 0], (unsigned long long)ox);
    atomicAdd(&facc[3 * (size_t)ip + 1], (unsigned long long)oy);
    atomicAdd(&facc[3 * (size_t)ip + 2], (unsigned long long)oz);
  }
  if (VIRIAL) {
#pragma unroll
    for (int k = 0; k < 9; ++k) {
      for (int o = 16; o > 0; o >>= 1) wv[k] += shfl_xor_ll(wv[k], o);   // integer sums: exact, order free
      if (lane == 0) wcentre[9 * (size_t)ip + k] = wv[k];
    }
  }
}

// (s1, s2) -> first float4 piece of the species pair's dE/dAEV block; threads 0 .. MAX_S^2 - 1 of the block fill it
__device__ __forceinline__ void fill_pairoff(const AevConst& c, const GroupInfo* __restrict__ grp, int* pairoff) {
  if (threadIdx.x < MAX_S * MAX_S) {
    const int sa = threadIdx.x / MAX_S, sb = threadIdx.x % MAX_S;
    const int s1 = min(sa, sb), s2 = max(sa, sb);
    int off = 0;
    if (s2 < c.S) { const int cp = grp->cpos[c.nRB + s1 * c.S - (s1 * (s1 - 1)) / 2 + (s2 - s1)]; off = max(cp, 0) * (BLK / 4); }
    pairoff[threadIdx.x] = off;
  }
}

// ---------------------------------------------------------------------------------------------- a team of warps per centre
// k_small_all (small.cu) has sixteen warps for two centres; one warp per centre walks the pair rounds and the radial
// passes one after the other (measured 5.6 us of a 33 us evaluation).  Here TW warps share the centre: the leader stages
// the environment; the iterations of the pair rounds (two rounds each) are dealt out over the warps from warp 0 upwards,
// the radial passes (32 neighbours each) over the warps from the last one downwards; every warp keeps the angular shares it
// produced in an array of its own (PaccW[warp]); after a team barrier the radial warps add the shares of their neighbours
// in warp order and scatter.  Orders are fixed (and the scatter is integer): bitwise reproducible; the result differs
// from the one-warp version by rounding (another summation order of the angular shares).
template <int TW>
struct BwdTeam {
  float PaccW[TW][ACAP_MAX][3];
};

template <int TW>
__device__ __forceinline__ void aev_backward_team(const AevConst& c, const GridInfo* __restrict__ g,
                                                  const GroupInfo* __restrict__ grp, const float4* __restrict__ spos,
                                                  const uint32_t* __restrict__ rowR, const uint8_t* __restrict__ rowA, int nR,
                                                  int nA, int ip, const float4* gb, int gs,
                                                  unsigned long long* __restrict__ facc, int lane, int tw, int bar, BwdEnv& e,
                                                  BwdTeam<TW>& tm, const int* pairoff) {
  if (nA > 32) {   // beyond liquid densities: the lanes-hold-neighbours rounds below stop at 32 -- the leader alone takes the
                   // centre through the one-warp version and its general pair loop (warp-uniform branch, before any barrier)
    if (tw == 0) aev_backward_centre<false>(c, g, grp, spos, rowR, rowA, nR, nA, ip, gb, gs, facc, nullptr, lane, e, tm.PaccW[0], pairoff);
    return;
  }
  if (tw == 0) {
    const float4 ci = spos[ip];
    bwd_load_env(c, g, spos, rowR, rowA, nR, nA, ci, lane, e);
  }
  float (*Pacc)[3] = tm.PaccW[tw];
  for (int j = lane; j < nA; j += 32) { Pacc[j][0] = 0.f; Pacc[j][1] = 0.f; Pacc[j][2] = 0.f; }
  asm volatile("bar.sync %0, %1;" ::"r"(bar), "r"(TW * 32) : "memory");

  // ---- angular shares of this warp's iterations -> PaccW[tw]  (nA <= 32 here: lanes hold the neighbours)
  {
    const int n = nA;
    const float zm1 = c.zeta - 1.0f;
    int it = 0;   // running iteration number over the passes: iteration i belongs to warp i mod TW
    auto rr_pass = [&](int base, int ns) {
      const int W = (ns <= 8) ? 8 : 16;
      const int NG = 32 / W, grp_id = lane / W, jl = lane & (W - 1);
      const bool act = jl < ns;
      const int nrounds = ns >> 1;
      float px = 0.f, py = 0.f, pz = 0.f;
      float4 uj = make_float4(0.f, 0.f, 1.f, 1.f);
      float fj = 0.f, dfj = 0.f;
      int sj = 0;
      if (act) { uj = e.ua[base + jl]; fj = e.fA[base + jl]; dfj = e.dfA[base + jl]; sj = e.slotA[base + jl]; }
      bool any = false;
      for (int m0 = 1; m0 <= nrounds; m0 += NG, ++it) {
        if (it % TW != tw) continue;
        any = true;
        const int m = m0 + grp_id;
        const bool last_half = ((ns & 1) == 0) && (m == nrounds);   // even ns: the round m = ns/2 holds each pair twice
        const bool on = act && m <= nrounds && (!last_half || jl < nrounds);
        float qx = 0.f, qy = 0.f, qz = 0.f;
        if (on) {
          int k = jl + m;
          if (k >= ns) k -= ns;
          k += base;
          const PairShares o = pair_shares(c, zm1, gb + pairoff[sj * MAX_S + e.slotA[k]] * gs, gs, uj, fj, dfj, e.ua[k], e.fA[k],
                                           e.dfA[k]);
          px += o.jx; py += o.jy; pz += o.jz;
          qx = o.kx; qy = o.ky; qz = o.kz;
        }
        int src = jl - m;
        if (src < 0) src += ns;
        const int srcl = (grp_id * W + src) & 31;
        const float rx = __shfl_sync(0xffffffffu, qx, srcl);
        const float ry = __shfl_sync(0xffffffffu, qy, srcl);
        const float rz = __shfl_sync(0xffffffffu, qz, srcl);
        if (act && m <= nrounds && (!last_half || jl >= nrounds)) { px += rx; py += ry; pz += rz; }
      }
      if (any) {   // (warp-uniform)
        for (int o = W; o < 32; o <<= 1) {
          px += __shfl_xor_sync(0xffffffffu, px, o);
          py += __shfl_xor_sync(0xffffffffu, py, o);
          pz += __shfl_xor_sync(0xffffffffu, pz, o);
        }
        if (act && grp_id == 0) { Pacc[base + jl][0] += px; Pacc[base + jl][1] += py; Pacc[base + jl][2] += pz; }
        __syncwarp();
      }
    };
    if (n <= 16) {
      rr_pass(0, n);
    } else {
      rr_pass(0, 16);
      rr_pass(16, n - 16);
      // cross pairs A x B
      const int g2 = lane >> 4, jl = lane & 15, nb = n - 16;
      const float4 uj = e.ua[jl];
      const float fj = e.fA[jl], dfj = e.dfA[jl];
      const int sj = e.slotA[jl];
      float px = 0.f, py = 0.f, pz = 0.f;
      bool any = false;
      for (int r0 = 0; r0 < nb; r0 += 2, ++it) {
        if (it % TW != tw) continue;
        any = true;
        const int r = r0 + g2, k = 16 + r;
        float qx = 0.f, qy = 0.f, qz = 0.f;
        if (r < nb) {
          const PairShares o = pair_shares(c, zm1, gb + pairoff[sj * MAX_S + e.slotA[k]] * gs, gs, uj, fj, dfj, e.ua[k], e.fA[k],
                                           e.dfA[k]);
          px += o.jx; py += o.jy; pz += o.jz;
          qx = o.kx; qy = o.ky; qz = o.kz;
        }
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) {   // k's share: sum over the 16 lanes of the group
          qx += __shfl_xor_sync(0xffffffffu, qx, o);
          qy += __shfl_xor_sync(0xffffffffu, qy, o);
          qz += __shfl_xor_sync(0xffffffffu, qz, o);
        }
        if (jl == 0 && r < nb) { Pacc[k][0] += qx; Pacc[k][1] += qy; Pacc[k][2] += qz; }
      }
      if (any) {
        px += __shfl_xor_sync(0xffffffffu, px, 16);
        py += __shfl_xor_sync(0xffffffffu, py, 16);
        pz += __shfl_xor_sync(0xffffffffu, pz, 16);
        __syncwarp();
        if (g2 == 0) { Pacc[jl][0] += px; Pacc[jl][1] += py; Pacc[jl][2] += pz; }
      }
    }
  }

  // ---- radial coefficients of this warp's pass (lane <-> radial neighbour), before the barrier: they need no shares
  const int q = 32 * (TW - 1 - tw) + lane;
  const bool mine = q < nR;
  float px = 0.f, py = 0.f, pz = 0.f;
  if (mine) {
    const float4 uq = e.u[q];
    const int s = e.slotR[q];
    const float4* gr = gb + (size_t)(grp->cpos[s >> 1] * (BLK / 4) + (s & 1) * 4) * gs;
    float fc, dfc;
    cutoff(fminf(uq.w, c.Rcr), c.inv_Rcr, fc, dfc);
    const float f = c.cR * fc, df = c.cR * dfc;
    const float2 R2 = make_float2(uq.w, uq.w), hf2 = make_float2(-2.0f * c.etaR * f, -2.0f * c.etaR * f), df2 = make_float2(df, df);
    float2 coef2 = make_float2(0.f, 0.f);
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      const float4 gv = gr[v * gs];
#pragma unroll
      for (int t = 0; t < 4; t += 2) {
        const float2 x = __fadd2_rn(R2, make_float2(-c.ShfR[4 * v + t], -c.ShfR[4 * v + t + 1]));
        const float2 y = __fmul2_rn(x, x);
        const float2 ex = make_float2(ex2f(-c.etaR_l2e * y.x), ex2f(-c.etaR_l2e * y.y));
        const float2 gg = (t == 0) ? make_float2(gv.x, gv.y) : make_float2(gv.z, gv.w);
        coef2 = __ffma2_rn(__fmul2_rn(gg, ex), __ffma2_rn(x, hf2, df2), coef2);
      }
    }
    const float coef = coef2.x + coef2.y;
    px = coef * uq.x; py = coef * uq.y; pz = coef * uq.z;
  }
  asm volatile("bar.sync %0, %1;" ::"r"(bar), "r"(TW * 32) : "memory");
  if (32 * (TW - 1 - tw) >= nR) return;   // (warp-uniform: no radial pass for this warp)

  // ---- assembly: angular shares in warp order, fixed point, scatter
  long long ox = 0, oy = 0, oz = 0;
  if (mine) {
    const int ia = e.ainv[q];
    if (ia != 255) {
      float ax = 0.f, ay = 0.f, az = 0.f;
#pragma unroll
      for (int w = 0; w < TW; ++w) { ax += tm.PaccW[w][ia][0]; ay += tm.PaccW[w][ia][1]; az += tm.PaccW[w][ia][2]; }
      px += ax; py += ay; pz += az;
    }
    const long long fx = to_fix(px), fy = to_fix(py), fz = to_fix(pz);
    ox = fx; oy = fy; oz = fz;
    const int jp = (int)(rowR[q] & JMASK);
    atomicAdd(&facc[3 * (size_t)jp + 0], (unsigned long long)(-fx));
    atomicAdd(&facc[3 * (size_t)jp + 1], (unsigned long long)(-fy));
    atomicAdd(&facc[3 * (size_t)jp + 2], (unsigned long long)(-fz));
  }
  for (int o = 16; o > 0; o >>= 1) { ox += shfl_xor_ll(ox, o); oy += shfl_xor_ll(oy, o); oz += shfl_xor_ll(oz, o); }
  if (lane == 0) {
    atomicAdd(&facc[3 * (size_t)ip + 0], (unsigned long long)ox);
    atomicAdd(&facc[3 * (size_t)ip + 1], (unsigned long long)oy);
    atomicAdd(&facc[3 * (size_t)ip + 2], (unsigned long long)oz);
  }
}

}  // namespace nnp
