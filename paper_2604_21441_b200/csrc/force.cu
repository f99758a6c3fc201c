// force.cu -- K7 + K8 of SURVEY.md section 8.a: chain rule dE/dAEV -> pair partials p_ij = dE_i/dr_j, and the
// deterministic force assembly F_a = sum_j (p_aj - p_ja)  (eq. 2 F = -grad E;
// BASELINE.json north_star stage (4); formulas SURVEY.md Appendix A "Forces").
//
// K7: one warp per centre.  Radial: lane <-> neighbour.  Angular: lanes hold the angular neighbours; every unordered
// triplet {j,k} is evaluated ONCE (round-robin pairing: in round m lane j pairs with k = (j + m) mod n), lane j keeps
// its own share p_ij and hands p_ik to lane k by shuffle; more than 32 angular neighbours fall back to a loop that
// visits every pair from both ends.
// K8: p_ij is converted to 2^-40 fixed point and accumulated with 64-bit INTEGER atomics (integer addition is
// associative, so the result does not depend on the arrival order): forces are bitwise reproducible.
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

template <bool VIRIAL>
// 3 blocks per SM: 80 registers.  (At 4 blocks / 64 registers the packed-arithmetic version spills ~250 bytes per thread
// inside the triplet loop -- local-memory loads are long-scoreboard stalls: 95 us against 86 us.)
__global__ void __launch_bounds__(AEV_WARPS * 32, 3)
k_aev_backward(AevConst c, const GridInfo* __restrict__ g, const GroupInfo* __restrict__ grp,
               const float4* __restrict__ spos, const uint32_t* __restrict__ nbrR, const uint8_t* __restrict__ nbrA,
               const int* __restrict__ cntR, const int* __restrict__ cntA, int n_ml, int rcap, int acap,
               const float* daev, unsigned long long* __restrict__ facc, long long* __restrict__ wcentre,
               const int* tile_done, int done_target, int* __restrict__ flags) {
  __shared__ BwdEnv env[AEV_WARPS];
  __shared__ int timed_out;
  __shared__ float Pacc[AEV_WARPS][ACAP_MAX][3];
  __shared__ int pairoff[MAX_S * MAX_S];   // (s1, s2) -> first float4 piece of the pair's dE/dAEV block
  pdl_trigger();
  if (!tile_done) pdl_wait();   // with per-tile flags the MLP kernel is NOT awaited as a whole (see below)
  if (threadIdx.x == 0) timed_out = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (threadIdx.x < MAX_S * MAX_S) {
    const int sa = threadIdx.x / MAX_S, sb = threadIdx.x % MAX_S;
    const int s1 = min(sa, sb), s2 = max(sa, sb);
    int off = 0;
    if (s2 < c.S) { const int cp = grp->cpos[c.nRB + s1 * c.S - (s1 * (s1 - 1)) / 2 + (s2 - s1)]; off = max(cp, 0) * (BLK / 4); }
    pairoff[threadIdx.x] = off;
  }
  // Overlap with the MLP kernel (programmatic dependent launch): this grid may start while the persistent MLP CTAs
  // are still on their last tiles; a centre only needs ITS OWN row of dE/dAEV, so the block waits for the completion
  // flags of its centres' 128-row tiles (released by the MLP epilogue after the tile's last store) instead of the
  // whole kernel.  Thread t looks after centre t and polls only where the tile changes (the rows of a block are
  // contiguous: one poller per block almost always -- thousands of polling warps saturate the L2 slice that holds
  // the flags and slow the MLP's weight stream down).  dE/dAEV is read through ordinary (coherent) loads.
  if (tile_done && threadIdx.x < AEV_WARPS) {
    const int ipw = blockIdx.x * AEV_WARPS + threadIdx.x;
    if (ipw < n_ml) {
      const int tw = (ipw + grp->pad_shift[(__float_as_int(spos[ipw].w) >> 28) & 7]) / TILE_M;
      bool poll = true;
      if (threadIdx.x > 0) poll = tw != (ipw - 1 + grp->pad_shift[(__float_as_int(spos[ipw - 1].w) >> 28) & 7]) / TILE_M;
      if (poll) {
        int seen, spins = 0;
        do {
          asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(seen) : "l"(tile_done + tw) : "memory");
          if (seen < done_target) __nanosleep(500);
        } while (seen < done_target && ++spins < (1 << 22));   // ~2 s: a flag that never comes must not hang the GPU
        // ... and must not pass silently either: the evaluation is flagged (nnp_status -> NNP_ERR_CUDA) and the block's
        // centres are skipped -- their dE/dAEV rows are not there
        if (seen < done_target) { atomicOr(flags, FLAG_TIMEOUT); atomicExch(&timed_out, 1); }
      }
    }
  }
  __syncthreads();
  if (timed_out) return;
  const int ip = blockIdx.x * AEV_WARPS + w;
  if (ip >= n_ml) return;
  BwdEnv& e = env[w];
  const float4 ci = spos[ip];
  const int si = (__float_as_int(ci.w) >> 28) & 7;
  const int nR = cntR[ip], nA = cntA[ip];
  const uint32_t* __restrict__ rowR = nbrR + (size_t)ip * rcap;
  const int Kc = grp->Kc;
  // row of dE/dAEV in the piece-major tile layout: float4 piece q of this row = gb[q * gs].  (Read through L1 where it
  // is needed: staging the row in shared memory first was measured twice -- round 1 and again with the packed
  // arithmetic, 86 -> 92 us -- and lost both times: extra registers across the gather and bank conflicts between the
  // lanes' different species-pair blocks.)
  const size_t grow = (size_t)(ip + grp->pad_shift[si]);
  const float4* gb = reinterpret_cast<const float4*>(daev + daev_off(grow, 0, Kc));
  constexpr int gs = TILE_M;
  bwd_load_env(c, g, spos, rowR, nbrA + (size_t)ip * acap, nR, nA, ci, lane, e);

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
    for (int j = lane; j < n; j += 32) { Pacc[w][j][0] = 0.f; Pacc[w][j][1] = 0.f; Pacc[w][j][2] = 0.f; }
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
      if (act && grp_id == 0) { Pacc[w][base + jl][0] += px; Pacc[w][base + jl][1] += py; Pacc[w][base + jl][2] += pz; }
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
        if (jl == 0 && r < nb) { Pacc[w][k][0] += qx; Pacc[w][k][1] += qy; Pacc[w][k][2] += qz; }
      }
      px += __shfl_xor_sync(0xffffffffu, px, 16);
      py += __shfl_xor_sync(0xffffffffu, py, 16);
      pz += __shfl_xor_sync(0xffffffffu, pz, 16);
      __syncwarp();
      if (g2 == 0) { Pacc[w][jl][0] += px; Pacc[w][jl][1] += py; Pacc[w][jl][2] += pz; }
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
    if (j < nA && h == 0) { Pacc[w][j][0] = px; Pacc[w][j][1] = py; Pacc[w][j][2] = pz; }
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
      if (ia != 255) { px += Pacc[w][ia][0]; py += Pacc[w][ia][1]; pz += Pacc[w][ia][2]; }
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

// K8b: facc (sorted order, fixed point; = sum_j (p_aj - p_ja) = +F) -> forces in the caller's atom order, and
// E = sum_i E_i in a fixed order: fp64 block partials (shuffle tree), then the last block to finish adds the
// partials in index order -- no floating-point atomics, bitwise reproducible.
__global__ void __launch_bounds__(256)
k_force_out(const float4* __restrict__ spos, const unsigned long long* __restrict__ facc,
            const int32_t* __restrict__ ml, int n_ml, float* __restrict__ forces, const GroupInfo* __restrict__ grp,
            const float* __restrict__ e_atom, double* __restrict__ epart, unsigned int* __restrict__ ticket,
            double* __restrict__ energy, const long long* __restrict__ wcentre, long long* __restrict__ wblk,
            double* __restrict__ virial, double e_scale, double f_scale) {
  __shared__ double wsum[8];
  __shared__ long long vsum[8][9];
  __shared__ bool last;
  pdl_trigger();
  pdl_wait();
  const int ip = blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
  double e = 0.0;
  if (ip < n_ml) {
    const int w = __float_as_int(spos[ip].w);
    const int a = w & 0x0fffffff, slot = (w >> 28) & 7;
    const size_t o = ml ? (size_t)ml[a] : (size_t)a;
    const double sc = f_scale / 1099511627776.0;   // fixed point -> eV/Angstrom -> caller units
#pragma unroll
    for (int d = 0; d < 3; ++d) forces[3 * o + d] = (float)((double)(long long)facc[3 * (size_t)ip + d] * sc);
    e = (double)e_atom[ip + grp->pad_shift[slot]];
  }
  for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
  if (lane == 0) wsum[wp] = e;
  if (virial) {   // per-centre strain derivatives (fixed point) -> block partial
#pragma unroll
    for (int k = 0; k < 9; ++k) {
      long long v = (ip < n_ml) ? wcentre[9 * (size_t)ip + k] : 0ll;
      for (int o = 16; o > 0; o >>= 1) v += shfl_xor_ll(v, o);
      if (lane == 0) vsum[wp][k] = v;
    }
  }
  __syncthreads();
  if (virial && threadIdx.x < 9) {
    long long v = 0;
    for (int i = 0; i < 8; ++i) v += vsum[i][threadIdx.x];
    wblk[9 * (size_t)blockIdx.x + threadIdx.x] = v;
  }
  if (virial) __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int i = 0; i < 8; ++i) t += wsum[i];
    epart[blockIdx.x] = t;
    __threadfence();
    last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (!last || wp != 0) return;
  __threadfence();
  double t = 0.0;
  for (int i = lane; i < (int)gridDim.x; i += 32) t += __ldcg(epart + i);
  for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
  if (virial && lane < 9) {
    long long v = 0;
    for (int i = 0; i < (int)gridDim.x; ++i) v += __ldcg(wblk + 9 * (size_t)i + lane);
    virial[lane] = (double)v * (e_scale / 4294967296.0);
  }
  if (lane == 0) { *energy = t * e_scale; *ticket = 0u; }
}

int launch_force_stage(nnp_workspace* ws, int64_t n_atoms, int64_t n_ml, const int32_t* d_ml, double* d_energy,
                       float* d_forces) {
  const nnp_model* m = ws->model;
  int nl = 0;
  // (rows of non-ML atoms are +0.0f: nnp_eval clears the force array before the first kernel when a subset is given)
  if (n_ml > 0) {
    const int nb = (int)((n_ml + AEV_WARPS - 1) / AEV_WARPS);
    // after the tcgen05 MLP kernel the launch is a programmatic dependent launch: blocks start on the SMs the
    // persistent MLP CTAs have left and wait per tile (see the kernel); stage profiling keeps the stages apart
    const int* done = ws->profiling ? nullptr : ws->tile_done;
    if (ws->d_virial)
      launch_pdl(done != nullptr, ws->stream, k_aev_backward<true>, dim3(nb), dim3(AEV_WARPS * 32), 0, m->aev, ws->grid,
                 ws->groups, ws->spos, ws->nbrR, ws->nbrA, ws->cntR, ws->cntA, (int)n_ml, ws->rcap, ws->acap, ws->daev,
                 ws->facc, ws->wcentre, done, ws->tile_done_target, ws->flags);
    else
      launch_pdl(done != nullptr, ws->stream, k_aev_backward<false>, dim3(nb), dim3(AEV_WARPS * 32), 0, m->aev, ws->grid,
                 ws->groups, ws->spos, ws->nbrR, ws->nbrA, ws->cntR, ws->cntA, (int)n_ml, ws->rcap, ws->acap, ws->daev,
                 ws->facc, nullptr, done, ws->tile_done_target, ws->flags);
    prof_mark(ws, 4);
    launch_pdl(!ws->profiling, ws->stream, k_force_out, dim3((unsigned)((n_ml + 255) / 256)), dim3(256), 0, ws->spos, ws->facc,
               d_ml, (int)n_ml, d_forces, ws->groups, ws->e_atom, ws->epart, ws->ticket, d_energy, ws->wcentre, ws->wblk,
               ws->d_virial, ws->e_scale, ws->e_scale * ws->len_scale);
    nl += 2;
  } else {
    cudaMemsetAsync(d_energy, 0, sizeof(double), ws->stream);
    if (ws->d_virial) cudaMemsetAsync(ws->d_virial, 0, 9 * sizeof(double), ws->stream);
  }
  return nl;
}

}  // namespace nnp
