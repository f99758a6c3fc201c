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
struct PairShares { float jx, jy, jz, kx, ky, kz; };
__device__ __forceinline__ PairShares pair_shares(const AevConst& c, float zm1, const float4* gb, float4 uj,
                                                  float fj, float dfj, float4 uk, float fk, float dfk) {
  const float u = fmaf(uj.x, uk.x, fmaf(uj.y, uk.y, uj.z * uk.z));
  const float cc = c.cTheta * u;
  const float ss = sqrtf(fmaxf(1.0f - cc * cc, 1e-12f));
  const float kd = 0.5f * c.zeta * c.cTheta / ss;            // -0.5 zeta dtheta/du
  float F1[NSHFZ], dF1[NSHFZ];
#pragma unroll
  for (int z = 0; z < NSHFZ; ++z) {
    const float cosd = fmaf(cc, c.cosZ[z], ss * c.sinZ[z]);
    const float sind = fmaf(ss, c.cosZ[z], -cc * c.sinZ[z]);
    const float B = fmaxf(fmaf(0.5f, cosd, 0.5f), 1e-30f);    // floor keeps lg2 finite (B^(zeta-1) -> 0 or 1)
    const float Bm = ex2f(zm1 * lg2f(B));                     // B^(zeta-1): two MUFU ops
    F1[z] = Bm * B;
    dF1[z] = kd * Bm * sind;                                  // dF1/du
  }
  const float Rbar = 0.5f * (uj.w + uk.w);
  float S0 = 0.f, S1 = 0.f, sV = 0.f;
#pragma unroll
  for (int a = 0; a < NSHFA; ++a) {
    const float4 g0 = gb[(2 * a) * TILE_M], g1 = gb[(2 * a + 1) * TILE_M];
    float Wv = g0.x * F1[0], V = g0.x * dF1[0];
    Wv = fmaf(g0.y, F1[1], Wv); V = fmaf(g0.y, dF1[1], V);
    Wv = fmaf(g0.z, F1[2], Wv); V = fmaf(g0.z, dF1[2], V);
    Wv = fmaf(g0.w, F1[3], Wv); V = fmaf(g0.w, dF1[3], V);
    Wv = fmaf(g1.x, F1[4], Wv); V = fmaf(g1.x, dF1[4], V);
    Wv = fmaf(g1.y, F1[5], Wv); V = fmaf(g1.y, dF1[5], V);
    Wv = fmaf(g1.z, F1[6], Wv); V = fmaf(g1.z, dF1[6], V);
    Wv = fmaf(g1.w, F1[7], Wv); V = fmaf(g1.w, dF1[7], V);
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
__global__ void __launch_bounds__(AEV_WARPS * 32, 32 / AEV_WARPS)
k_aev_backward(AevConst c, const GridInfo* __restrict__ g, const GroupInfo* __restrict__ grp,
               const float4* __restrict__ spos, const uint32_t* __restrict__ nbrR, const uint8_t* __restrict__ nbrA,
               const int* __restrict__ cntR, const int* __restrict__ cntA, int n_ml, int rcap, int acap,
               const float* daev, unsigned long long* __restrict__ facc, long long* __restrict__ wcentre,
               const int* tile_done, int done_target, int* __restrict__ flags) {
  __shared__ WarpEnv env[AEV_WARPS];
  __shared__ int timed_out;
  __shared__ float Pacc[AEV_WARPS][ACAP_MAX][3];
  __shared__ int pairoff[MAX_S * MAX_S];   // (s1, s2) -> first float4 piece of the pair's dE/dAEV block, times TILE_M
  pdl_trigger();
  if (!tile_done) pdl_wait();   // with per-tile flags the MLP kernel is NOT awaited as a whole (see below)
  if (threadIdx.x == 0) timed_out = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (threadIdx.x < MAX_S * MAX_S) {
    const int sa = threadIdx.x / MAX_S, sb = threadIdx.x % MAX_S;
    const int s1 = min(sa, sb), s2 = max(sa, sb);
    int off = 0;
    if (s2 < c.S) { const int cp = grp->cpos[c.nRB + s1 * c.S - (s1 * (s1 - 1)) / 2 + (s2 - s1)]; off = max(cp, 0) * (BLK / 4) * TILE_M; }
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
  WarpEnv& e = env[w];
  const float4 ci = spos[ip];
  const int si = (__float_as_int(ci.w) >> 28) & 7;
  const int nR = cntR[ip], nA = cntA[ip];
  const uint32_t* __restrict__ rowR = nbrR + (size_t)ip * rcap;
  load_env(c, g, spos, rowR, nbrA + (size_t)ip * acap, nR, nA, ci, lane, e);
  const int Kc = grp->Kc;
  // row of dE/dAEV in the piece-major tile layout: float4 piece q of this row = gi4[q * TILE_M]
  const size_t grow = (size_t)(ip + grp->pad_shift[si]);
  const float4* gi4 = reinterpret_cast<const float4*>(daev + daev_off(grow, 0, Kc));

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
          const PairShares o = pair_shares(c, zm1, gi4 + pairoff[sj * MAX_S + e.slotA[k]], uj, fj, dfj, e.ua[k], e.fA[k],
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
          const PairShares o = pair_shares(c, zm1, gi4 + pairoff[sj * MAX_S + e.slotA[k]], uj, fj, dfj, e.ua[k], e.fA[k],
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
        const float4* gb = gi4 + (size_t)grp->cpos[c.nRB + pidx] * (BLK / 4) * TILE_M;
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
          const float4 g0 = gb[(2 * a) * TILE_M], g1 = gb[(2 * a + 1) * TILE_M];
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
      const float4* gr = gi4 + (size_t)(grp->cpos[s >> 1] * (BLK / 4) + (s & 1) * 4) * TILE_M;
      const float f = e.wR[q];   // c_R f_C
      float fc, dfc;
      cutoff(fminf(uq.w, c.Rcr), c.inv_Rcr, fc, dfc);
      const float df = c.cR * dfc;
      float coef = 0.f;
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        const float4 gv = gr[v * TILE_M];
        const float gg[4] = {gv.x, gv.y, gv.z, gv.w};
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          const float x = uq.w - c.ShfR[4 * v + t];
          const float ex = ex2f(-c.etaR_l2e * x * x);
          coef = fmaf(gg[t] * ex, fmaf(-2.0f * c.etaR * x, f, df), coef);
        }
      }
      float px = coef * uq.x, py = coef * uq.y, pz = coef * uq.z;
      // angular share of this neighbour, if it is one: binary search of q in posA
      int lo = 0, hi = nA;
      while (lo < hi) { int mid = (lo + hi) >> 1; if (e.posA[mid] < q) lo = mid + 1; else hi = mid; }
      if (lo < nA && e.posA[lo] == q) { px += Pacc[w][lo][0]; py += Pacc[w][lo][1]; pz += Pacc[w][lo][2]; }
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
