// aev_forward.cuh -- the per-centre AEV evaluation (K3), shared by k_aev_forward (aev.cu) and the single-kernel front
// end for small systems (small.cu).  One warp per centre (BASELINE.json north_star: "one warp per centre atom, coalesced
// float4 coordinate loads, triplet loop in registers/smem").  Formulas: SURVEY.md Appendix A "Radial block", "Angular block".
//
// Angular part, two phases per chunk of 32 triplets (all species pairs of the centre in ONE triplet index space, so the
// lanes are full whatever the species mix):
//   phase 1  lane <-> triplet: the 12 factors that do not depend on the sub-feature -- F2_a = 2 f_j f_k exp(-eta (Rbar -
//            ShfA_a)^2) (a = 0..3) and B_z^zeta (z = 0..7) -- in packed fp32 arithmetic (fma.rn.f32x2: two z per
//            instruction), stored transposed in the warp's shared staging;
//   phase 2  lane <-> sub-feature (a, z): acc += F2_a[t] * B_z[t] over the chunk's triplets, four triplets per pair of
//            128-bit shared loads.  The accumulator of a species-pair block lives in ONE register per lane and is stored
//            with one coalesced 128-byte write when the block's triplets are through.
// Against the first version (lane <-> triplet with 32 accumulators per lane and a 31-shuffle transposing butterfly per
// species pair): no butterflies, no under-filled per-pair loops, a third of the instructions.  All summation orders are
// fixed by (row order, lane id): results are bitwise reproducible.
#pragma once
#include "aev_common.cuh"

namespace nnp {

constexpr int FWD_TCH = 32;                         // triplets per chunk (one phase-1 pass)
constexpr int FWD_TP = FWD_TCH + 4;                 // pitch of the factor rows: rows land on distinct banks for LDS.128
constexpr int FWD_MAXB = MAX_S * (MAX_S + 1) / 2;   // species-pair blocks

struct FwdEnv {
  union {
    float4 u[RCAP_MAX];        // radial neighbours: unit vector and R (while the environment is being staged)
    float fac[12][FWD_TP];     // phase-1 factors of the chunk in flight: rows 0-3 F2_a, rows 4-11 B_z^zeta
  };
  float4 rad[RCAP_MAX / 2];    // radial neighbours in pairs: {R0', R1', w0, w1}, R' = R sqrt(etaR log2 e), w = c_R f_C(R; Rcr)
  float4 ua[ACAP_MAX];         // angular neighbours (subset, same order): unit vector and R
  float fA[ACAP_MAX];          // f_C(R; Rca)
  uint8_t slotR[RCAP_MAX];
  uint8_t slotA[ACAP_MAX];
  int segR[MAX_S + 1];         // the rows are sorted by species slot: segment starts
  int segA[MAX_S + 1];
  int boff[FWD_MAXB + 1];      // species-pair block b holds the triplets [boff[b], boff[b + 1]) (padded to multiples of 4)
  int2 btab[FWD_MAXB];         // x = a1 | n1 << 8 | a2 << 16 | n2 << 24,  y = compact column block | same << 8 | triplets << 16
  float binv[FWD_MAXB];        // 1 / (same ? n1 : n2)
};

// Segment starts of a species-sorted row of n entries whose slots sit in shared memory: lane s (0..MAX_S) finds the
// first entry with slot >= s by bisection (seven steps for 128 entries, the nine lanes in parallel).
template <class SlotOf>
__device__ __forceinline__ void seg_starts(int n, int lane, int* seg, SlotOf slot_of) {
  int lo = 0, hi = n;   // first q in [0, n] with slot(q) >= lane
#pragma unroll 1
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (slot_of(mid) < lane) lo = mid + 1; else hi = mid;
  }
  if (lane <= MAX_S) seg[lane] = lo;
}

// Stages the centre's environment (all lanes participate).
__device__ __forceinline__ void fwd_load_env(const AevConst& c, const GridInfo* __restrict__ g,
                                             const GroupInfo* __restrict__ grp, const float4* __restrict__ spos, const uint32_t* __restrict__ rowR,
                                             const uint8_t* __restrict__ rowA, int nR, int nA, float4 ci, int lane,
                                             FwdEnv& e) {
  float ev[9];   // cell edge vectors (orthorhombic: diagonal)
#pragma unroll
  for (int k = 0; k < 9; ++k) ev[k] = g->ev[k];
  const float rscale = sqrtf(c.etaR_l2e);
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
      const float R = d2 * rinv;
      const int slot = (__float_as_int(pj.w) >> 28) & 7;
      const float f = fmaf(0.5f, __cosf(3.14159265358979f * fminf(R, c.Rcr) * c.inv_Rcr), 0.5f);
      e.u[q] = make_float4(dx * rinv, dy * rinv, dz * rinv, R);
      float* rp = reinterpret_cast<float*>(e.rad) + ((q >> 1) << 2) + (q & 1);
      rp[0] = R * rscale; rp[2] = c.cR * f;
      e.slotR[q] = (uint8_t)slot;
    }
  }
  __syncwarp();
  seg_starts(nR, lane, e.segR, [&](int q) { return (int)e.slotR[q]; });
  for (int a0 = 0; a0 < nA; a0 += 32) {
    const int a = a0 + lane;
    if (a < nA) {
      const int p = rowA[a];
      const float4 v = e.u[p];
      e.slotA[a] = e.slotR[p];
      e.ua[a] = v;
      e.fA[a] = fmaf(0.5f, __cosf(3.14159265358979f * fminf(v.w, c.Rca) * c.inv_Rca), 0.5f);
    }
  }
  __syncwarp();
  seg_starts(nA, lane, e.segA, [&](int a) { return (int)e.slotA[a]; });
  __syncwarp();
}

// triplet t of a same-species segment of n neighbours -> (j,k) by round-robin pairing: round m = 1 + t / n,
// j = t mod n, k = (j + m) mod n; for even n the last round m = n/2 only has j < n/2.  Every unordered pair
// is visited exactly once for t in [0, n(n-1)/2).
__device__ __forceinline__ void decode_same(int t, int n, float inv_n, int& j, int& k) {
  int r = (int)(((float)t + 0.5f) * inv_n);
  j = t - r * n;
  k = j + r + 1;
  if (k >= n) k -= n;
}

// Radial block b of a centre: species 2b (columns 0-15) and 2b+1 (columns 16-31); lane & 15 <-> shift.  The two
// half-warps take alternate PAIRS of neighbours of the species' segment (one 128-bit load, packed arithmetic); the at
// most two entries of a segment that do not fill an aligned pair are taken one by one.
__device__ __forceinline__ float fwd_radial_block(const AevConst& c, const FwdEnv& e, int b, int lane) {
  const int m = lane & 15, half = lane >> 4;
  const float shf = c.ShfR[m] * sqrtf(c.etaR_l2e);
  const float2 nshf2 = make_float2(-shf, -shf);
  const float* radf = reinterpret_cast<const float*>(e.rad);
  float out = 0.f;
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int s = 2 * b + h;
    float acc = 0.f;
    const int q0 = (s < c.S) ? e.segR[s] : 0, q1 = (s < c.S) ? e.segR[s + 1] : 0;
    if (q1 > q0) {   // (warp-uniform; a species without neighbours -- most of the slots in water -- costs nothing)
      const int qa = (q0 + 1) & ~1, qb = q1 & ~1;
      float2 acc2 = make_float2(0.f, 0.f);
      for (int pp = (qa >> 1) + half; pp < (qb >> 1); pp += 2) {
        const float4 v = e.rad[pp];
        const float2 x = __fadd2_rn(make_float2(v.x, v.y), nshf2);
        const float2 t = __fmul2_rn(x, x);
        acc2 = __ffma2_rn(make_float2(v.z, v.w), make_float2(ex2f(-t.x), ex2f(-t.y)), acc2);
      }
      acc = acc2.x + acc2.y;
      int ql = -1;
      if (half == 0 && (q0 & 1) && q0 < q1) ql = q0;
      if (half == 1 && (q1 & 1) && q1 - 1 >= qa) ql = q1 - 1;
      if (ql >= 0) {
        const float* rp = radf + ((ql >> 1) << 2) + (ql & 1);
        const float x = rp[0] - shf;
        acc = fmaf(rp[2], ex2f(-x * x), acc);
      }
      acc += __shfl_xor_sync(0xffffffffu, acc, 16);
    }
    if (half == h) out = acc;
  }
  return out;
}

// Phase 1 of the angular part for the chunk of FWD_TCH triplets at c0: lane <-> triplet c0 + lane; the 12 factors go to
// fac[0..3][lane] (F2_a) and fac[4..11][lane] (B_z^zeta).  bp1 = first block that reaches into the chunk (advanced here).
__device__ __forceinline__ void fwd_factors(const AevConst& c, const FwdEnv& e, float (*fac)[FWD_TP], int npb, int c0, int lane,
                                            int& bp1) {
      const int tp = c0 + lane;
  while (e.boff[bp1 + 1] <= c0) ++bp1;             // first block that reaches into this chunk (warp-uniform)
  int b = bp1;
  for (int bb = bp1 + 1; bb < npb && e.boff[bb] < c0 + FWD_TCH; ++bb) if (tp >= e.boff[bb]) b = bb;
  const int2 ent = e.btab[b];
  const int t = tp - e.boff[b], T = ent.y >> 16;
  const int a1 = ent.x & 255, a2 = (ent.x >> 16) & 255;
  const bool live = t < T;
  int j = a1, k = a1;
  if (live) {
    // same species: round-robin pairing over the n1 neighbours (decode_same); else the n1 x n2 grid, k fastest
    const bool same = (ent.y & 256) != 0;
    const int n = same ? ((ent.x >> 8) & 255) : ((ent.x >> 24) & 255);
    const int r = (int)(((float)t + 0.5f) * e.binv[b]);
    const int rem = t - r * n;
    int ks = rem + r + 1;
    if (ks >= n) ks -= n;
    j = a1 + (same ? rem : r);
    k = same ? a1 + ks : a2 + rem;
  }
  const float4 uj = e.ua[j], uk = e.ua[k];
  const float u = fmaf(uj.x, uk.x, fmaf(uj.y, uk.y, uj.z * uk.z));
  const float cc = c.cTheta * u;
  const float ss = sqrtf(fmaxf(1.0f - cc * cc, 0.f));
  const float Rbar = 0.5f * (uj.w + uk.w);
  const float ff2 = live ? 2.0f * e.fA[j] * e.fA[k] : 0.f;
#pragma unroll
  for (int a = 0; a < NSHFA; a += 2) {
    const float2 x = __fadd2_rn(make_float2(Rbar, Rbar), make_float2(-c.ShfA[a], -c.ShfA[a + 1]));
    const float2 y = __fmul2_rn(x, x);
    const float2 F = __fmul2_rn(make_float2(ex2f(-c.etaA_l2e * y.x), ex2f(-c.etaA_l2e * y.y)), make_float2(ff2, ff2));
    fac[a][lane] = F.x; fac[a + 1][lane] = F.y;
  }
  if (c.zeta_is_32) {
    const float2 cc2 = make_float2(cc, cc), ss2 = make_float2(ss, ss), h2 = make_float2(0.5f, 0.5f);
#pragma unroll
    for (int z = 0; z < NSHFZ; z += 2) {
      const float2 cd = __ffma2_rn(cc2, make_float2(c.cosZ[z], c.cosZ[z + 1]), __fmul2_rn(ss2, make_float2(c.sinZ[z], c.sinZ[z + 1])));
      const float2 B = __ffma2_rn(h2, cd, h2);      // (1 + cos(theta - ShfZ)) / 2; B^32 >= 0 whatever the rounding of B
      const float2 B2 = __fmul2_rn(B, B), B4 = __fmul2_rn(B2, B2), B8 = __fmul2_rn(B4, B4), B16 = __fmul2_rn(B8, B8);
      const float2 B32 = __fmul2_rn(B16, B16);
      fac[4 + z][lane] = B32.x; fac[5 + z][lane] = B32.y;
    }
  } else {
#pragma unroll
    for (int z = 0; z < NSHFZ; ++z) {
      const float B = fmaf(0.5f, fmaf(cc, c.cosZ[z], ss * c.sinZ[z]), 0.5f);
      float Bz, Bm;
      bpow(c, fmaxf(B, 0.f), Bz, Bm);
      fac[4 + z][lane] = Bz;
    }
  }
}

// Species-pair block table of a centre (lane b <-> b-th pair of species present, i1 <= i2): e.btab / e.binv / e.boff.
__device__ __forceinline__ void fwd_block_table(const AevConst& c, const GroupInfo* __restrict__ grp, FwdEnv& e, int np, int npb,
                                                int lane) {
  int run = 0;
  for (int b0 = 0; b0 < npb; b0 += 32) {
    const int b = b0 + lane;
    int T = 0;
    int2 ent = make_int2(0, 0);
    float inv = 0.f;
    if (b < npb) {
      int p = b, i1 = 0;
      while (p >= np - i1) { p -= np - i1; ++i1; }
      const int s1 = grp->pres[i1], s2 = grp->pres[i1 + p];
      const int a1 = e.segA[s1], n1 = e.segA[s1 + 1] - a1, a2 = e.segA[s2], n2 = e.segA[s2 + 1] - a2;
      const bool same = (s1 == s2);
      T = same ? (n1 * (n1 - 1)) / 2 : n1 * n2;
      const int cp = grp->cpos[c.nRB + s1 * c.S - (s1 * (s1 - 1)) / 2 + (s2 - s1)];
      ent = make_int2(a1 | (n1 << 8) | (a2 << 16) | (n2 << 24), (cp & 255) | ((same ? 1 : 0) << 8) | (T << 16));
      inv = 1.0f / (float)max(same ? n1 : n2, 1);
    }
    int inc = (T + 3) & ~3;
    const int own = inc;
    for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
    if (b < npb) { e.btab[b] = ent; e.binv[b] = inv; e.boff[b] = run + inc - own; }
    run += __shfl_sync(0xffffffffu, inc, 31);
  }
  if (lane == 0) e.boff[npb] = run;
}

// AEV row of centre ip (sorted index) from its neighbour rows rowR / rowA; all 32 lanes of the warp call this with the
// warp's FwdEnv staging.  (spos, g, grp and the rows may live in shared memory: small.cu.)
__device__ __forceinline__ void aev_forward_centre(const AevConst& c, const GridInfo* __restrict__ g,
                                                   const GroupInfo* __restrict__ grp, const float4* __restrict__ spos,
                                                   const uint32_t* __restrict__ rowR, const uint8_t* __restrict__ rowA,
                                                   int nR, int nA, int ip, float* __restrict__ aev, int lane, FwdEnv& e) {
  const float4 ci = spos[ip];
  const int si = (__float_as_int(ci.w) >> 28) & 7;
  fwd_load_env(c, g, grp, spos, rowR, rowA, nR, nA, ci, lane, e);
  const int Kc = grp->Kc;
  float* __restrict__ row = aev + (size_t)(ip + grp->pad_shift[si]) * Kc;

  const int np = grp->npres;
  const int npb = np * (np + 1) / 2;
  fwd_block_table(c, grp, e, np, npb, lane);

  // ---- radial
  {
    for (int b = 0; b < c.nRB; ++b) {
      const int cp = grp->cpos[b];
      if (cp < 0) continue;
      row[cp * BLK + lane] = fwd_radial_block(c, e, b, lane);
    }
  }
  // in dense-K mode the angular blocks of absent species pairs are zero-filled (same lane, same address as any later
  // store: program order keeps the later value)
  if (grp->nblk == c.nblk_full && np < c.S)
    for (int b = c.nRB; b < c.nblk_full; ++b) row[grp->cpos[b] * BLK + lane] = 0.f;
  __syncwarp();   // the staging of the radial neighbours (u) is dead from here on: the factor rows take its place

  // ---- angular
  const int Ttot = e.boff[npb];
  const int fa = lane >> 3, fz = lane & 7;
  const float* __restrict__ f2row = e.fac[fa];
  const float* __restrict__ bzrow = e.fac[4 + fz];
  float2 acc2 = make_float2(0.f, 0.f);
  int bcur = 0;   // block the phase-2 accumulator belongs to
  int bp1 = 0;    // first block of the chunk phase 1 is working on
  for (int c0 = 0; c0 < Ttot; c0 += FWD_TCH) {
    fwd_factors(c, e, e.fac, npb, c0, lane, bp1);
    __syncwarp();
    // phase 2: lane <-> sub-feature (a, z): acc += F2_a[t] * B_z[t]; block boundaries are multiples of 4
    {
      int q = c0;
      const int qend = min(c0 + FWD_TCH, Ttot);
      while (q < qend) {
        while (e.boff[bcur + 1] <= q) {   // block through (or empty): store it
          row[(e.btab[bcur].y & 255) * BLK + lane] = acc2.x + acc2.y;
          acc2 = make_float2(0.f, 0.f); ++bcur;
        }
        const int bend = min(e.boff[bcur + 1], qend);
        const float4* fp = reinterpret_cast<const float4*>(f2row + (q - c0));
        const float4* bp = reinterpret_cast<const float4*>(bzrow + (q - c0));
        const int n4 = (bend - q) >> 2;
#pragma unroll 2
        for (int i = 0; i < n4; ++i) {
          const float4 f = fp[i], bz = bp[i];
          acc2 = __ffma2_rn(make_float2(f.x, f.y), make_float2(bz.x, bz.y), acc2);
          acc2 = __ffma2_rn(make_float2(f.z, f.w), make_float2(bz.z, bz.w), acc2);
        }
        q = bend;
      }
    }
    __syncwarp();
  }
  for (; bcur < npb; ++bcur) {   // the last block and the empty ones behind it
    row[(e.btab[bcur].y & 255) * BLK + lane] = acc2.x + acc2.y;
    acc2 = make_float2(0.f, 0.f);
  }
}

// ---------------------------------------------------------------------------------------------- a team of warps per centre
// The single-kernel evaluation of small systems (small.cu, k_small_all) has two centres per CTA and sixteen warps: one
// warp per centre leaves the rest idle while it walks through ~2000 dependent-latency-bound instructions (measured:
// 7.3 us of a 37 us evaluation).  Here TW warps share one centre: the leader stages the environment and the block table;
// the radial blocks and the chunks of 32 triplets are then dealt out over the team; every warp adds its chunks' sums
// into accumulators of its own (team.acc[warp]), and the blocks are finished by adding the warps' accumulators in warp
// order -- fixed orders throughout, so the row is bitwise reproducible (it differs from the one-warp row by rounding).
template <int TW>
struct alignas(16) FwdTeam {
  float fac[TW][12][FWD_TP];         // phase-1 factors, one staging per warp (rows read with 128-bit loads)
  float acc[TW][FWD_MAXB][32];       // per warp: sub-feature sums of the blocks its chunks touched
};

__device__ __forceinline__ void team_bar(int id, int nthreads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }

// All TW warps of the team call this (tw = warp within the team, 0 = leader, which alone needs the rows and counts);
// bar = a named barrier of the CTA that belongs to this team.
template <int TW>
__device__ __forceinline__ void aev_forward_team(const AevConst& c, const GridInfo* __restrict__ g,
                                                 const GroupInfo* __restrict__ grp, const float4* __restrict__ spos,
                                                 const uint32_t* __restrict__ rowR, const uint8_t* __restrict__ rowA, int nR,
                                                 int nA, int ip, float* __restrict__ aev, int lane, int tw, int bar, FwdEnv& e,
                                                 FwdTeam<TW>& tm) {
  const float4 ci = spos[ip];
  const int si = (__float_as_int(ci.w) >> 28) & 7;
  const int Kc = grp->Kc;
  float* __restrict__ row = aev + (size_t)(ip + grp->pad_shift[si]) * Kc;
  const int np = grp->npres;
  const int npb = np * (np + 1) / 2;
  if (tw == 0) {
    fwd_load_env(c, g, grp, spos, rowR, rowA, nR, nA, ci, lane, e);
    fwd_block_table(c, grp, e, np, npb, lane);
    // dense-K: the angular blocks of absent species pairs are zero (before the barrier: the blocks present are stored after it)
    if (grp->nblk == c.nblk_full && np < c.S)
      for (int b = c.nRB; b < c.nblk_full; ++b) row[grp->cpos[b] * BLK + lane] = 0.f;
  }
  team_bar(bar, TW * 32);
  // ---- radial blocks: from the last warp downwards (the first warps have the most chunks)
  {
    int idx = 0;
    for (int b = 0; b < c.nRB; ++b) {
      const int cp = grp->cpos[b];
      if (cp < 0) continue;
      if (TW - 1 - (idx % TW) == tw) row[cp * BLK + lane] = fwd_radial_block(c, e, b, lane);
      ++idx;
    }
  }
  // ---- angular: chunk i of 32 triplets goes to warp i mod TW
  for (int b = 0; b < npb; ++b) tm.acc[tw][b][lane] = 0.f;
  const int Ttot = e.boff[npb];
  const int fa = lane >> 3, fz = lane & 7;
  const float* __restrict__ f2row = tm.fac[tw][fa];
  const float* __restrict__ bzrow = tm.fac[tw][4 + fz];
  int bp1 = 0, bcur = 0;
  for (int c0 = FWD_TCH * tw; c0 < Ttot; c0 += FWD_TCH * TW) {
    fwd_factors(c, e, tm.fac[tw], npb, c0, lane, bp1);
    __syncwarp();
    int q = c0;
    const int qend = min(c0 + FWD_TCH, Ttot);
    while (q < qend) {
      while (e.boff[bcur + 1] <= q) ++bcur;
      const int bend = min(e.boff[bcur + 1], qend);
      const float4* fp = reinterpret_cast<const float4*>(f2row + (q - c0));
      const float4* bp = reinterpret_cast<const float4*>(bzrow + (q - c0));
      const int n4 = (bend - q) >> 2;
      float2 acc2 = make_float2(0.f, 0.f);
#pragma unroll 2
      for (int i = 0; i < n4; ++i) {
        const float4 f = fp[i], bz = bp[i];
        acc2 = __ffma2_rn(make_float2(f.x, f.y), make_float2(bz.x, bz.y), acc2);
        acc2 = __ffma2_rn(make_float2(f.z, f.w), make_float2(bz.z, bz.w), acc2);
      }
      tm.acc[tw][bcur][lane] += acc2.x + acc2.y;
      q = bend;
    }
    __syncwarp();
  }
  team_bar(bar, TW * 32);
  for (int b = tw; b < npb; b += TW) {
    float v = 0.f;
#pragma unroll
    for (int w = 0; w < TW; ++w) v += tm.acc[w][b][lane];
    row[(e.btab[b].y & 255) * BLK + lane] = v;
  }
}

}  // namespace nnp
