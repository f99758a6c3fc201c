// aev_forward.cuh -- the per-centre AEV evaluation (K3), shared by k_aev_forward (aev.cu) and the single-kernel front
// end for small systems (small.cu).  One warp per centre; see aev.cu for the layout notes.
#pragma once
#include "aev_common.cuh"

namespace nnp {

// transposing butterfly: on return acc[0] of lane l = sum over lanes of acc[l]
__device__ __forceinline__ float reduce32(float (&acc)[32], int lane) {
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const bool up = lane & 16;
    const float send = up ? acc[i] : acc[i + 16], keep = up ? acc[i + 16] : acc[i];
    acc[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const bool up = lane & 8;
    const float send = up ? acc[i] : acc[i + 8], keep = up ? acc[i + 8] : acc[i];
    acc[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const bool up = lane & 4;
    const float send = up ? acc[i] : acc[i + 4], keep = up ? acc[i + 4] : acc[i];
    acc[i] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
  }
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    const bool up = lane & 2;
    const float send = up ? acc[i] : acc[i + 2], keep = up ? acc[i + 2] : acc[i];
    acc[i] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
  }
  {
    const bool up = lane & 1;
    const float send = up ? acc[0] : acc[1], keep = up ? acc[1] : acc[0];
    acc[0] = keep + __shfl_xor_sync(0xffffffffu, send, 1);
  }
  return acc[0];
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

// AEV row of centre ip (sorted index) from its neighbour rows rowR / rowA; all 32 lanes of the warp call this with the
// warp's WarpEnv staging.  (spos, g, grp and the rows may live in shared memory: small.cu.)
__device__ __forceinline__ void aev_forward_centre(const AevConst& c, const GridInfo* __restrict__ g,
                                                   const GroupInfo* __restrict__ grp, const float4* __restrict__ spos,
                                                   const uint32_t* __restrict__ rowR, const uint8_t* __restrict__ rowA,
                                                   int nR, int nA, int ip, float* __restrict__ aev, int lane, WarpEnv& e) {
  const float4 ci = spos[ip];
  const int si = (__float_as_int(ci.w) >> 28) & 7;
  load_env(c, g, spos, rowR, rowA, nR, nA, ci, lane, e);
  const int Kc = grp->Kc;
  float* __restrict__ row = aev + (size_t)(ip + grp->pad_shift[si]) * Kc;

  // ---- radial: block b holds species 2b (columns 0-15) and 2b+1 (columns 16-31)
  const int m = lane & 15, half = lane >> 4;
  const float shf = c.ShfR[m];
  for (int b = 0; b < c.nRB; ++b) {
    const int cp = grp->cpos[b];
    if (cp < 0) continue;
    float out = 0.f;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int s = 2 * b + h;
      float acc = 0.f;
      if (s < c.S) {
        const int q1 = e.segR[s + 1];
        for (int q = e.segR[s] + half; q < q1; q += 2) {
          const float x = e.u[q].w - shf;
          acc = fmaf(e.wR[q], ex2f(-c.etaR_l2e * x * x), acc);
        }
      }
      acc += __shfl_xor_sync(0xffffffffu, acc, 16);
      if (half == h) out = acc;
    }
    row[cp * BLK + lane] = out;
  }

  // ---- angular: only pairs of species that are present can hold triplets; in dense-K mode the other
  // materialised blocks are zero-filled first (same lane, same address: program order keeps the later value)
  const int np = grp->npres;
  if (grp->nblk == c.nblk_full && np < c.S)
    for (int b = c.nRB; b < c.nblk_full; ++b) row[grp->cpos[b] * BLK + lane] = 0.f;
  for (int i1 = 0; i1 < np; ++i1) {
    const int s1 = grp->pres[i1];
    const int a1 = e.segA[s1], n1 = e.segA[s1 + 1] - a1;
    for (int i2 = i1; i2 < np; ++i2) {
      const int s2 = grp->pres[i2];
      const int p = s1 * c.S - (s1 * (s1 - 1)) / 2 + (s2 - s1);
      const int cp = grp->cpos[c.nRB + p];
      if (cp < 0) continue;
      const int a2 = e.segA[s2], n2 = e.segA[s2 + 1] - a2;
      const bool same = (s1 == s2);
      const int T = same ? (n1 * (n1 - 1)) / 2 : n1 * n2;
      if (T == 0) { row[cp * BLK + lane] = 0.f; continue; }
      const float inv_n = 1.0f / (float)(same ? n1 : n2);
      float acc[32];
#pragma unroll
      for (int i = 0; i < 32; ++i) acc[i] = 0.f;
      for (int t = lane; t < T; t += 32) {
        int j, k;
        if (same) { decode_same(t, n1, inv_n, j, k); j += a1; k += a1; }
        else { int r = (int)(((float)t + 0.5f) * inv_n); j = a1 + r; k = a2 + (t - r * n2); }
        const float4 uj = e.ua[j], uk = e.ua[k];
        const float u = fmaf(uj.x, uk.x, fmaf(uj.y, uk.y, uj.z * uk.z));
        const float cc = c.cTheta * u;
        const float ss = sqrtf(fmaxf(1.0f - cc * cc, 0.f));
        const float Rbar = 0.5f * (uj.w + uk.w);
        const float ff2 = 2.0f * e.fA[j] * e.fA[k];
        float F2[NSHFA];
#pragma unroll
        for (int a = 0; a < NSHFA; ++a) {
          const float x = Rbar - c.ShfA[a];
          F2[a] = ex2f(-c.etaA_l2e * x * x) * ff2;
        }
#pragma unroll
        for (int z = 0; z < NSHFZ; ++z) {
          const float B = fmaf(0.5f, fmaf(cc, c.cosZ[z], ss * c.sinZ[z]), 0.5f);
          float Bz, Bm;
          bpow(c, fmaxf(B, 0.f), Bz, Bm);
#pragma unroll
          for (int a = 0; a < NSHFA; ++a) acc[a * NSHFZ + z] = fmaf(Bz, F2[a], acc[a * NSHFZ + z]);
        }
      }
      row[cp * BLK + lane] = reduce32(acc, lane);
    }
  }
}

}  // namespace nnp
