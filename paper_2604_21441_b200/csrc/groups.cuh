// groups.cuh -- species groups, MLP tiles and the compacted AEV column map from the per-slot atom counts (the tail of
// K1's scan), shared by the cell-list prep kernel (neighbor.cu) and the small-system front end (small.cu).
#pragma once
#include "nnp_internal.h"

namespace nnp {

// ONE thread: gs[q] = first sorted index of slot q (gs[S] = n_ml).  Fills *grp, pshift[MAX_S] (row = sorted index +
// pshift[slot]) and tb[MAX_S + 1] (first tile of each slot).
__device__ inline void d_groups(const int* gs, int S, int n_ml, int max_tiles, int dense_k, GroupInfo* __restrict__ grp,
                                int* pshift, int* tb, int* __restrict__ flags) {
  int rows = 0, nt = 0, cnt[MAX_S];
  for (int q = 0; q < MAX_S; ++q) {
    cnt[q] = (q < S) ? gs[q + 1] - gs[q] : 0;
    grp->count[q] = cnt[q];
    grp->start[q] = (q < S) ? gs[q] : n_ml;
    pshift[q] = rows - ((q < S) ? gs[q] : 0);
    grp->pad_shift[q] = pshift[q];
    tb[q] = nt;
    int t = (cnt[q] + TILE_M - 1) / TILE_M;
    nt += t; rows += t * TILE_M;
  }
  grp->start[MAX_S] = n_ml;
  tb[MAX_S] = nt;
  grp->n_tiles = min(nt, max_tiles);
  grp->n_rows = rows;
  if (nt > max_tiles) atomicOr(flags, FLAG_CAP);
  // compacted AEV column blocks: a radial block holds species (2b, 2b+1), an angular block one pair p(s1,s2)
  const int nRB = (S + 1) / 2;
  int nb = 0;
  for (int b = 0; b < nRB; ++b) {
    bool on = dense_k || cnt[2 * b] > 0 || (2 * b + 1 < S && cnt[2 * b + 1] > 0);
    grp->cpos[b] = on ? nb : -1;
    if (on) grp->blkmap[nb++] = b;
  }
  int p = 0;
  for (int s1 = 0; s1 < S; ++s1)
    for (int s2 = s1; s2 < S; ++s2, ++p) {
      bool on = dense_k || (cnt[s1] > 0 && cnt[s2] > 0);
      grp->cpos[nRB + p] = on ? nb : -1;
      if (on) grp->blkmap[nb++] = nRB + p;
    }
  for (int b = nRB + p; b < MAX_BLK; ++b) grp->cpos[b] = -1;
  for (int b = nb; b < MAX_BLK; ++b) grp->blkmap[b] = 0;
  grp->nblk = nb;
  grp->Kc = nb * BLK;
  int npres = 0;
  for (int q = 0; q < MAX_S; ++q) { if (cnt[q] > 0) grp->pres[npres++] = q; }
  for (int q = npres; q < MAX_S; ++q) grp->pres[q] = 0;
  grp->npres = npres;
  // identifies what the layer-1 operand images were packed for: the materialised blocks AND the species present (in
  // dense-K mode every block is materialised whatever the species, but only networks of present species are packed)
  unsigned long long key = 1ull << 63;
  for (int b = 0; b < nb; ++b) key |= 1ull << grp->blkmap[b];
  for (int q = 0; q < MAX_S; ++q) if (cnt[q] > 0) key |= 1ull << (44 + q);
  grp->colkey = key;
}

// The same by ONE WARP (all 32 lanes call it): slots and column blocks are handled lane-parallel with ballots instead of
// one thread's serial loops (measured 3.4 us for the serial version -- on the critical path of every evaluation).
__device__ inline void d_groups_warp(const int* gs, int S, int n_ml, int max_tiles, int dense_k, GroupInfo* grp, int* pshift,
                                     int* tb, int* __restrict__ flags) {
  const int lane = threadIdx.x & 31;
  const unsigned full = 0xffffffffu, lt = (1u << lane) - 1u;
  int cnt = 0, start = n_ml, t = 0;
  if (lane < S) { cnt = gs[lane + 1] - gs[lane]; start = gs[lane]; }
  t = (cnt + TILE_M - 1) / TILE_M;
  int inc = t;
  for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(full, inc, o); if (lane >= o) inc += v; }
  const int tex = inc - t, nt = __shfl_sync(full, inc, 31);
  if (lane < MAX_S) {
    grp->count[lane] = cnt; grp->start[lane] = start;
    const int ps = tex * TILE_M - ((lane < S) ? gs[lane] : 0);
    pshift[lane] = ps; grp->pad_shift[lane] = ps; tb[lane] = tex;
  }
  const unsigned presmask = __ballot_sync(full, cnt > 0);
  const int nRB = (S + 1) / 2, nfull = nRB + S * (S + 1) / 2;
  int nb = 0;
  unsigned long long key = 1ull << 63;
  for (int b0 = 0; b0 < MAX_BLK; b0 += 32) {
    const int b = b0 + lane;
    bool on = false;
    if (b < nRB) {
      on = dense_k || ((presmask >> (2 * b)) & 1u) || (2 * b + 1 < S && ((presmask >> (2 * b + 1)) & 1u));
    } else if (b < nfull) {
      int p = b - nRB, s1 = 0;
      while (p >= S - s1) { p -= S - s1; ++s1; }
      on = dense_k || (((presmask >> s1) & 1u) && ((presmask >> (s1 + p)) & 1u));
    }
    const unsigned m = __ballot_sync(full, on);
    const int cp = nb + __popc(m & lt);
    if (b < MAX_BLK) grp->cpos[b] = on ? cp : -1;
    if (on) grp->blkmap[cp] = b;
    nb += __popc(m);
    key |= (unsigned long long)m << b0;
  }
  for (int b = nb + lane; b < MAX_BLK; b += 32) grp->blkmap[b] = 0;
  const int npres = __popc(presmask);
  if (lane < MAX_S) {
    if (cnt > 0) grp->pres[__popc(presmask & lt)] = lane;
    if (lane >= npres) grp->pres[lane] = 0;
  }
  if (lane == 0) {
    grp->start[MAX_S] = n_ml; tb[MAX_S] = nt;
    grp->n_tiles = min(nt, max_tiles); grp->n_rows = nt * TILE_M;
    if (nt > max_tiles) atomicOr(flags, FLAG_CAP);
    grp->nblk = nb; grp->Kc = nb * BLK; grp->npres = npres;
    grp->colkey = key | ((unsigned long long)presmask << 44);
  }
  __syncwarp();
}

// whole block: the tile table
__device__ inline void d_tiles(const int* gs, const int* pshift, const int* tb, int S, int max_tiles,
                               TileInfo* __restrict__ tiles) {
  const int nt = min(tb[MAX_S], max_tiles);
  for (int t = threadIdx.x; t < nt; t += blockDim.x) {
    int q = 0;
    while (q + 1 < MAX_S && t >= tb[q + 1]) ++q;
    int r = t - tb[q];
    int cnt = gs[min(q + 1, S)] - gs[min(q, S)];
    TileInfo ti;
    ti.slot = q; ti.row0 = pshift[q] + gs[q] + r * TILE_M; ti.nvalid = min(TILE_M, cnt - r * TILE_M); ti.pad = 0;
    tiles[t] = ti;
  }
}

}  // namespace nnp
