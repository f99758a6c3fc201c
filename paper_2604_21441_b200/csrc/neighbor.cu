// neighbor.cu -- K0-K2 of SURVEY.md section 8.a: species map + ML gather, periodic cell binning with a
// counting sort, and pair enumeration under the minimum-image convention into radial (R <= Rcr) and
// angular (R <= Rca) neighbour rows (BASELINE.json north_star stage (1)).
//
// Layout decisions:
//  * atoms are sorted by key = slot * ncell + cell (slot-major), so AEV rows come out grouped by element
//    for the MLP tiles and neighbour rows come out sorted by species without any extra pass;
//  * sorted positions are stored RELATIVE TO THEIR CELL ORIGIN (computed in fp64, rounded to fp32), so the
//    fp32 displacement d = (l_j - l_i) + o * edge has an error of a few 1e-7 Angstrom for any box size;
//  * the neighbour predicate is the pinned fp64 expression of SURVEY.md section 8.c step 2 (reading #6):
//    fp32 decides outside a guard band, inside it the expression is re-evaluated in fp64 from the original
//    fp32 coordinates, so lists are bit-identical to the oracle's O(N^2) definition.
#include "nnp_internal.h"

namespace nnp {

__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// ---------------------------------------------------------------- grid setup (1 block)
__global__ void k_grid_setup(GridInfo* g, GroupInfo* grp, int pbc, float Lx, float Ly, float Lz, float Rcr,
                             int max_cells, const float* __restrict__ pos, const int32_t* __restrict__ ml,
                             int n_ml) {
  __shared__ float smin[3][32], smax[3][32];
  double ext[3], org[3] = {0.0, 0.0, 0.0};
  const double cutoff = (double)Rcr * (1.0 + 1e-4);
  if (pbc) {
    ext[0] = (double)Lx; ext[1] = (double)Ly; ext[2] = (double)Lz;
  } else {
    float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
    for (int a = threadIdx.x; a < n_ml; a += blockDim.x) {
      int i = ml ? ml[a] : a;
      for (int d = 0; d < 3; ++d) {
        float x = pos[3 * (size_t)i + d];
        lo[d] = fminf(lo[d], x); hi[d] = fmaxf(hi[d], x);
      }
    }
    for (int d = 0; d < 3; ++d) {
      for (int o = 16; o > 0; o >>= 1) {
        lo[d] = fminf(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
        hi[d] = fmaxf(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
      }
      if ((threadIdx.x & 31) == 0) { smin[d][threadIdx.x >> 5] = lo[d]; smax[d][threadIdx.x >> 5] = hi[d]; }
    }
    __syncthreads();
    for (int d = 0; d < 3; ++d) {
      float l = 3.0e38f, h = -3.0e38f;
      for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { l = fminf(l, smin[d][w]); h = fmaxf(h, smax[d][w]); }
      if (n_ml == 0) { l = 0.f; h = 0.f; }
      org[d] = (double)l; ext[d] = (double)h - (double)l;
    }
  }
  if (threadIdx.x != 0) return;
  int nc[3];
  for (int d = 0; d < 3; ++d) {
    int n = (int)floor(ext[d] / cutoff);
    if (pbc) { if (n < 3) n = 1; } else { if (n < 1) n = 1; }
    nc[d] = n;
  }
  // respect the workspace's cell capacity: shrink the largest dimension (cells only get bigger)
  while ((long long)nc[0] * nc[1] * nc[2] > (long long)max_cells) {
    int d = 0;
    if (nc[1] > nc[d]) d = 1;
    if (nc[2] > nc[d]) d = 2;
    nc[d] -= 1;
    if (pbc && nc[d] < 3) nc[d] = 1;
  }
  for (int d = 0; d < 3; ++d) {
    double e = ext[d] / nc[d];
    if (!pbc && e < cutoff) e = cutoff;
    g->nc[d] = nc[d];
    g->edge_d[d] = e; g->inv_edge_d[d] = 1.0 / e; g->edge[d] = (float)e;
    g->origin_d[d] = org[d];
  }
  g->L_d[0] = (double)Lx; g->L_d[1] = (double)Ly; g->L_d[2] = (double)Lz;
  g->L[0] = Lx; g->L[1] = Ly; g->L[2] = Lz;
  g->ncell = nc[0] * nc[1] * nc[2];
  g->pbc = pbc;
  (void)grp;
}

// ---------------------------------------------------------------- K0: species map, ML gather, cell key
__global__ void k_bin(AevConst c, const GridInfo* __restrict__ g, const float* __restrict__ pos,
                      const int32_t* __restrict__ Z, const int32_t* __restrict__ ml, int n_atoms, int n_ml,
                      float4* __restrict__ tmp4, int* __restrict__ rank, int* __restrict__ cell_count,
                      unsigned long long* __restrict__ facc, int* __restrict__ flags) {
  int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n_ml) return;
  int i = a;
  if (ml) {
    i = ml[a];
    bool bad = (i < 0 || i >= n_atoms) || (a > 0 && ml[a - 1] >= i);
    if (bad) { atomicOr(flags, FLAG_ARG); i = min(max(i, 0), n_atoms - 1); }
  }
  int z = Z[i];
  int slot = (z >= 0 && z < 128) ? (int)c.zlut[z] : -1;
  if (slot < 0) { atomicOr(flags, FLAG_SPECIES); slot = 0; }
  int cc[3];
  float loc[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    double x = (double)pos[3 * (size_t)i + d];
    double t;
    if (g->pbc) {
      t = x / g->L_d[d];
      t -= floor(t);
      if (!(t < 1.0)) t = 0.0;
      t *= (double)g->nc[d];
    } else {
      t = (x - g->origin_d[d]) * g->inv_edge_d[d];
      if (t < 0.0) t = 0.0;
    }
    int ci = (int)t;
    if (ci >= g->nc[d]) ci = g->nc[d] - 1;
    cc[d] = ci;
    loc[d] = (float)((t - (double)ci) * g->edge_d[d]);
  }
  int cell = (cc[0] * g->nc[1] + cc[1]) * g->nc[2] + cc[2];
  int key = slot * g->ncell + cell;
  rank[a] = atomicAdd(&cell_count[key], 1);
  tmp4[a] = make_float4(loc[0], loc[1], loc[2], __int_as_float(key));
  facc[3 * (size_t)a + 0] = 0ull; facc[3 * (size_t)a + 1] = 0ull; facc[3 * (size_t)a + 2] = 0ull;
}

// ---------------------------------------------------------------- K1a: exclusive scan + groups + tiles
__global__ void __launch_bounds__(1024) k_scan(const GridInfo* __restrict__ g, const int* __restrict__ count,
                                               int* __restrict__ bstart, GroupInfo* __restrict__ grp,
                                               TileInfo* __restrict__ tiles, int S, int n_ml, int max_tiles,
                                               int dense_k, int* __restrict__ flags) {
  __shared__ int part[1024];
  __shared__ int gs[MAX_S + 1], tb[MAX_S + 1];
  const int n = S * g->ncell;
  const int per = (n + 1023) / 1024;
  const int lo = min(threadIdx.x * per, n), hi = min(lo + per, n);
  int s = 0;
  for (int k = lo; k < hi; ++k) s += count[k];
  part[threadIdx.x] = s;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {  // Hillis-Steele inclusive scan
    int v = (threadIdx.x >= o) ? part[threadIdx.x - o] : 0;
    __syncthreads();
    part[threadIdx.x] += v;
    __syncthreads();
  }
  int run = part[threadIdx.x] - s;
  for (int k = lo; k < hi; ++k) { bstart[k] = run; run += count[k]; }
  if (threadIdx.x == 1023) { bstart[n] = part[1023]; if (part[1023] != n_ml) atomicOr(flags, FLAG_ARG); }
  __syncthreads();
  if (threadIdx.x <= S) gs[threadIdx.x] = bstart[threadIdx.x * g->ncell];
  __syncthreads();
  if (threadIdx.x == 0) {
    int rows = 0, nt = 0;
    for (int q = 0; q < MAX_S; ++q) {
      int cnt = (q < S) ? gs[q + 1] - gs[q] : 0;
      grp->count[q] = cnt;
      grp->start[q] = (q < S) ? gs[q] : n_ml;
      grp->pad_shift[q] = rows - ((q < S) ? gs[q] : 0);
      tb[q] = nt;
      int t = (cnt + TILE_M - 1) / TILE_M;
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
      bool on = dense_k || grp->count[2 * b] > 0 || (2 * b + 1 < S && grp->count[2 * b + 1] > 0);
      grp->cpos[b] = on ? nb : -1;
      if (on) grp->blkmap[nb++] = b;
    }
    int p = 0;
    for (int s1 = 0; s1 < S; ++s1)
      for (int s2 = s1; s2 < S; ++s2, ++p) {
        bool on = dense_k || (grp->count[s1] > 0 && grp->count[s2] > 0);
        grp->cpos[nRB + p] = on ? nb : -1;
        if (on) grp->blkmap[nb++] = nRB + p;
      }
    for (int b = nRB + p; b < MAX_BLK; ++b) grp->cpos[b] = -1;
    for (int b = nb; b < MAX_BLK; ++b) grp->blkmap[b] = 0;
    grp->nblk = nb;
    grp->Kc = nb * BLK;
  }
  __syncthreads();
  const int nt = min(tb[MAX_S], max_tiles);
  for (int t = threadIdx.x; t < nt; t += 1024) {
    int q = 0;
    while (q + 1 < MAX_S && t >= tb[q + 1]) ++q;
    int r = t - tb[q];
    int cnt = gs[min(q + 1, S)] - gs[min(q, S)];
    TileInfo ti;
    ti.slot = q; ti.row0 = grp->pad_shift[q] + gs[q] + r * TILE_M; ti.nvalid = min(TILE_M, cnt - r * TILE_M); ti.pad = 0;
    tiles[t] = ti;
  }
}

// ---------------------------------------------------------------- K1b: scatter into slot-major cell order
__global__ void k_scatter(const GridInfo* __restrict__ g, const float4* __restrict__ tmp4,
                          const int* __restrict__ rank, const int* __restrict__ bstart, int n_ml,
                          float4* __restrict__ spos, int* __restrict__ scell) {
  int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n_ml) return;
  float4 t = tmp4[a];
  int key = __float_as_int(t.w);
  int slot = key / g->ncell;
  int cell = key - slot * g->ncell;
  int dst = bstart[key] + rank[a];
  spos[dst] = make_float4(t.x, t.y, t.z, __int_as_float(a | (slot << 28)));
  scell[dst] = cell;
}

// K1c: the atomic ranks above are not reproducible; order every bucket by ML index so that the sorted order
// (and with it every summation order downstream) is identical from run to run.
__global__ void k_bucket_sort(const GridInfo* __restrict__ g, int S, const int* __restrict__ bstart,
                              float4* __restrict__ spos) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= S * g->ncell) return;
  int lo = bstart[k], hi = bstart[k + 1];
  for (int p = lo + 1; p < hi; ++p) {
    float4 v = spos[p];
    int key = __float_as_int(v.w) & 0x0fffffff;
    int q = p - 1;
    while (q >= lo && (__float_as_int(spos[q].w) & 0x0fffffff) > key) { spos[q + 1] = spos[q]; --q; }
    spos[q + 1] = v;
  }
}

// ---------------------------------------------------------------- K2: neighbour rows, one warp per centre
__device__ __forceinline__ double exact_d2(const float* __restrict__ pos, int oi, int oj, const GridInfo* g) {
  double d[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    double x = (double)pos[3 * (size_t)oj + a] - (double)pos[3 * (size_t)oi + a];
    if (g->pbc) x -= g->L_d[a] * rint(x / g->L_d[a]);
    d[a] = x;
  }
  return __fma_rn(d[2], d[2], __fma_rn(d[1], d[1], __dmul_rn(d[0], d[0])));
}

constexpr float GUARD_BAND = 2.0e-3f;  // Angstrom^2; >> fp32 error of d2 (~1e-5), reading #6

__global__ void __launch_bounds__(256) k_neighbors(AevConst c, const GridInfo* __restrict__ g,
                                                   const GroupInfo* __restrict__ grp,
                                                   const float4* __restrict__ spos, const int* __restrict__ scell,
                                                   const int* __restrict__ bstart, const float* __restrict__ pos,
                                                   const int32_t* __restrict__ ml, int n_ml, int rcap, int acap,
                                                   uint32_t* __restrict__ nbrR, uint8_t* __restrict__ nbrA,
                                                   int* __restrict__ cntR, int* __restrict__ cntA,
                                                   int* __restrict__ flags) {
  const int lane = threadIdx.x & 31;
  const int ip = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (ip >= n_ml) return;
  const float4 ci = spos[ip];
  const int cell = scell[ip];
  const int nc0 = g->nc[0], nc1 = g->nc[1], nc2 = g->nc[2], ncell = g->ncell, pbc = g->pbc;
  const int cz = cell % nc2, cy = (cell / nc2) % nc1, cx = cell / (nc1 * nc2);
  const float ex = g->edge[0], ey = g->edge[1], ez = g->edge[2];
  const int a_i = __float_as_int(ci.w) & 0x0fffffff;
  const int o_i = ml ? ml[a_i] : a_i;
  uint32_t* rowR = nbrR + (size_t)ip * rcap;
  uint8_t* rowA = nbrA + (size_t)ip * acap;
  int nR = 0, nA = 0, bad = 0;
  const unsigned lt = lanemask_lt();
  // offsets per dimension: one cell => {0}; otherwise {-1,0,1} (wrapped if periodic, clipped if open)
  const int nox = (nc0 == 1) ? 1 : 3, noy = (nc1 == 1) ? 1 : 3, noz = (nc2 == 1) ? 1 : 3;
  for (int s = 0; s < c.S; ++s) {
    if (grp->count[s] == 0) continue;
    const int* bs = bstart + s * ncell;
    for (int ix = 0; ix < nox; ++ix) {
      int ox = (nox == 1) ? 0 : ix - 1;
      int nx = cx + ox;
      if (nx < 0 || nx >= nc0) { if (!pbc) continue; nx += (nx < 0) ? nc0 : -nc0; }
      for (int iy = 0; iy < noy; ++iy) {
        int oy = (noy == 1) ? 0 : iy - 1;
        int ny = cy + oy;
        if (ny < 0 || ny >= nc1) { if (!pbc) continue; ny += (ny < 0) ? nc1 : -nc1; }
        // up to three z segments flattened into one candidate list
        int segS[3], segL[3], segO[3], nseg = 0, total = 0;
        for (int iz = 0; iz < noz; ++iz) {
          int oz = (noz == 1) ? 0 : iz - 1;
          int nz = cz + oz;
          if (nz < 0 || nz >= nc2) { if (!pbc) continue; nz += (nz < 0) ? nc2 : -nc2; }
          int k = (nx * nc1 + ny) * nc2 + nz;
          int b0 = bs[k], b1 = bs[k + 1];
          segS[nseg] = b0; segL[nseg] = b1 - b0; segO[nseg] = oz; total += b1 - b0; ++nseg;
        }
        for (int q0 = 0; q0 < total; q0 += 32) {
          int q = q0 + lane;
          bool valid = q < total;
          int jp = 0, oz = 0;
          if (valid) {
            int r = q;
            int sg = 0;
            if (nseg > 1 && r >= segL[0]) { r -= segL[0]; sg = 1; if (nseg > 2 && r >= segL[1]) { r -= segL[1]; sg = 2; } }
            jp = segS[sg] + r; oz = segO[sg];
          }
          bool inR = false, inA = false;
          int cox = ox, coy = oy, coz = oz;
          if (valid && jp != ip) {
            float4 pj = spos[jp];
            float dx = pj.x - ci.x, dy = pj.y - ci.y, dz = pj.z - ci.z;
            if (nc0 == 1) { cox = pbc ? -(int)rintf(dx / ex) : 0; }
            if (nc1 == 1) { coy = pbc ? -(int)rintf(dy / ey) : 0; }
            if (nc2 == 1) { coz = pbc ? -(int)rintf(dz / ez) : 0; }
            dx += (float)cox * ex; dy += (float)coy * ey; dz += (float)coz * ez;
            float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            if (d2 < c.Rcr2 + GUARD_BAND) {
              bool nearR = fabsf(d2 - c.Rcr2) <= GUARD_BAND, nearA = fabsf(d2 - c.Rca2) <= GUARD_BAND;
              inR = !nearR;
              inA = d2 < c.Rca2;
              if (nearR || nearA || d2 < 1e-6f) {
                int a_j = __float_as_int(pj.w) & 0x0fffffff;
                int o_j = ml ? ml[a_j] : a_j;
                double e2 = exact_d2(pos, o_i, o_j, g);
                if (nearR) inR = e2 <= c.Rcr2_d;
                if (nearA) inA = e2 <= c.Rca2_d;
                if (e2 == 0.0) bad |= FLAG_COINCIDENT;
              }
            }
          }
          unsigned mR = __ballot_sync(0xffffffffu, inR);
          unsigned mA = __ballot_sync(0xffffffffu, inA);
          int pR = nR + __popc(mR & lt);
          if (inR) {
            if (pR < rcap) rowR[pR] = (uint32_t)jp | ((uint32_t)((cox + 1) | ((coy + 1) << 2) | ((coz + 1) << 4)) << JBITS);
            else bad |= FLAG_CAP;
          }
          if (inA) {
            int pA = nA + __popc(mA & lt);
            if (pA < acap && pR < rcap) rowA[pA] = (uint8_t)pR; else bad |= FLAG_CAP;
          }
          nR += __popc(mR); nA += __popc(mA);
        }
      }
    }
  }
  if (bad) atomicOr(flags, bad);
  if (lane == 0) { cntR[ip] = min(nR, rcap); cntA[ip] = min(nA, acap); }
}

// ---------------------------------------------------------------- host launcher
int launch_neighbor_stage(nnp_workspace* ws, const float* d_pos, const int32_t* d_Z, const float* box, int pbc,
                          const int32_t* d_ml, int64_t n_atoms, int64_t n_ml) {
  const nnp_model* m = ws->model;
  cudaStream_t st = ws->stream;
  const int S = m->aev.S;
  int nl = 0;
  k_grid_setup<<<1, 1024, 0, st>>>(ws->grid, ws->groups, pbc, box[0], box[4], box[8], m->aev.Rcr, ws->max_cells,
                                   d_pos, d_ml, (int)n_ml);
  ++nl;
  cudaMemsetAsync(ws->cell_count, 0, sizeof(int) * ((size_t)MAX_S * ws->max_cells + 1), st);
  const int nb = (int)((n_ml + 255) / 256);
  if (n_ml > 0) {
    k_bin<<<nb, 256, 0, st>>>(m->aev, ws->grid, d_pos, d_Z, d_ml, (int)n_atoms, (int)n_ml, ws->tmp4, ws->rank,
                              ws->cell_count, ws->facc, ws->flags);
    ++nl;
  }
  k_scan<<<1, 1024, 0, st>>>(ws->grid, ws->cell_count, ws->bstart, ws->groups, ws->tiles, S, (int)n_ml,
                             ws->max_tiles, ws->dense_k, ws->flags);
  ++nl;
  if (n_ml > 0) {
    k_scatter<<<nb, 256, 0, st>>>(ws->grid, ws->tmp4, ws->rank, ws->bstart, (int)n_ml, ws->spos, ws->scell);
    // the bucket count is only known on the device: launch for the capacity, guard on S * ncell inside
    k_bucket_sort<<<(S * ws->max_cells + 255) / 256, 256, 0, st>>>(ws->grid, S, ws->bstart, ws->spos);
    k_neighbors<<<(int)((n_ml * 32 + 255) / 256), 256, 0, st>>>(m->aev, ws->grid, ws->groups, ws->spos, ws->scell,
                                                                ws->bstart, d_pos, d_ml, (int)n_ml, ws->rcap,
                                                                ws->acap, ws->nbrR, ws->nbrA, ws->cntR, ws->cntA,
                                                                ws->flags);
    nl += 3;
  }
  return nl;
}

}  // namespace nnp
