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
#include <cooperative_groups.h>
#include <algorithm>
#include "nnp_internal.h"
#include "groups.cuh"
#include "neighbor_common.cuh"

namespace cg = cooperative_groups;

namespace nnp {

// Cell grid from the extent of the system (thread 0 of the prep kernel; for periodic boxes also the HOST, which passes
// the result to the kernel by value and saves the set-up phase and one grid-wide barrier -- same doubles, same code).
__host__ __device__ inline void grid_from_extent(GridInfo* g, int pbc, const double ext[3], const double org[3], float Lx,
                                                 float Ly, float Lz, double cutoff, int max_cells) {
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
  g->tric = 0;
  for (int k = 0; k < 9; ++k) { g->ev[k] = 0.f; g->ev_d[k] = 0.0; }
  for (int d = 0; d < 3; ++d) { g->ev[4 * d] = g->edge[d]; g->ev_d[4 * d] = g->edge_d[d]; }
  g->H_d[0] = (double)Lx; g->H_d[1] = (double)Ly; g->H_d[2] = (double)Lz; g->H_d[3] = g->H_d[4] = g->H_d[5] = 0.0;
}

// Periodic triclinic box (HOST; GROMACS rows, reading #35): cells are cut in fractional coordinates, nc[d] =
// floor(width_d / cutoff) with width_d the distance between the box faces normal to reciprocal direction d, so that
// neighbours within the cut-off always sit in adjacent cells.  Every dimension needs >= 3 cells (the one-cell
// minimum-image sweep is orthorhombic only): returns false otherwise.
inline bool grid_triclinic(GridInfo* g, const float* box, double cutoff, int max_cells) {
  const double a[3] = {(double)box[0], 0.0, 0.0}, b[3] = {(double)box[3], (double)box[4], 0.0},
               c[3] = {(double)box[6], (double)box[7], (double)box[8]};
  auto cross_norm = [](const double* u, const double* v) {
    const double x = u[1] * v[2] - u[2] * v[1], y = u[2] * v[0] - u[0] * v[2], z = u[0] * v[1] - u[1] * v[0];
    return sqrt(x * x + y * y + z * z);
  };
  const double vol = a[0] * b[1] * c[2];
  const double width[3] = {vol / cross_norm(b, c), vol / cross_norm(c, a), vol / cross_norm(a, b)};
  int nc[3];
  for (int d = 0; d < 3; ++d) { nc[d] = (int)floor(width[d] / cutoff); if (nc[d] < 3) return false; }
  while ((long long)nc[0] * nc[1] * nc[2] > (long long)max_cells) {
    int d = 0;
    if (nc[1] > nc[d]) d = 1;
    if (nc[2] > nc[d]) d = 2;
    nc[d] -= 1;
    if (nc[d] < 3) return false;
  }
  const double* rows[3] = {a, b, c};
  for (int d = 0; d < 3; ++d) {
    g->nc[d] = nc[d];
    for (int k = 0; k < 3; ++k) { g->ev_d[3 * d + k] = rows[d][k] / nc[d]; g->ev[3 * d + k] = (float)g->ev_d[3 * d + k]; }
    g->edge_d[d] = width[d] / nc[d]; g->inv_edge_d[d] = 1.0 / g->edge_d[d]; g->edge[d] = (float)g->edge_d[d];
    g->origin_d[d] = 0.0;
    g->L_d[d] = rows[d][d]; g->L[d] = (float)rows[d][d];
  }
  g->H_d[0] = a[0]; g->H_d[1] = b[1]; g->H_d[2] = c[2]; g->H_d[3] = b[0]; g->H_d[4] = c[0]; g->H_d[5] = c[1];
  g->ncell = nc[0] * nc[1] * nc[2];
  g->pbc = 1;
  g->tric = 1;
  return true;
}

bool box_is_triclinic(const float* box) { return box[3] != 0.f || box[6] != 0.f || box[7] != 0.f; }

// the box of a periodic evaluation can be gridded (orthorhombic: always)
bool neighbor_box_ok(const nnp_workspace* ws, const float* box) {
  if (!box_is_triclinic(box)) return true;
  GridInfo g;
  const double skin = ws->reuse_every > 1 ? ws->reuse_skin * ws->len_scale : 0.0;
  return grid_triclinic(&g, box, (double)ws->model->aev.Rcr * (1.0 + 1e-4) + skin, ws->max_cells);
}

// ---------------------------------------------------------------- grid setup (1 block)
__device__ void d_grid_setup(GridInfo* g, GroupInfo* grp, int pbc, float Lx, float Ly, float Lz, float Rcr,
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
  grid_from_extent(g, pbc, ext, org, Lx, Ly, Lz, cutoff, max_cells);
  (void)grp;
}

// ---------------------------------------------------------------- K0: species map, ML gather, cell key
// ML atom a (ML-local index): species slot, cell and cell-local coordinates (fp64 cell coordinates, rounded to fp32 once)
__device__ __forceinline__ void bin_coords(const AevConst& c, const GridInfo* __restrict__ g, const float* __restrict__ pos,
                                           const int32_t* __restrict__ Z, const int32_t* __restrict__ ml, int n_atoms, int a,
                                           int* __restrict__ flags, int& slot, int& cell, float (&loc)[3]) {
  int i = a;
  if (ml) {
    i = ml[a];
    bool bad = (i < 0 || i >= n_atoms) || (a > 0 && ml[a - 1] >= i);
    if (bad) { atomicOr(flags, FLAG_ARG); i = min(max(i, 0), n_atoms - 1); }
  }
  int z = Z[i];
  slot = (z >= 0 && z < 128) ? (int)c.zlut[z] : -1;
  if (slot < 0) { atomicOr(flags, FLAG_SPECIES); slot = 0; }
  int cc[3];
  if (g->tric) {
    // fractional coordinates of the lower-triangular box (fp64), wrapped into [0, 1); local position = the fractional
    // remainder inside the cell times the cell's edge vectors
    const double x = (double)pos[3 * (size_t)i], y = (double)pos[3 * (size_t)i + 1], z = (double)pos[3 * (size_t)i + 2];
    double s[3];
    s[2] = z / g->H_d[2];
    s[1] = (y - s[2] * g->H_d[5]) / g->H_d[1];
    s[0] = (x - s[1] * g->H_d[3] - s[2] * g->H_d[4]) / g->H_d[0];
    double f[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      double t = s[d] - floor(s[d]);
      if (!(t < 1.0)) t = 0.0;
      t *= (double)g->nc[d];
      int ci = (int)t;
      if (ci >= g->nc[d]) ci = g->nc[d] - 1;
      cc[d] = ci;
      f[d] = t - (double)ci;
    }
    loc[0] = (float)(f[0] * g->ev_d[0] + f[1] * g->ev_d[3] + f[2] * g->ev_d[6]);
    loc[1] = (float)(f[1] * g->ev_d[4] + f[2] * g->ev_d[7]);
    loc[2] = (float)(f[2] * g->ev_d[8]);
  } else {
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
  }
  cell = (cc[0] * g->nc[1] + cc[1]) * g->nc[2] + cc[2];
}

__device__ void d_bin(int vb, const AevConst& c, const GridInfo* __restrict__ g, const float* __restrict__ pos,
                      const int32_t* __restrict__ Z, const int32_t* __restrict__ ml, int n_atoms, int n_ml,
                      float4* __restrict__ tmp4, int* __restrict__ rank, int* __restrict__ cell_count,
                      unsigned long long* __restrict__ facc, int* __restrict__ flags) {
  int a = vb * blockDim.x + threadIdx.x;
  if (a >= n_ml) return;
  int slot, cell;
  float loc[3];
  bin_coords(c, g, pos, Z, ml, n_atoms, a, flags, slot, cell, loc);
  int key = slot * g->ncell + cell;
  rank[a] = atomicAdd(&cell_count[key], 1);
  tmp4[a] = make_float4(loc[0], loc[1], loc[2], __int_as_float(key));
  facc[3 * (size_t)a + 0] = 0ull; facc[3 * (size_t)a + 1] = 0ull; facc[3 * (size_t)a + 2] = 0ull;
}

// ---------------------------------------------------------------- K1a: exclusive scan + groups + tiles
__device__ void d_scan(const GridInfo* __restrict__ g, int* __restrict__ count,
                                               int* __restrict__ bstart, GroupInfo* __restrict__ grp,
                                               TileInfo* __restrict__ tiles, int S, int n_ml, int max_tiles,
                                               int dense_k, int* __restrict__ flags) {
  // block-wide exclusive scan of S * ncell bucket counts: each warp owns a contiguous span.  Pass A sums the span
  // (coalesced, loads batched four deep); pass B re-reads it (L1 hits), scans with the warp's base and writes the
  // bucket starts.  The counts are zeroed behind the read, so the next evaluation needs no memset.
  __shared__ int wtot[32];
  __shared__ int gs[MAX_S + 1], tb[MAX_S + 1];
  const int ncell = g->ncell, n = S * ncell;
  const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5, nw = (int)blockDim.x >> 5;
  const int span = (((n + nw - 1) / nw + 31) / 32) * 32;
  const int lo = min(wp * span, n), hi = min(lo + span, n);
  int sum = 0;
  for (int k0 = lo; k0 < hi; k0 += 128) {
#pragma unroll
    for (int u = 0; u < 4; ++u) { const int k = k0 + 32 * u + lane; sum += (k < hi) ? count[k] : 0; }
  }
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
  if (lane == 0) wtot[wp] = sum;
  __syncthreads();
  int carry = 0, total = 0;
  for (int w = 0; w < nw; ++w) { const int t = wtot[w]; if (w < wp) carry += t; total += t; }
  for (int k0 = lo; k0 < hi; k0 += 128) {
    int v[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { const int k = k0 + 32 * u + lane; v[u] = (k < hi) ? count[k] : 0; }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      int inc = v[u];
      for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
      const int k = k0 + 32 * u + lane;
      if (k < hi) {
        const int st = carry + inc - v[u];
        bstart[k] = st;
        count[k] = 0;
        if (k % ncell == 0) gs[k / ncell] = st;    // first bucket of a species slot = start of its group
      }
      carry += __shfl_sync(0xffffffffu, inc, 31);
    }
  }
  if (threadIdx.x == 0) { bstart[n] = total; gs[S] = total; if (total != n_ml) atomicOr(flags, FLAG_ARG); }
  __syncthreads();
  __shared__ int pshift[MAX_S];
  __shared__ GroupInfo grp_s;   // filled by one thread in shared memory, published by all (one thread's ~150 dependent global stores cost microseconds)
  if (threadIdx.x == 0) d_groups(gs, S, n_ml, max_tiles, dense_k, &grp_s, pshift, tb, flags);
  __syncthreads();
  {
    const int* src = reinterpret_cast<const int*>(&grp_s);
    int* dst = reinterpret_cast<int*>(grp);
    for (int k = threadIdx.x; k < (int)(sizeof(GroupInfo) / sizeof(int)); k += blockDim.x) dst[k] = src[k];
  }
  d_tiles(gs, pshift, tb, S, max_tiles, tiles);
}

// ---------------------------------------------------------------- K1b: scatter into slot-major cell order
__device__ void d_scatter(int vb, const GridInfo* __restrict__ g, const float4* __restrict__ tmp4,
                          const int* __restrict__ rank, const int* __restrict__ bstart, int n_ml,
                          float4* __restrict__ spos, int* __restrict__ scell) {
  int a = vb * blockDim.x + threadIdx.x;
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
// (and with it every summation order downstream) is identical from run to run.  One warp per bucket, ranking by
// counting (keys = ML indices are distinct, so ranks are a permutation): buckets of <= 32 atoms compare through
// shuffles in registers; longer ones (a box of one cell: cfg 0 holds 64 H in one bucket) count against the bucket
// in global memory, permute into the free tmp4 scratch and copy back.
__device__ void d_bucket_sort(int vb, const GridInfo* __restrict__ g, int S, const int* __restrict__ bstart,
                              float4* spos, float4* scratch) {
  const int k = (vb * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (k >= S * g->ncell) return;
  const int lo = bstart[k], n = bstart[k + 1] - lo;
  if (n <= 1) return;
  if (n <= 32) {
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    int key = 0x7fffffff;
    if (lane < n) { v = spos[lo + lane]; key = __float_as_int(v.w) & 0x0fffffff; }
    int rank = 0;
    for (int o = 0; o < n; ++o) rank += (__shfl_sync(0xffffffffu, key, o) < key) ? 1 : 0;
    __syncwarp();
    if (lane < n) spos[lo + rank] = v;
  } else {
    for (int e = lane; e < n; e += 32) {
      const float4 v = spos[lo + e];
      const int key = __float_as_int(v.w) & 0x0fffffff;
      int rank = 0;
      for (int o = 0; o < n; ++o) rank += ((__float_as_int(spos[lo + o].w) & 0x0fffffff) < key) ? 1 : 0;
      scratch[lo + rank] = v;
    }
    __syncwarp();
    for (int e = lane; e < n; e += 32) spos[lo + e] = scratch[lo + e];
  }
}

// ---------------------------------------------------------------- K0-K1, fast variant: append + per-cell ordering
// Periodic boxes with >= 3 cells in every dimension (the grid is known on the host).
//   k_bin_cells : every ML atom is appended to a fixed-capacity buffer of its CELL (the atomic rank is the destination:
//                 no scatter pass) and counted per (species, cell) bucket;
//   k_cell_sort : one warp per cell.  Bucket starts come from sums every block forms for itself over the bucket counts
//                 of the species present (cfg 2: 2 x 1331 counts, ten loads per thread): no grid-wide scan, no barrier.
//                 (Counting per group of cells with atomics as a second level was measured and dropped: a few hundred
//                 atomics on one address serialise in L2 -- 11 us for 24 000 atoms on 84 counters.)  The
//                 cell's atoms then go to their place in the slot-major sorted order of the general path: an atom's
//                 place inside its (species, cell) bucket is its rank by ML index among the bucket's atoms -- a pure
//                 function of the cell's content, so the order is reproducible although the append order is not.
// Block 0 of k_cell_sort also derives groups, tiles and the column set.  The counters are cleared by k_neighbors (every
// cell has a block there).  Against k_prep (five phases, four grid-wide barriers): cfg 2 27 us -> ~10 us.
constexpr int CELL_CAP = 96;            // atoms per cell in the append buffer (liquid water at Rcr-wide cells: ~18)
constexpr int BIN_THREADS = 256;
constexpr int FAST_MAX_CELLS = 32768;   // every k_cell_sort block reads all bucket counts of the species present: beyond this k_prep's scan

struct BinArgs {
  AevConst c;
  GridInfo hg;
  GridInfo* grid;
  const float* pos; const int32_t* Z; const int32_t* ml;
  float4* cellbuf; int* cellfill; int* cell_count; int* present;
  unsigned long long* facc; int* flags;
  int n_atoms, n_ml;
  const float* pos_src; float* pos_dst;   // nnp_eval_host: the caller's pinned positions, to be staged into pos (= pos_dst) here
};

__global__ void __launch_bounds__(BIN_THREADS) k_bin_cells(const __grid_constant__ BinArgs a) {
  TL_SCOPE(0);
  __shared__ int spres;
  pdl_trigger();
  const GridInfo* g = &a.hg;
  if (threadIdx.x == 0) spres = 0;
  if (blockIdx.x == 0 && threadIdx.x == 0) *a.grid = a.hg;
  if (a.pos_src) {
    // the host entry point's upload, done here: the block streams the 768 floats of ITS atoms from the caller's pinned
    // buffer (whole 128-byte lines over PCIe) into the device copy every later reader uses, and goes on with them
    // (all atoms are ML atoms in this mode: atom i = thread i).  Saves the copy's launch and its ~10 us ahead of this kernel.
    const size_t base = (size_t)blockIdx.x * (3 * BIN_THREADS), lim = 3 * (size_t)a.n_atoms;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const size_t idx = base + threadIdx.x + BIN_THREADS * k;
      if (idx < lim) a.pos_dst[idx] = a.pos_src[idx];
    }
  }
  __syncthreads();
  const int i = blockIdx.x * BIN_THREADS + threadIdx.x;
  int bit = 0;
  if (i < a.n_ml) {
    int slot, cell;
    float loc[3];
    bin_coords(a.c, g, a.pos, a.Z, a.ml, a.n_atoms, i, a.flags, slot, cell, loc);
    atomicAdd(&a.cell_count[slot * g->ncell + cell], 1);
    const int r = atomicAdd(&a.cellfill[cell], 1);
    if (r < CELL_CAP) a.cellbuf[(size_t)cell * CELL_CAP + r] = make_float4(loc[0], loc[1], loc[2], __int_as_float(i | (slot << 28)));
    else atomicOr(a.flags, FLAG_CAP);
    a.facc[3 * (size_t)i + 0] = 0ull; a.facc[3 * (size_t)i + 1] = 0ull; a.facc[3 * (size_t)i + 2] = 0ull;
    bit = 1 << slot;
  }
  bit = __reduce_or_sync(0xffffffffu, bit);
  if ((threadIdx.x & 31) == 0 && bit) atomicOr(&spres, bit);
  __syncthreads();
  if (threadIdx.x == 0 && spres) atomicOr(a.present, spres);
}

struct SortArgs {
  GroupInfo* groups; TileInfo* tiles;
  const float4* cellbuf; const int* cell_count; const int* present;
  int* bstart; float4* spos; int* scell; int* flags;
  int* inv;   // [n_ml] ML-local index -> sorted index (k_force_out writes the forces in the caller's order through it)
  int S, ncell, n_ml, max_tiles, dense_k;
};

__global__ void __launch_bounds__(256) k_cell_sort(const __grid_constant__ SortArgs a) {
  __shared__ int red[8][2][MAX_S];
  __shared__ int cnt8[8][MAX_S], bst8[8][MAX_S];
  __shared__ int gs[MAX_S + 1], pre_s[MAX_S], pshift[MAX_S], tb[MAX_S + 1];
  __shared__ GroupInfo grp_s;
  TL_SCOPE(1);
  pdl_trigger();
  pdl_wait();
  TL_WAITED(1);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int S = a.S, ncell = a.ncell;
  const int c0 = blockIdx.x * 8, cell = c0 + warp;
  // the cell's appended atoms, three per lane (the slots beyond the cell's count hold stale data and are masked below)
  constexpr int PER = CELL_CAP / 32;
  float4 e[PER];
#pragma unroll
  for (int u = 0; u < PER; ++u)
    e[u] = (cell < ncell) ? a.cellbuf[(size_t)cell * CELL_CAP + u * 32 + lane] : make_float4(0.f, 0.f, 0.f, 0.f);
  const int pm = *a.present;
  // ---- per species present: atoms in all cells (tot) and in the cells before this block's (pre)
  int tot[MAX_S], pre[MAX_S];
#pragma unroll
  for (int s = 0; s < MAX_S; ++s) {
    tot[s] = 0; pre[s] = 0;
    if (s < S && ((pm >> s) & 1)) {
      for (int c = tid; c < ncell; c += 256) { const int v = a.cell_count[s * ncell + c]; tot[s] += v; if (c < c0) pre[s] += v; }
    }
  }
#pragma unroll
  for (int s = 0; s < MAX_S; ++s) {
    if (s < S && ((pm >> s) & 1)) {
      for (int o = 16; o > 0; o >>= 1) { tot[s] += __shfl_xor_sync(0xffffffffu, tot[s], o); pre[s] += __shfl_xor_sync(0xffffffffu, pre[s], o); }
    }
    if (lane == 0) { red[warp][0][s] = tot[s]; red[warp][1][s] = pre[s]; }
  }
  if (lane < MAX_S) cnt8[warp][lane] = (lane < S && cell < ncell && ((pm >> lane) & 1)) ? a.cell_count[lane * ncell + cell] : 0;
  __syncthreads();
  if (tid < MAX_S) {
    int T = 0, P = 0;
    for (int w = 0; w < 8; ++w) { T += red[w][0][tid]; P += red[w][1][tid]; }
    red[0][0][tid] = T; pre_s[tid] = P;   // (only thread tid touches column tid of red[0][0] here)
  }
  __syncthreads();
  if (tid == 0) {
    int run = 0;
    for (int q = 0; q <= MAX_S; ++q) { gs[q] = run; if (q < MAX_S) run += red[0][0][q]; }
  }
  __syncthreads();
  // ---- bucket starts of this block's cells
  if (lane < MAX_S) {
    int b = gs[lane] + pre_s[lane];
    for (int w = 0; w < warp; ++w) b += cnt8[w][lane];
    bst8[warp][lane] = b;
    if (lane < S && cell < ncell) a.bstart[lane * ncell + cell] = b;
  }
  if (blockIdx.x == 0 && tid == 0) {
    a.bstart[S * ncell] = gs[MAX_S];
    if (gs[MAX_S] != a.n_ml) atomicOr(a.flags, FLAG_ARG);
  }
  __syncwarp();
  // ---- rank inside the (species, cell) bucket by ML index, write to the sorted order
  if (cell < ncell) {
    int n = 0;
    for (int s = 0; s < S; ++s) n += cnt8[warp][s];
    n = min(n, CELL_CAP);
    int key[PER], rank[PER];
#pragma unroll
    for (int u = 0; u < PER; ++u) { key[u] = (u * 32 + lane < n) ? __float_as_int(e[u].w) : 0x7fffffff; rank[u] = 0; }
#pragma unroll
    for (int v = 0; v < PER; ++v) {
      if (v * 32 < n) {
        const int m = min(32, n - v * 32);
        for (int o = 0; o < m; ++o) {
          const int ko = __shfl_sync(0xffffffffu, key[v], o);
#pragma unroll
          for (int u = 0; u < PER; ++u) rank[u] += (((ko ^ key[u]) >> 28) == 0 && ko < key[u]) ? 1 : 0;
        }
      }
    }
#pragma unroll
    for (int u = 0; u < PER; ++u) {
      if (u * 32 + lane < n) {
        const int dst = bst8[warp][(key[u] >> 28) & 7] + rank[u];
        if (dst < a.n_ml) { a.spos[dst] = e[u]; a.scell[dst] = cell; a.inv[key[u] & 0x0fffffff] = dst; }
      }
    }
  }
  // ---- block 0: groups, tiles, column set
  if (blockIdx.x == 0) {
    if (warp == 0) d_groups_warp(gs, S, a.n_ml, a.max_tiles, a.dense_k, &grp_s, pshift, tb, a.flags);
    __syncthreads();
    const int* src = reinterpret_cast<const int*>(&grp_s);
    int* dst = reinterpret_cast<int*>(a.groups);
    for (int k = tid; k < (int)(sizeof(GroupInfo) / sizeof(int)); k += 256) dst[k] = src[k];
    d_tiles(gs, pshift, tb, S, a.max_tiles, a.tiles);
  }
}

// ---------------------------------------------------------------- K2: neighbour rows, one warp per centre
constexpr int NB_CAP = 1024;            // candidates staged in shared memory per chunk
constexpr int NB_SEG = MAX_S * 27;      // (species, neighbour cell) segments of one centre cell
constexpr int SURV_CAP = 256;           // candidates of one centre that pass the cheap distance filter, per chunk

// The decision on 32 candidates of centre ip (one per lane; d = displacement from the centre, ent = row entry, a_j = the
// candidate's ML-local index): radial / angular membership by the fp32 value outside the guard bands, by the pinned
// fp64 predicate on the ORIGINAL coordinates inside them (reading #6); ballot compaction into the rows.  Shared by the
// cell sweep and the row refresh from stored wide rows, so both give the same rows.
template <bool TRIC>
__device__ __forceinline__ void decide32(const AevConst& c, const GridInfo* __restrict__ g, const float* __restrict__ pos,
                                         const int32_t* __restrict__ ml, bool live, float dx, float dy, float dz, uint32_t ent,
                                         int a_j, int ip, int o_i, unsigned lt, uint32_t* rR, uint8_t* rA, int rcap, int acap,
                                         int& nR, int& nA, int& bad) {
  const float Rcr2 = c.Rcr2, Rca2 = c.Rca2, loR = c.Rcr2 - GUARD_BAND, loA = c.Rca2 - GUARD_BAND;
  const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
  const bool other = live && (int)(ent & JMASK) != ip;
  bool inR = other && d2 < loR, inA = other && d2 < loA;
  // guard bands (and coincident atoms): the pinned fp64 predicate on the original coordinates decides
  const bool near = other && (fabsf(d2 - Rcr2) <= GUARD_BAND || fabsf(d2 - Rca2) <= GUARD_BAND || d2 < 1e-6f);
  if (near) {
    const int o_j = ml ? ml[a_j] : a_j;
    const double e2 = TRIC ? exact_d2_tric(pos, o_i, o_j, g) : exact_d2(pos, o_i, o_j, g);
    if (fabsf(d2 - Rcr2) <= GUARD_BAND) inR = e2 <= c.Rcr2_d;
    if (fabsf(d2 - Rca2) <= GUARD_BAND) inA = e2 <= c.Rca2_d;
    if (e2 == 0.0) bad |= FLAG_COINCIDENT;
  }
  const unsigned mR = __ballot_sync(0xffffffffu, inR);
  const unsigned mA = __ballot_sync(0xffffffffu, inA);
  const int pR = nR + __popc(mR & lt), pA = nA + __popc(mA & lt);
  if (inR && pR < rcap) rR[pR] = ent;
  if (inA && pA < acap && pR < rcap) rA[pA] = (uint8_t)pR;
  nR += __popc(mR); nA += __popc(mA);
}

// One block per cell.  The atoms of the 27 neighbouring cells (per species: 27 buckets of the slot-major sort) are
// staged once in shared memory, already shifted into the centre cell's frame; then each warp takes a centre of the
// cell and goes over the staged candidates in TWO stages:
//   1. filter: 32 candidates per iteration, fp32 distance against Rcr^2 + guard, ballot compaction of the survivors'
//      staging indices into a per-warp list (~20 instructions per 32 candidates; ~12 % survive);
//   2. decide: the survivors, 32 at a time with full lanes: radial / angular membership by the fp32 value outside the
//      guard bands and by the pinned fp64 predicate on the ORIGINAL coordinates inside them (reading #6), ballot
//      compaction into the rows.
// Candidates are ordered species-major, so rows come out sorted by species.
template <bool TRIC>
__global__ void __launch_bounds__(256, 4) k_neighbors(AevConst c, const GridInfo* __restrict__ g,
                                                   const GroupInfo* __restrict__ grp,
                                                   const float4* __restrict__ spos,
                                                   const int* __restrict__ bstart, const float* __restrict__ pos,
                                                   const int32_t* __restrict__ ml, int n_ml, int rcap, int acap,
                                                   uint32_t* __restrict__ nbrR, uint8_t* __restrict__ nbrA,
                                                   int* __restrict__ cntR, int* __restrict__ cntA,
                                                   int* __restrict__ flags, int* __restrict__ zcount,
                                                   int* __restrict__ zfill, int* __restrict__ zpresent,
                                                   uint32_t* __restrict__ wide, int* __restrict__ cntW, int wcap, float wide_r2) {
  __shared__ float4 cand[NB_CAP];
  __shared__ int candA[NB_CAP];           // ML-local index of the candidate (for the fp64 re-check)
  __shared__ int segStart[NB_SEG], segOff[NB_SEG + 1], segCode[NB_SEG];
  __shared__ float segSx[NB_SEG], segSy[NB_SEG], segSz[NB_SEG];   // Cartesian shift of the segment's cell offset
  __shared__ int cenStart[MAX_S], cenOff[MAX_S + 1];
  __shared__ int wsum[8];
  __shared__ unsigned short surv[8][SURV_CAP];
  TL_SCOPE(2);
  pdl_trigger();
  pdl_wait();
  TL_WAITED(2);
  const int cell = blockIdx.x, ncell = g->ncell;
  if (cell >= ncell) return;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (cell == 0 && tid == 0 && (int)gridDim.x < ncell) atomicOr(flags, FLAG_ARG);   // host / device cell counts differ
  if (zcount && blockIdx.y == 0) {   // fast binning: its counters go back to zero here (every cell has a block; nobody reads them any more)
    if (tid < c.S) zcount[tid * ncell + cell] = 0;
    if (tid == 32) zfill[cell] = 0;
    if (tid == 33 && cell == 0) *zpresent = 0;
  }
  const int nc0 = g->nc[0], nc1 = g->nc[1], nc2 = g->nc[2], pbc = g->pbc, S = c.S;
  const int cz = cell % nc2, cy = (cell / nc2) % nc1, cx = cell / (nc1 * nc2);
  const float ex = g->edge[0], ey = g->edge[1], ez = g->edge[2];

  // ---- centres of this cell (one bucket per species)
  if (tid == 0) {
    int run = 0;
    for (int s = 0; s < MAX_S; ++s) {
      int b0 = 0, n = 0;
      if (s < S) { b0 = bstart[s * ncell + cell]; n = bstart[s * ncell + cell + 1] - b0; }
      cenStart[s] = b0; cenOff[s] = run; run += n;
    }
    cenOff[MAX_S] = run;
  }
  // ---- segment table: thread t <-> (species, neighbour cell offset)
  int len = 0, b0 = 0, code = 0;
  if (tid < S * 27) {
    const int s = tid / 27, r = tid - 27 * s;
    const int ox = r / 9 - 1, oy = (r / 3) % 3 - 1, oz = r % 3 - 1;
    bool ok = true;
    int nx = cx + ox, ny = cy + oy, nz = cz + oz;
    if (nc0 == 1) ok &= (ox == 0); else if (nx < 0 || nx >= nc0) { if (pbc) nx += (nx < 0) ? nc0 : -nc0; else ok = false; }
    if (nc1 == 1) ok &= (oy == 0); else if (ny < 0 || ny >= nc1) { if (pbc) ny += (ny < 0) ? nc1 : -nc1; else ok = false; }
    if (nc2 == 1) ok &= (oz == 0); else if (nz < 0 || nz >= nc2) { if (pbc) nz += (nz < 0) ? nc2 : -nc2; else ok = false; }
    if (ok) {
      const int k = s * ncell + (nx * nc1 + ny) * nc2 + nz;
      b0 = bstart[k]; len = bstart[k + 1] - b0;
      code = (ox + 1) | ((oy + 1) << 2) | ((oz + 1) << 4);
    }
  }
  int incl = len;
  for (int o = 1; o < 32; o <<= 1) { int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
  if (lane == 31) wsum[warp] = incl;
  __syncthreads();
  int base = 0;
  for (int w = 0; w < warp; ++w) base += wsum[w];
  if (tid < NB_SEG) {
    segStart[tid] = b0; segOff[tid] = base + incl - len; segCode[tid] = code;
    float sx, sy, sz;
    cell_shift(g->ev, (code & 3) - 1, ((code >> 2) & 3) - 1, ((code >> 4) & 3) - 1, sx, sy, sz);
    segSx[tid] = sx; segSy[tid] = sy; segSz[tid] = sz;
  }
  int total = 0;
  for (int w = 0; w < 8; ++w) total += wsum[w];
  if (tid == 0) segOff[NB_SEG] = total;
  __syncthreads();
  const int nC = cenOff[MAX_S];
  if (nC == 0) return;
  const unsigned lt = lanemask_lt();
  int bad = 0;

  for (int chunk0 = 0; chunk0 < total; chunk0 += NB_CAP) {
    const int nin = min(NB_CAP, total - chunk0);
    const int nin32 = (nin + 31) & ~31;   // the filter sweeps whole groups of 32: the tail holds far-away dummies
    if (chunk0 > 0) __syncthreads();
    // ---- stage the candidates of this chunk, shifted into the centre cell's frame
    {
      for (int idx = tid; idx < nin32; idx += 256) {
        if (idx >= nin) { cand[idx] = make_float4(1.0e18f, 1.0e18f, 1.0e18f, __int_as_float(0)); continue; }
        const int gq = chunk0 + idx;
        int lo = 0, hi = NB_SEG - 1;            // last segment with segOff <= gq
        while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (segOff[mid] <= gq) lo = mid; else hi = mid - 1; }
        const int jp = segStart[lo] + (gq - segOff[lo]), cd = segCode[lo];
        float4 pj = spos[jp];
        pj.x += segSx[lo]; pj.y += segSy[lo]; pj.z += segSz[lo];
        candA[idx] = __float_as_int(pj.w) & 0x0fffffff;
        pj.w = __int_as_float(jp | (cd << JBITS));
        cand[idx] = pj;
      }
    }
    __syncthreads();
    // ---- sweep: one warp per centre
    const bool wrap = pbc && (nc0 == 1 || nc1 == 1 || nc2 == 1);
    const float hi2 = (wide ? wide_r2 : c.Rcr2) + 2.0f * GUARD_BAND;
    unsigned short* sv = surv[warp];
    for (int ci = warp + 8 * blockIdx.y; ci < nC; ci += 8 * gridDim.y) {   // small systems: gridDim.y blocks share a cell
      int s = 0;
      while (s + 1 < MAX_S && ci >= cenOff[s + 1]) ++s;
      const int ip = cenStart[s] + (ci - cenOff[s]);
      const float4 pi = spos[ip];
      const int a_i = __float_as_int(pi.w) & 0x0fffffff;
      const int o_i = ml ? ml[a_i] : a_i;
      // ---- stage 1: cheap filter
      int ns = 0;
      {
        const float4* cp = cand + lane;
        for (int q0 = 0; q0 < nin32; q0 += 32, cp += 32) {
          const float4 pj = *cp;
          float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
          if (wrap) {   // block-uniform: a dimension with a single cell takes the minimum image per pair
            if (nc0 == 1) dx -= rintf(dx / ex) * ex;
            if (nc1 == 1) dy -= rintf(dy / ey) * ey;
            if (nc2 == 1) dz -= rintf(dz / ez) * ez;
          }
          const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
          const bool pass = d2 <= hi2;
          const unsigned m = __ballot_sync(0xffffffffu, pass);
          const int p = ns + __popc(m & lt);
          if (pass && p < SURV_CAP) sv[p] = (unsigned short)(q0 + lane);
          ns += __popc(m);
        }
      }
      if (ns > SURV_CAP) { bad |= FLAG_CAP; ns = SURV_CAP; }
      __syncwarp();
      // ---- stage 2: decide the survivors
      uint32_t* rR = nbrR + (size_t)ip * rcap;
      uint8_t* rA = nbrA + (size_t)ip * acap;
      int nR = 0, nA = 0, nW = 0;
      if (chunk0 > 0) { nR = cntR[ip]; nA = cntA[ip]; if (wide) nW = cntW[ip]; }
      for (int s0 = 0; s0 < ns; s0 += 32) {
        const bool live = s0 + lane < ns;
        const int q = live ? (int)sv[s0 + lane] : 0;
        const float4 pj = cand[q];
        uint32_t ent = (uint32_t)__float_as_int(pj.w);
        float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
        if (wrap) {
          if (nc0 == 1) { const int o = -(int)rintf(dx / ex); dx += (float)o * ex; ent += (uint32_t)o << JBITS; }
          if (nc1 == 1) { const int o = -(int)rintf(dy / ey); dy += (float)o * ey; ent += (uint32_t)(o * 4) << JBITS; }
          if (nc2 == 1) { const int o = -(int)rintf(dz / ez); dz += (float)o * ez; ent += (uint32_t)(o * 16) << JBITS; }
        }
        // row reuse (nnp_workspace_set_bin_reuse): the filter ran with the cut-off widened by the skin, and everything it
        // let through is kept as the centre's WIDE row, from which the rows of the following steps are decided
        if (wide && live && nW + s0 + lane < wcap) wide[(size_t)ip * wcap + nW + s0 + lane] = ent;
        decide32<TRIC>(c, g, pos, ml, live, dx, dy, dz, ent, candA[q], ip, o_i, lt, rR, rA, rcap, acap, nR, nA, bad);
      }
      if (nR > rcap || nA > acap) bad |= FLAG_CAP;
      if (wide) {
        if (nW + ns > wcap) bad |= FLAG_CAP;
        if (lane == 0) cntW[ip] = min(nW + ns, wcap);
      }
      if (lane == 0) { cntR[ip] = min(nR, rcap); cntA[ip] = min(nA, acap); }
      __syncwarp();
    }
  }
  if (bad) atomicOr(flags, bad);
}

// ---------------------------------------------------------------- K0-K1 as ONE cooperative kernel
// grid setup -> binning -> scan -> scatter -> bucket ordering are five dependent steps over < 1 MB: as separate
// launches each costs a launch + drain (~4 us); here they are phases of one persistent grid separated by grid-wide
// barriers.  Blocks of 1024 threads, one per SM at most (co-residency is what makes the barrier legal).
struct PrepArgs {
  AevConst c;
  GridInfo* grid; GroupInfo* groups; TileInfo* tiles;
  const float* pos; const int32_t* Z; const int32_t* ml;
  float4* tmp4; int* rank; int* cell_count; int* bstart; float4* spos; int* scell;
  unsigned long long* facc; int* flags;
  float Lx, Ly, Lz;
  int pbc, n_atoms, n_ml, max_cells, max_tiles, dense_k;
  int host_grid;   // 1: hg holds the cell grid (periodic boxes: computed on the host), no set-up phase
  GridInfo hg;
};

// CLUSTER = true: the whole grid is ONE thread-block cluster (<= 16 CTAs) and the phases are separated by the
// hardware cluster barrier (~0.2 us) -- these steps are latency-bound, a few SMs are plenty up to ~1e5 atoms.
// CLUSTER = false: cooperative launch over up to one CTA per SM with grid-wide barriers (larger systems).
template <bool CLUSTER>
__global__ void __launch_bounds__(1024, 1) k_prep(const __grid_constant__ PrepArgs a) {
  auto sync_all = [&]() {
    if (CLUSTER) cg::this_cluster().sync(); else cg::this_grid().sync();
  };
  const int S = a.c.S;
  const GridInfo* gbin = a.grid;
  if (a.host_grid) {   // binning reads the by-value copy; everybody else reads a.grid after the next barrier
    if (blockIdx.x == 0 && threadIdx.x == 0) *a.grid = a.hg;
    gbin = &a.hg;
  } else {
    if (blockIdx.x == 0)
      d_grid_setup(a.grid, a.groups, a.pbc, a.Lx, a.Ly, a.Lz, a.c.Rcr, a.max_cells, a.pos, a.ml, a.n_ml);
    sync_all();
  }
  const int nbA = (a.n_ml + (int)blockDim.x - 1) / (int)blockDim.x;
  for (int vb = blockIdx.x; vb < nbA; vb += gridDim.x)
    d_bin(vb, a.c, gbin, a.pos, a.Z, a.ml, a.n_atoms, a.n_ml, a.tmp4, a.rank, a.cell_count, a.facc, a.flags);
  sync_all();
  if (blockIdx.x == 0)
    d_scan(a.grid, a.cell_count, a.bstart, a.groups, a.tiles, S, a.n_ml, a.max_tiles, a.dense_k, a.flags);
  sync_all();
  for (int vb = blockIdx.x; vb < nbA; vb += gridDim.x)
    d_scatter(vb, a.grid, a.tmp4, a.rank, a.bstart, a.n_ml, a.spos, a.scell);
  sync_all();
  const int nbS = (S * a.grid->ncell * 32 + (int)blockDim.x - 1) / (int)blockDim.x;
  for (int vb = blockIdx.x; vb < nbS; vb += gridDim.x) d_bucket_sort(vb, a.grid, S, a.bstart, a.spos, a.tmp4);
}

// ---------------------------------------------------------------- external pair list
// "The 2026 version adds the internal pair-list built by GROMACS ... as available inputs."  With a
// list set (nnp_workspace_set_pair_list) K2's cell sweep is replaced by a filter over the engine's candidate pairs:
// every pair is decided by the pinned fp64 predicate on the original coordinates (so a Verlet-buffered superset gives
// exactly the rows of the cell search), appended to both rows, and the rows are then put in sorted-index order
// (species-major, reproducible) with the angular subset marked.  K0-K1 still run: the sort groups atoms by element.

// inv[ML-local index] = sorted position; row counters cleared
__global__ void __launch_bounds__(256) k_pair_index(const float4* __restrict__ spos, int n_ml, int* __restrict__ inv,
                                                    int* __restrict__ cntR) {
  const int ip = blockIdx.x * blockDim.x + threadIdx.x;
  if (ip >= n_ml) return;
  inv[__float_as_int(spos[ip].w) & 0x0fffffff] = ip;
  cntR[ip] = 0;
}

__device__ __forceinline__ int ml_local(const int32_t* __restrict__ ml, int n_ml, int gidx) {
  if (!ml) return (gidx >= 0 && gidx < n_ml) ? gidx : -1;
  int lo = 0, hi = n_ml - 1;
  while (lo < hi) { const int mid = (lo + hi) >> 1; if (ml[mid] < gidx) lo = mid + 1; else hi = mid; }
  return (n_ml > 0 && ml[lo] == gidx) ? lo : -1;
}

// one thread per candidate pair.  Like the cell sweep, the pair is decided in fp32 from the cell-local coordinates
// (displacement = local_j - local_i + cell offset * edge, the form the AEV kernels rebuild) and only a pair inside a
// guard band of the cut-off goes through the pinned fp64 predicate: no fp64 division for > 99 % of the candidates.
__global__ void __launch_bounds__(256)
k_pair_fill(AevConst c, const GridInfo* __restrict__ g, const float4* __restrict__ spos, const int* __restrict__ scell,
            const int* __restrict__ inv, const float* __restrict__ pos, const int32_t* __restrict__ ml, int n_ml,
            const int32_t* __restrict__ pairs, long long n_pairs, int rcap, uint32_t* __restrict__ nbrR,
            int* __restrict__ cntR, int* __restrict__ flags) {
  const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_pairs) return;
  const int gi = pairs[2 * p], gj = pairs[2 * p + 1];
  const int ai = ml_local(ml, n_ml, gi), aj = ml_local(ml, n_ml, gj);
  if (ai < 0 || aj < 0) return;             // a pair with a non-ML end does not feed the AEV
  if (ai == aj) { atomicOr(flags, FLAG_ARG); return; }
  const int ip = inv[ai], jp = inv[aj];
  const float4 pi = spos[ip], pj = spos[jp];
  const int ci = scell[ip], cj = scell[jp];
  const int nc[3] = {g->nc[0], g->nc[1], g->nc[2]};
  const int ic[3] = {ci / (nc[1] * nc[2]), (ci / nc[2]) % nc[1], ci % nc[2]};
  const int jc[3] = {cj / (nc[1] * nc[2]), (cj / nc[2]) % nc[1], cj % nc[2]};
  const float li[3] = {pi.x, pi.y, pi.z}, lj[3] = {pj.x, pj.y, pj.z};
  float dd[3];
  int offs[3];
  uint32_t code_i = 0u, code_j = 0u;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const float e = g->edge[a];
    float dl = lj[a] - li[a];
    int off;
    if (nc[a] == 1) {
      off = g->pbc ? -(int)rintf(dl / e) : 0;      // one cell: the minimum image of the pair
    } else {
      off = jc[a] - ic[a];
      if (g->pbc) { if (off == nc[a] - 1) off = -1; else if (off == 1 - nc[a]) off = 1; }
      if (off < -1 || off > 1) return;             // two cells apart: farther than the cut-off (edge >= Rcr)
    }
    dd[a] = dl;
    offs[a] = off;
    code_i |= (uint32_t)(off + 1) << (2 * a);
    code_j |= (uint32_t)(1 - off) << (2 * a);
  }
  {
    float sx, sy, sz;
    cell_shift(g->ev, offs[0], offs[1], offs[2], sx, sy, sz);
    dd[0] += sx; dd[1] += sy; dd[2] += sz;
  }
  const float d2 = fmaf(dd[2], dd[2], fmaf(dd[1], dd[1], dd[0] * dd[0]));
  bool in = d2 < c.Rcr2 - GUARD_BAND;
  if (fabsf(d2 - c.Rcr2) <= GUARD_BAND || d2 < 1e-6f) {
    const double e2 = exact_d2_any(pos, gi, gj, g);
    if (fabsf(d2 - c.Rcr2) <= GUARD_BAND) in = e2 <= c.Rcr2_d;
    if (e2 == 0.0) atomicOr(flags, FLAG_COINCIDENT);
  }
  if (!in) return;
  const int qi = atomicAdd(&cntR[ip], 1), qj = atomicAdd(&cntR[jp], 1);
  if (qi < rcap) nbrR[(size_t)ip * rcap + qi] = (uint32_t)jp | (code_i << JBITS);
  if (qj < rcap) nbrR[(size_t)jp * rcap + qj] = (uint32_t)ip | (code_j << JBITS);
  if (qi >= rcap || qj >= rcap) atomicOr(flags, FLAG_CAP);
}

// one warp per centre: order the row by sorted index (ranking by counting; a neighbour appears once), then the angular
// subset (fp32 decision on the row's own displacement, pinned fp64 predicate inside the guard band), in row order
__global__ void __launch_bounds__(256)
k_pair_rows(AevConst c, const GridInfo* __restrict__ g, const float4* __restrict__ spos, const float* __restrict__ pos,
            const int32_t* __restrict__ ml, int n_ml, int rcap, int acap, uint32_t* __restrict__ nbrR,
            uint8_t* __restrict__ nbrA, int* __restrict__ cntR, int* __restrict__ cntA, int* __restrict__ flags) {
  __shared__ uint32_t raw[8][RCAP_MAX], srt[8][RCAP_MAX];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int ip = blockIdx.x * 8 + w;
  if (ip >= n_ml) return;
  const int n = min(cntR[ip], rcap);
  uint32_t* row = nbrR + (size_t)ip * rcap;
  for (int q = lane; q < n; q += 32) raw[w][q] = row[q];
  __syncwarp();
  // keys below position q count with <=, keys above with <: a permutation even for a (faulty) repeated pair
  for (int q = lane; q < n; q += 32) {
    const uint32_t e = raw[w][q], key = e & JMASK;
    int rank = 0;
    for (int o = 0; o < q; ++o) rank += ((raw[w][o] & JMASK) <= key) ? 1 : 0;
    for (int o = q + 1; o < n; ++o) rank += ((raw[w][o] & JMASK) < key) ? 1 : 0;
    srt[w][rank] = e;
  }
  __syncwarp();
  int dup = 0;   // a pair listed twice shows up as equal neighbours in the ordered row
  for (int q = lane + 1; q < n; q += 32) dup |= ((srt[w][q] & JMASK) == (srt[w][q - 1] & JMASK)) ? 1 : 0;
  if (dup) atomicOr(flags, FLAG_ARG);
  const float4 pi = spos[ip];
  const int a_i = __float_as_int(pi.w) & 0x0fffffff;
  int nA = 0;
  for (int q0 = 0; q0 < n; q0 += 32) {
    const int q = q0 + lane;
    bool inA = false;
    if (q < n) {
      const uint32_t e = srt[w][q];
      row[q] = e;
      const float4 pj = spos[e & JMASK];
      const int oc = (int)(e >> JBITS);
      float sx, sy, sz;
      cell_shift(g->ev, (oc & 3) - 1, ((oc >> 2) & 3) - 1, ((oc >> 4) & 3) - 1, sx, sy, sz);
      const float dx = (pj.x - pi.x) + sx, dy = (pj.y - pi.y) + sy, dz = (pj.z - pi.z) + sz;
      const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
      inA = d2 < c.Rca2 - GUARD_BAND;
      if (fabsf(d2 - c.Rca2) <= GUARD_BAND) {
        const int a_j = __float_as_int(pj.w) & 0x0fffffff;
        inA = exact_d2_any(pos, ml ? ml[a_i] : a_i, ml ? ml[a_j] : a_j, g) <= c.Rca2_d;
      }
    }
    const unsigned m = __ballot_sync(0xffffffffu, inA);
    const int pA = nA + __popc(m & lanemask_lt());
    if (inA && pA < acap) nbrA[(size_t)ip * acap + pA] = (uint8_t)q;
    nA += __popc(m);
  }
  if (lane == 0) {
    cntR[ip] = n; cntA[ip] = min(nA, acap);
    if (nA > acap) atomicOr(flags, FLAG_CAP);
  }
}

// ---------------------------------------------------------------- binning reuse
// The evaluations between two full binnings keep the stored order (spos.w, scell, bstart, groups, tiles) and only
// re-read the positions: local coordinate = position relative to the atom's (old) cell, by the nearest image of the
// cell centre in fp64.  An atom may have drifted out of its cell by up to skin / 2 (the grid was cut with edges
// >= Rcr + skin, so neighbours within Rcr still sit in adjacent cells); beyond that the step is flagged stale.
__global__ void __launch_bounds__(256)
k_refresh(const GridInfo* __restrict__ g, const float* __restrict__ pos, const int32_t* __restrict__ ml, int n_ml,
          double half_skin, float4* __restrict__ spos, const int* __restrict__ scell, unsigned long long* __restrict__ facc,
          int* __restrict__ flags, const float4* __restrict__ spos_ref) {
  pdl_trigger();
  const int ip = blockIdx.x * blockDim.x + threadIdx.x;
  if (ip >= n_ml) return;
  const float w = spos[ip].w;
  const int a = __float_as_int(w) & 0x0fffffff;
  const size_t i = ml ? (size_t)ml[a] : (size_t)a;
  const int cell = scell[ip];
  const int nc1 = g->nc[1], nc2 = g->nc[2];
  const int cc[3] = {cell / (nc1 * nc2), (cell / nc2) % nc1, cell % nc2};
  float loc[3];
  bool stale = false;
  if (g->tric) {
    // fractional coordinates (as in the binning), offset from the cell centre in units of cells, nearest image
    const double x = (double)pos[3 * i], y = (double)pos[3 * i + 1], z = (double)pos[3 * i + 2];
    double sf[3], f[3];
    sf[2] = z / g->H_d[2];
    sf[1] = (y - sf[2] * g->H_d[5]) / g->H_d[1];
    sf[0] = (x - sf[1] * g->H_d[3] - sf[2] * g->H_d[4]) / g->H_d[0];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const double ncd = (double)g->nc[d];
      double t = sf[d] * ncd - ((double)cc[d] + 0.5);
      t -= ncd * rint(t / ncd);
      t += 0.5;
      // edge_d = distance between the cell's faces: the excursion beyond a face in Angstrom
      stale |= (t * g->edge_d[d] < -half_skin) || ((t - 1.0) * g->edge_d[d] > half_skin);
      f[d] = t;
    }
    loc[0] = (float)(f[0] * g->ev_d[0] + f[1] * g->ev_d[3] + f[2] * g->ev_d[6]);
    loc[1] = (float)(f[1] * g->ev_d[4] + f[2] * g->ev_d[7]);
    loc[2] = (float)(f[2] * g->ev_d[8]);
  } else {
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const double e = g->edge_d[d], L = g->L_d[d];
    double t = (double)pos[3 * i + d] - ((double)cc[d] + 0.5) * e;   // relative to the cell centre
    t -= L * rint(t / L);
    t += 0.5 * e;
    stale |= (t < -half_skin) || (t > e + half_skin);
    loc[d] = (float)t;
  }
  }
  if (spos_ref) {   // the ROWS are reused too: every pair within Rcr now must have been within Rcr + skin when the wide rows
                    // were built, i.e. no atom may have moved by more than skin / 2 since (same cell frame: plain difference)
    const float4 r = spos_ref[ip];
    const float ux = loc[0] - r.x, uy = loc[1] - r.y, uz = loc[2] - r.z;
    stale |= (double)(ux * ux + uy * uy + uz * uz) > half_skin * half_skin;
  }
  if (stale) atomicOr(flags, FLAG_STALE);
  spos[ip] = make_float4(loc[0], loc[1], loc[2], w);
  facc[3 * (size_t)ip + 0] = 0ull; facc[3 * (size_t)ip + 1] = 0ull; facc[3 * (size_t)ip + 2] = 0ull;
}

// Row reuse ("Verlet-buffered list reuse"; the engine's pair list lives
// for many steps): on the steps between two full builds the rows are decided from the stored WIDE rows (everything within
// Rcr + skin at build time) instead of the 27-cell sweep: one warp per centre, 32 wide entries at a time, the refreshed
// cell-local coordinates, and the same decision (decide32: fp32 outside the guard bands, pinned fp64 predicate inside) --
// so the rows are exactly those of a full build on the same order of atoms, at a fraction of the candidates (~80 / centre
// against 486).
template <bool TRIC>
__global__ void __launch_bounds__(256, 4)   // latency-bound (two dependent gathers per group): 64 registers, no spills
k_rows_from_wide(AevConst c, const GridInfo* __restrict__ g, const float4* __restrict__ spos, const float* __restrict__ pos,
                 const int32_t* __restrict__ ml, int n_ml, int rcap, int acap, const uint32_t* __restrict__ wide,
                 const int* __restrict__ cntW, int wcap, uint32_t* __restrict__ nbrR, uint8_t* __restrict__ nbrA,
                 int* __restrict__ cntR, int* __restrict__ cntA, int* __restrict__ flags) {
  pdl_trigger();
  pdl_wait();
  const int lane = threadIdx.x & 31, ip = blockIdx.x * 8 + (threadIdx.x >> 5);
  if (ip >= n_ml) return;
  float ev[9];
#pragma unroll
  for (int k = 0; k < 9; ++k) ev[k] = g->ev[k];
  const float4 pi = spos[ip];
  const int a_i = __float_as_int(pi.w) & 0x0fffffff;
  const int o_i = ml ? ml[a_i] : a_i;
  const unsigned lt = lanemask_lt();
  const int nW = cntW[ip];
  const uint32_t* wr = wide + (size_t)ip * wcap;
  uint32_t* rR = nbrR + (size_t)ip * rcap;
  uint8_t* rA = nbrA + (size_t)ip * acap;
  int nR = 0, nA = 0, bad = 0;
  // three groups of 32 entries per pass: all entry loads, then all position gathers in flight before the first decision
  // (the pass is a chain of two dependent global loads per group; a wide row of liquid water holds ~85 entries)
  for (int s0 = 0; s0 < nW; s0 += 96) {
    uint32_t ent[3];
    float4 pj[3];
#pragma unroll
    for (int u = 0; u < 3; ++u) ent[u] = (s0 + 32 * u + lane < nW) ? wr[s0 + 32 * u + lane] : (uint32_t)ip;
#pragma unroll
    for (int u = 0; u < 3; ++u) pj[u] = spos[ent[u] & JMASK];
#pragma unroll
    for (int u = 0; u < 3; ++u) {
      if (s0 + 32 * u < nW) {   // warp-uniform
        const int oc = (int)(ent[u] >> JBITS);
        float sx, sy, sz;
        cell_shift(ev, (oc & 3) - 1, ((oc >> 2) & 3) - 1, ((oc >> 4) & 3) - 1, sx, sy, sz);
        decide32<TRIC>(c, g, pos, ml, s0 + 32 * u + lane < nW, (pj[u].x - pi.x) + sx, (pj[u].y - pi.y) + sy, (pj[u].z - pi.z) + sz,
                       ent[u], __float_as_int(pj[u].w) & 0x0fffffff, ip, o_i, lt, rR, rA, rcap, acap, nR, nA, bad);
      }
    }
  }
  if (nR > rcap || nA > acap) bad |= FLAG_CAP;
  if (lane == 0) { cntR[ip] = min(nR, rcap); cntA[ip] = min(nA, acap); }
  if (bad) atomicOr(flags, bad);
}

// ---------------------------------------------------------------- host launcher
int cell_cap() { return CELL_CAP; }

// Largest cluster (16, else the portable 8) that can hold k_prep's 1024-thread CTAs on this device; 0 = none.
int prep_cluster_size() {
  cudaFuncSetAttribute((const void*)k_prep<true>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  for (int cs = 16; cs >= 8; cs >>= 1) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(cs); cfg.blockDim = dim3(1024);
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    int ncl = 0;
    if (cudaOccupancyMaxActiveClusters(&ncl, (const void*)k_prep<true>, &cfg) == cudaSuccess && ncl >= 1) return cs;
    cudaGetLastError();
  }
  return 0;
}

int launch_neighbor_stage(nnp_workspace* ws, const float* d_pos, const int32_t* d_Z, const float* box, int pbc,
                          const int32_t* d_ml, int64_t n_atoms, int64_t n_ml) {
  const nnp_model* m = ws->model;
  cudaStream_t st = ws->stream;
  // cell_count is all zero here: allocated zeroed, and the scan phase clears every count it reads
  PrepArgs a;
  a.c = m->aev;
  a.grid = ws->grid; a.groups = ws->groups; a.tiles = ws->tiles;
  a.pos = d_pos; a.Z = d_Z; a.ml = d_ml;
  a.tmp4 = ws->tmp4; a.rank = ws->rank; a.cell_count = ws->cell_count; a.bstart = ws->bstart; a.spos = ws->spos;
  a.scell = ws->scell; a.facc = ws->facc; a.flags = ws->flags;
  a.Lx = box[0]; a.Ly = box[4]; a.Lz = box[8];
  a.pbc = pbc; a.n_atoms = (int)n_atoms; a.n_ml = (int)n_ml; a.max_cells = ws->max_cells; a.max_tiles = ws->max_tiles;
  a.dense_k = ws->dense_k;
  a.host_grid = 0;
  // binning reuse: orthorhombic periodic boxes; the grid is cut skin wider on every step while it is switched on
  const bool reuse_ok = ws->reuse_every > 1 && pbc && n_ml > 0;
  const double skin = reuse_ok ? ws->reuse_skin * ws->len_scale : 0.0;
  bool same = reuse_ok && ws->reuse_left > 0 && ws->reuse_n_atoms == n_atoms && ws->reuse_n_ml == n_ml &&
              ws->reuse_ml == (const void*)d_ml && ws->reuse_Z == (const void*)d_Z;
  for (int k = 0; k < 9 && same; ++k) same = ws->reuse_box[k] == box[k];
  if (pbc && box_is_triclinic(box)) {
    grid_triclinic(&a.hg, box, (double)m->aev.Rcr * (1.0 + 1e-4) + skin, ws->max_cells);   // nnp_eval checked neighbor_box_ok
    a.host_grid = 1;
  } else if (pbc) {   // the cell grid of a periodic box needs no device data
    const double ext[3] = {(double)box[0], (double)box[4], (double)box[8]}, org[3] = {0.0, 0.0, 0.0};
    grid_from_extent(&a.hg, 1, ext, org, box[0], box[4], box[8], (double)m->aev.Rcr * (1.0 + 1e-4) + skin, ws->max_cells);
    a.host_grid = 1;
  }
  void* args[] = {&a};
  // fast binning (k_bin_cells + ranking inside k_neighbors): periodic boxes cut into >= 3 cells per dimension, own cell
  // search; a cell that overflowed its append buffer (NNP_ERR_CAPACITY) sends the workspace back to the general path
  // row reuse: own cell search only (an external pair list is itself the engine's buffered list)
  const bool rows_reuse = reuse_ok && !ws->ext_pairs && ws->wideR != nullptr;
  const bool tric_box = pbc && box_is_triclinic(box);
  const bool fast = a.host_grid && a.hg.nc[0] >= 3 && a.hg.nc[1] >= 3 && a.hg.nc[2] >= 3 && !ws->ext_pairs && !ws->slow_prep &&
                    a.hg.ncell <= ws->max_cells && a.hg.ncell <= FAST_MAX_CELLS;
  if (same || !fast) flush_pos_upload(ws);   // (k_bin_cells stages a pending upload itself)
  int extra = 0;   // kernels launched beyond the first
  bool fast_bin = false;   // this evaluation binned with k_bin_cells (k_neighbors clears its counters)
  if (same) {
    // refresh-only step: the stored order stays, positions are re-read (the grid on the device is the same one)
    --ws->reuse_left;
    k_refresh<<<(unsigned)((n_ml + 255) / 256), 256, 0, st>>>(ws->grid, d_pos, d_ml, (int)n_ml, 0.5 * skin, ws->spos, ws->scell,
                                                             ws->facc, ws->flags, rows_reuse ? ws->spos_ref : nullptr);
    if (rows_reuse) {   // the rows from the stored wide rows: no cell sweep on this step
      if (tric_box)
        launch_pdl(!ws->profiling, st, k_rows_from_wide<true>, dim3((unsigned)((n_ml + 7) / 8)), dim3(256), 0, m->aev, ws->grid, ws->spos,
                   d_pos, d_ml, (int)n_ml, ws->rcap, ws->acap, ws->wideR, ws->cntW, ws->wcap, ws->nbrR, ws->nbrA, ws->cntR, ws->cntA, ws->flags);
      else
        launch_pdl(!ws->profiling, st, k_rows_from_wide<false>, dim3((unsigned)((n_ml + 7) / 8)), dim3(256), 0, m->aev, ws->grid, ws->spos,
                   d_pos, d_ml, (int)n_ml, ws->rcap, ws->acap, ws->wideR, ws->cntW, ws->wcap, ws->nbrR, ws->nbrA, ws->cntR, ws->cntA, ws->flags);
      return 2;
    }
  } else {
  ws->inv_valid = 0;   // (set again below when k_cell_sort writes the inverse order)
  if (reuse_ok) {
    ws->reuse_left = ws->reuse_every - 1; ws->reuse_n_atoms = n_atoms; ws->reuse_n_ml = n_ml;
    ws->reuse_ml = d_ml; ws->reuse_Z = d_Z;
    for (int k = 0; k < 9; ++k) ws->reuse_box[k] = box[k];
  } else {
    ws->reuse_left = 0;
  }
  if (fast) {
    BinArgs b;
    b.c = m->aev; b.hg = a.hg; b.grid = ws->grid;
    b.pos = d_pos; b.Z = d_Z; b.ml = d_ml;
    b.cellbuf = ws->cellbuf; b.cellfill = ws->cellfill; b.cell_count = ws->cell_count; b.present = ws->present;
    b.facc = ws->facc; b.flags = ws->flags;
    b.n_atoms = (int)n_atoms; b.n_ml = (int)n_ml;
    b.pos_src = nullptr; b.pos_dst = nullptr;
    if (ws->pos_src_dev && !d_ml && d_pos == ws->hd_pos) {   // (the pending upload of nnp_eval_host: staged by the kernel)
      b.pos_src = ws->pos_src_dev; b.pos_dst = ws->hd_pos;
      ws->pos_src_host = nullptr; ws->pos_src_dev = nullptr;
    }
    k_bin_cells<<<(unsigned)((n_ml + BIN_THREADS - 1) / BIN_THREADS), BIN_THREADS, 0, st>>>(b);
    SortArgs q;
    q.groups = ws->groups; q.tiles = ws->tiles;
    q.cellbuf = ws->cellbuf; q.cell_count = ws->cell_count; q.present = ws->present;
    q.bstart = ws->bstart; q.spos = ws->spos; q.scell = ws->scell; q.flags = ws->flags; q.inv = ws->inv;
    q.S = m->aev.S; q.ncell = a.hg.ncell; q.n_ml = (int)n_ml; q.max_tiles = ws->max_tiles; q.dense_k = ws->dense_k;
    launch_pdl(!ws->profiling, st, k_cell_sort, dim3((unsigned)((a.hg.ncell + 7) / 8)), dim3(256), 0, q);
    fast_bin = true;
    extra = 1;
    ws->inv_valid = 1;
    // the MLP's layer-1 image check and operand prefetch: off the AEV -> MLP edge (mlp_tc.cu launch_tc_pack); stage
    // profiling keeps it with the MLP stage
    if (n_ml > 0 && !ws->profiling && !ws->ext_pairs) extra += launch_tc_pack(ws);
  } else if (ws->prep_cluster > 0 && n_ml <= ws->prep_cluster_max) {   // small systems: barrier latency dominates, a few SMs suffice
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(ws->prep_cluster); cfg.blockDim = dim3(1024); cfg.dynamicSmemBytes = 0; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = ws->prep_cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelExC(&cfg, (const void*)k_prep<true>, args);
  } else {
    // enough blocks for the atoms and the buckets, never more than one per SM (co-residency)
    const int64_t want = std::max<int64_t>((n_ml + 1023) / 1024, ((int64_t)m->aev.S * ws->max_cells * 32 + 1023) / 1024);
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(want, ws->num_sms));
    cudaLaunchCooperativeKernel((const void*)k_prep<false>, dim3(grid), dim3(1024), args, 0, st);
  }
  }
  int nl = 1 + extra;
  if (n_ml > 0 && ws->ext_pairs) {
    // external candidate pairs instead of the cell sweep (plain launches: fully ordered behind k_prep)
    k_pair_index<<<(unsigned)((n_ml + 255) / 256), 256, 0, st>>>(ws->spos, (int)n_ml, ws->rank, ws->cntR);
    if (ws->n_ext_pairs > 0)
      k_pair_fill<<<(unsigned)((ws->n_ext_pairs + 255) / 256), 256, 0, st>>>(m->aev, ws->grid, ws->spos, ws->scell, ws->rank, d_pos, d_ml,
                                                                            (int)n_ml, ws->ext_pairs, (long long)ws->n_ext_pairs,
                                                                            ws->rcap, ws->nbrR, ws->cntR, ws->flags);
    k_pair_rows<<<(unsigned)((n_ml + 7) / 8), 256, 0, st>>>(m->aev, ws->grid, ws->spos, d_pos, d_ml, (int)n_ml, ws->rcap, ws->acap,
                                                           ws->nbrR, ws->nbrA, ws->cntR, ws->cntA, ws->flags);
    return nl + 3;
  }
  if (n_ml > 0) {
    // one block per cell, guard on ncell inside.  Periodic boxes: the host knows the cell count; open boundaries: the
    // extent is only known on the device, one block per cell of the capacity.
    const int ncell_host = a.host_grid ? a.hg.ncell : ws->max_cells;
    // few atoms in few cells (a 96-atom box is ONE cell): several blocks per cell split its centres, or one SM does it all
    const int ysplit = (n_ml <= 2048) ? 8 : 1;
    const bool tric = a.host_grid && a.hg.tric;
    auto kern = tric ? k_neighbors<true> : k_neighbors<false>;
    launch_pdl(!ws->profiling, st, kern, dim3(ncell_host, ysplit), dim3(256), 0, m->aev, ws->grid, ws->groups, ws->spos,
               ws->bstart, d_pos, d_ml, (int)n_ml, ws->rcap, ws->acap, ws->nbrR, ws->nbrA, ws->cntR, ws->cntA, ws->flags,
               fast_bin ? ws->cell_count : nullptr, ws->cellfill, ws->present, rows_reuse ? ws->wideR : nullptr, ws->cntW, ws->wcap,
               (float)((m->aev.Rcr + skin) * (m->aev.Rcr + skin)));
    if (rows_reuse)   // reference positions of the displacement check on the reuse steps (a full step: 1 in every_n)
      cudaMemcpyAsync(ws->spos_ref, ws->spos, sizeof(float4) * (size_t)n_ml, cudaMemcpyDeviceToDevice, st);
    ++nl;
  }
  return nl;
}

}  // namespace nnp

TL_EXPORT(nnp_debug_step_timeline_neighbor)
