// small.cu -- the front end of one evaluation (K0-K3: species map, ordering, neighbour rows, AEV) as ONE kernel for
// small periodic ML regions ("Small-N latency path -- the regime the paper says matters
// most for ML/MM": 14-107 ML atoms; plateau analysis lines 154, 164).
//
// For <= 256 ML atoms the four dependent launches of the general path (k_prep's five barrier-separated phases,
// k_neighbors, k_aev_forward) cost far more in launch / barrier latency than in work.  Here every CTA repeats the
// cheap part redundantly in its own shared memory -- species slots, positions relative to the first ML atom (fp64
// minimum image, rounded to fp32), ordering by (slot, ML index) through ranking by counting (reproducible, no
// atomics), groups / tiles / column map -- so NO grid-wide synchronisation is needed; then each of its 8 warps takes one
// centre: all-pairs sweep over the shared-memory copy of the sorted positions (same fp32 pre-filter + pinned fp64
// guard-band predicate as k_neighbors, so the rows are bit-identical to the oracle's O(N^2) list) and, straight
// away, that centre's AEV row.  The whole box is treated as ONE cell (edge = box length): the image of a neighbour is
// the per-pair minimum image, exactly the single-cell case of the general path.  Everything the later stages read
// (spos, rows, groups, tiles, grid) is written in the general path's layout; CTAs write identical values.
#include "aev_forward.cuh"
#include "groups.cuh"
#include "neighbor_common.cuh"

namespace nnp {

constexpr int SMALL_MAX = 256;       // ML atoms (one per thread in the ordering phases)
constexpr int SMALL_WARPS = 8;       // centres per CTA
constexpr float SMALL_MAX_BOX = 64.f;  // Angstrom: positions are held relative to ONE origin in fp32 (error <= 4e-6 A)

struct SmallArgs {
  AevConst c;
  GridInfo* grid; GroupInfo* groups; TileInfo* tiles;
  const float* pos; const int32_t* Z; const int32_t* ml;
  float4* spos; int* scell; int* bstart;
  unsigned long long* facc;
  uint32_t* nbrR; uint8_t* nbrA; int* cntR; int* cntA;
  float* aev; int* flags;
  float Lx, Ly, Lz;
  int n_atoms, n_ml, max_tiles, dense_k, rcap, acap;
};

__global__ void __launch_bounds__(SMALL_WARPS * 32, 1) k_small_front(SmallArgs a) {
  __shared__ FwdEnv env[SMALL_WARPS];
  __shared__ float4 sp[SMALL_MAX];                       // sorted: local xyz, w = ML-local index | slot << 28
  __shared__ uint32_t rowR_s[SMALL_WARPS][RCAP_MAX];     // first the unsorted positions (float4 tmp[SMALL_MAX]), then rows
  __shared__ uint8_t rowA_s[SMALL_WARPS][ACAP_MAX];
  __shared__ uint8_t skey[SMALL_MAX];
  __shared__ GridInfo g_s;
  __shared__ GroupInfo grp_s;
  __shared__ int cnt_s[MAX_S], gs[MAX_S + 1], pshift[MAX_S], tb[MAX_S + 1];
  static_assert(sizeof(float4) * SMALL_MAX <= sizeof(uint32_t) * SMALL_WARPS * RCAP_MAX, "tmp aliases the row staging");
  float4* tmp = reinterpret_cast<float4*>(&rowR_s[0][0]);
  pdl_trigger();
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int n = a.n_ml, S = a.c.S;
  const double L[3] = {(double)a.Lx, (double)a.Ly, (double)a.Lz};

  // ---- P0: species slot and local coordinates of atom `tid`; force accumulators cleared (sliced over the grid)
  if (tid < MAX_S) cnt_s[tid] = 0;
  for (int k = blockIdx.x * blockDim.x + tid; k < 3 * n; k += gridDim.x * blockDim.x) a.facc[k] = 0ull;
  __syncthreads();
  if (tid < n) {
    int i = tid;
    if (a.ml) {
      i = a.ml[tid];
      const bool bad = (i < 0 || i >= a.n_atoms) || (tid > 0 && a.ml[tid - 1] >= i);
      if (bad) { atomicOr(a.flags, FLAG_ARG); i = min(max(i, 0), a.n_atoms - 1); }
    }
    int i0 = a.ml ? min(max(a.ml[0], 0), a.n_atoms - 1) : 0;
    const int z = a.Z[i];
    int slot = (z >= 0 && z < 128) ? (int)a.c.zlut[z] : -1;
    if (slot < 0) { atomicOr(a.flags, FLAG_SPECIES); slot = 0; }
    float loc[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      double x = (double)a.pos[3 * (size_t)i + d] - (double)a.pos[3 * (size_t)i0 + d];
      x -= L[d] * rint(x / L[d]);
      loc[d] = (float)x;
    }
    tmp[tid] = make_float4(loc[0], loc[1], loc[2], 0.f);
    skey[tid] = (uint8_t)slot;
    atomicAdd(&cnt_s[slot], 1);   // integer count: order free
  }
  __syncthreads();
  // ---- P1: groups, tiles, column map, the one-cell grid
  if (tid == 0) {
    int run = 0;
    for (int q = 0; q <= MAX_S; ++q) { if (q <= S) gs[q] = run; if (q < S) run += cnt_s[q]; }
    for (int q = S + 1; q <= MAX_S; ++q) gs[q] = run;
    d_groups(gs, S, n, a.max_tiles, a.dense_k, &grp_s, pshift, tb, a.flags);
    g_s.nc[0] = g_s.nc[1] = g_s.nc[2] = 1; g_s.ncell = 1; g_s.pbc = 1; g_s.tric = 0;
    for (int k = 0; k < 9; ++k) { g_s.ev[k] = 0.f; g_s.ev_d[k] = 0.0; }
    for (int k = 0; k < 6; ++k) g_s.H_d[k] = (k < 3) ? L[k] : 0.0;
    for (int d = 0; d < 3; ++d) {
      g_s.edge[d] = (float)L[d]; g_s.edge_d[d] = L[d]; g_s.inv_edge_d[d] = 1.0 / L[d]; g_s.origin_d[d] = 0.0;
      g_s.L_d[d] = L[d]; g_s.L[d] = (float)L[d];
      g_s.ev[4 * d] = (float)L[d]; g_s.ev_d[4 * d] = L[d];
    }
  }
  __syncthreads();
  d_tiles(gs, pshift, tb, S, a.max_tiles, a.tiles);
  {
    // publish (every CTA writes the same values)
    const int* src = reinterpret_cast<const int*>(&grp_s);
    int* dst = reinterpret_cast<int*>(a.groups);
    for (int k = tid; k < (int)(sizeof(GroupInfo) / sizeof(int)); k += blockDim.x) dst[k] = src[k];
    const int* gsrc = reinterpret_cast<const int*>(&g_s);
    int* gdst = reinterpret_cast<int*>(a.grid);
    for (int k = tid; k < (int)(sizeof(GridInfo) / sizeof(int)); k += blockDim.x) gdst[k] = gsrc[k];
    if (tid <= S) a.bstart[tid] = gs[tid];
  }
  // ---- P2: order by (slot, ML index): rank by counting
  if (tid < n) {
    const int slot = skey[tid];
    int rank = gs[slot];
    for (int b = 0; b < tid; ++b) rank += (skey[b] == slot) ? 1 : 0;
    float4 v = tmp[tid];
    v.w = __int_as_float(tid | (slot << 28));
    sp[rank] = v;
    a.spos[rank] = v;
    a.scell[rank] = 0;
  }
  __syncthreads();   // tmp (= the row staging) is free from here on

  // ---- P3: neighbour rows of centre ip: all-pairs sweep, 32 candidates at a time (minimum image per pair)
  const int ip = blockIdx.x * SMALL_WARPS + w;
  if (ip >= n) return;
  const float4 pi = sp[ip];
  const int a_i = __float_as_int(pi.w) & 0x0fffffff;
  const int o_i = a.ml ? a.ml[a_i] : a_i;
  const float ex = g_s.edge[0], ey = g_s.edge[1], ez = g_s.edge[2];
  const float Rcr2 = a.c.Rcr2, Rca2 = a.c.Rca2, loR = a.c.Rcr2 - GUARD_BAND, loA = a.c.Rca2 - GUARD_BAND;
  const unsigned lt = lanemask_lt();
  uint32_t* rowR = a.nbrR + (size_t)ip * a.rcap;
  uint8_t* rowA = a.nbrA + (size_t)ip * a.acap;
  int nR = 0, nA = 0, bad = 0;
  for (int q0 = 0; q0 < n; q0 += 32) {
    const int q = q0 + lane;
    const float4 pj = (q < n) ? sp[q] : make_float4(1.0e18f, 1.0e18f, 1.0e18f, 0.f);
    float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
    uint32_t ent = (uint32_t)q | (21u << JBITS);   // cell offset code (1,1,1) = the same image
    if (q < n) {
      const int ox = -(int)rintf(dx / ex), oy = -(int)rintf(dy / ey), oz = -(int)rintf(dz / ez);
      dx += (float)ox * ex; dy += (float)oy * ey; dz += (float)oz * ez;
      ent += (uint32_t)(ox + 4 * oy + 16 * oz) << JBITS;
    }
    const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    const bool other = q != ip && q < n;
    bool inR = other && d2 < loR, inA = other && d2 < loA;
    // guard bands (and coincident atoms): the pinned fp64 predicate on the original coordinates decides
    const bool near = other && (fabsf(d2 - Rcr2) <= GUARD_BAND || fabsf(d2 - Rca2) <= GUARD_BAND || d2 < 1e-6f);
    if (near) {
      const int a_j = __float_as_int(pj.w) & 0x0fffffff;
      const double e2 = exact_d2(a.pos, o_i, a.ml ? a.ml[a_j] : a_j, &g_s);
      if (fabsf(d2 - Rcr2) <= GUARD_BAND) inR = e2 <= a.c.Rcr2_d;
      if (fabsf(d2 - Rca2) <= GUARD_BAND) inA = e2 <= a.c.Rca2_d;
      if (e2 == 0.0) bad |= FLAG_COINCIDENT;
    }
    const unsigned mR = __ballot_sync(0xffffffffu, inR);
    const unsigned mA = __ballot_sync(0xffffffffu, inA);
    const int pR = nR + __popc(mR & lt), pA = nA + __popc(mA & lt);
    if (inR && pR < a.rcap) { rowR[pR] = ent; rowR_s[w][pR] = ent; }
    if (inA && pA < a.acap && pR < a.rcap) { rowA[pA] = (uint8_t)pR; rowA_s[w][pA] = (uint8_t)pR; }
    nR += __popc(mR); nA += __popc(mA);
  }
  if (nR > a.rcap || nA > a.acap) bad |= FLAG_CAP;
  nR = min(nR, a.rcap); nA = min(nA, a.acap);
  if (lane == 0) { a.cntR[ip] = nR; a.cntA[ip] = nA; }
  if (bad) atomicOr(a.flags, bad);
  __syncwarp();
  // ---- P4: this centre's AEV row, from the shared-memory copies of positions, rows, grid and groups
  aev_forward_centre(a.c, &g_s, &grp_s, sp, rowR_s[w], rowA_s[w], nR, nA, ip, a.aev, lane, env[w]);
}

bool small_front_applicable(const nnp_workspace* ws, const float* box, int pbc, int64_t n_ml) {
  return ws->small_path && pbc && !box_is_triclinic(box) && n_ml > 0 && n_ml <= SMALL_MAX && !ws->ext_pairs && ws->rcap <= RCAP_MAX &&
         ws->acap <= ACAP_MAX && box[0] <= SMALL_MAX_BOX && box[4] <= SMALL_MAX_BOX && box[8] <= SMALL_MAX_BOX;
}

// replaces launch_neighbor_stage + launch_aev_forward; returns the number of kernels launched
int launch_small_front(nnp_workspace* ws, const float* d_pos, const int32_t* d_Z, const float* box,
                       const int32_t* d_ml, int64_t n_atoms, int64_t n_ml) {
  const nnp_model* m = ws->model;
  SmallArgs a;
  a.c = m->aev;
  a.grid = ws->grid; a.groups = ws->groups; a.tiles = ws->tiles;
  a.pos = d_pos; a.Z = d_Z; a.ml = d_ml;
  a.spos = ws->spos; a.scell = ws->scell; a.bstart = ws->bstart; a.facc = ws->facc;
  a.nbrR = ws->nbrR; a.nbrA = ws->nbrA; a.cntR = ws->cntR; a.cntA = ws->cntA;
  a.aev = ws->aev; a.flags = ws->flags;
  a.Lx = box[0]; a.Ly = box[4]; a.Lz = box[8];
  a.n_atoms = (int)n_atoms; a.n_ml = (int)n_ml; a.max_tiles = ws->max_tiles; a.dense_k = ws->dense_k;
  a.rcap = ws->rcap; a.acap = ws->acap;
  k_small_front<<<(unsigned)((n_ml + SMALL_WARPS - 1) / SMALL_WARPS), SMALL_WARPS * 32, 0, ws->stream>>>(a);
  return 1;
}

}  // namespace nnp
