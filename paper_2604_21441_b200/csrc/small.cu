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
#include "aev_backward.cuh"
#include "aev_forward.cuh"
#include "groups.cuh"
#include "neighbor_common.cuh"
#include <algorithm>

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

template <int NW>   // NW = centres (warps at work in the row / AEV phase) per CTA
struct SmallFrontSmemT {
  FwdEnv env[NW];
  float4 sp[SMALL_MAX];                       // sorted: local xyz, w = ML-local index | slot << 28
  float4 tmp[SMALL_MAX];                      // unsorted positions
  uint32_t rowR_s[NW][RCAP_MAX];
  uint8_t rowA_s[NW][ACAP_MAX];
  uint8_t skey[SMALL_MAX];
  GridInfo g_s;
  GroupInfo grp_s;
  int cnt_s[MAX_S], gs[MAX_S + 1], pshift[MAX_S], tb[MAX_S + 1];
  int wcnt[SMALL_MAX / 32][MAX_S];            // atoms per (warp of the ordering phase, species)
};

// The centres of CTA b.  Plain: NW consecutive sorted indices.  ALIGNED (k_small_all): every species group is cut into
// chunks of NW of its own, so the centres of a CTA share one network (the MLP phase streams one set of weights) --
// gs = group starts; CTAs beyond the last chunk have no centres.
template <int NW, bool ALIGNED>
__device__ __forceinline__ void small_centres(const int* gs, int S, int n, int& ip_first, int& n_rows) {
  if (!ALIGNED) { ip_first = blockIdx.x * NW; n_rows = max(0, min(NW, n - ip_first)); return; }
  int b = blockIdx.x;
  ip_first = 0; n_rows = 0;
  for (int s = 0; s < S; ++s) {
    const int cnt = gs[s + 1] - gs[s], nb = (cnt + NW - 1) / NW;
    if (b < nb) { ip_first = gs[s] + b * NW; n_rows = min(NW, gs[s + 1] - ip_first); return; }
    b -= nb;
  }
}

// K0-K3 of the block's centres (whole block; no early exit: the single-kernel evaluation goes on afterwards).  facc =
// the accumulator array cleared here (sliced over the grid), or nullptr.
// TW > 1 (k_small_all): a team of TW warps per centre for the AEV row (aev_forward.cuh aev_forward_team): warp c < NW leads
// centre c, warps NW + (TW - 1) c .. are its helpers; team = the teams' staging.
template <int NW, bool ALIGNED, int TW = 1>
__device__ __forceinline__ void small_front(const SmallArgs& a, SmallFrontSmemT<NW>& sm, unsigned long long* facc,
                                            FwdTeam<TW>* team = nullptr) {
  FwdEnv* env = sm.env;
  float4* sp = sm.sp;
  uint32_t (*rowR_s)[RCAP_MAX] = sm.rowR_s;
  uint8_t (*rowA_s)[ACAP_MAX] = sm.rowA_s;
  uint8_t* skey = sm.skey;
  GridInfo& g_s = sm.g_s;
  GroupInfo& grp_s = sm.grp_s;
  int *cnt_s = sm.cnt_s, *gs = sm.gs, *pshift = sm.pshift, *tb = sm.tb;
  float4* tmp = sm.tmp;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int n = a.n_ml, S = a.c.S;
  const double L[3] = {(double)a.Lx, (double)a.Ly, (double)a.Lz};

  // ---- P0: species slot and local coordinates of atom `tid`; force accumulators cleared (sliced over the grid)
  int myslot = -1, pfx = 0;
  if (facc) for (int k = blockIdx.x * blockDim.x + tid; k < 3 * n; k += gridDim.x * blockDim.x) facc[k] = 0ull;
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
    myslot = slot;
  }
  // place inside the species group = atoms of the same species with a smaller ML index: per warp by ballot (pfx = the
  // lanes below), across warps by the per-warp counts
  if (w < SMALL_MAX / 32) {
    for (int q = 0; q < S; ++q) {
      const unsigned mq = __ballot_sync(0xffffffffu, myslot == q);
      if (myslot == q) pfx = __popc(mq & ((1u << lane) - 1u));
      if (lane == 0) sm.wcnt[w][q] = __popc(mq);
    }
  }
  __syncthreads();
  if (tid < MAX_S) {
    int t = 0;
    if (tid < S) for (int ww = 0; ww < SMALL_MAX / 32; ++ww) t += sm.wcnt[ww][tid];
    cnt_s[tid] = t;
  }
  __syncthreads();
  // ---- P1: groups, tiles, column map, the one-cell grid
  if (w == 0) {   // groups, tiles and the column set by one warp (d_groups_warp); the grid by a thread of the next warp
    if (lane == 0) {
      int run = 0;
      for (int q = 0; q <= MAX_S; ++q) { if (q <= S) gs[q] = run; if (q < S) run += cnt_s[q]; }
      for (int q = S + 1; q <= MAX_S; ++q) gs[q] = run;
    }
    __syncwarp();
    d_groups_warp(gs, S, n, a.max_tiles, a.dense_k, &grp_s, pshift, tb, a.flags);
  }
  if (tid == 32) {
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
    int rank = gs[slot] + pfx;
    for (int ww = 0; ww < w; ++ww) rank += sm.wcnt[ww][slot];
    float4 v = tmp[tid];
    v.w = __int_as_float(tid | (slot << 28));
    sp[rank] = v;
    a.spos[rank] = v;
    a.scell[rank] = 0;
  }
  __syncthreads();

  // ---- P3: neighbour rows of centre ip: all-pairs sweep, 32 candidates at a time (minimum image per pair)
  int ip_first, n_rows;
  small_centres<NW, ALIGNED>(gs, S, n, ip_first, n_rows);
  const int cidx = (TW == 1 || w < NW) ? w : (w - NW) / (TW > 1 ? TW - 1 : 1);   // centre this warp works for
  const int tw = (TW == 1 || w < NW) ? 0 : 1 + (w - NW) % (TW > 1 ? TW - 1 : 1);
  const int ip = ip_first + cidx;
  if (TW > 1 && tw > 0) {
    if (cidx < n_rows) aev_forward_team<TW>(a.c, &g_s, &grp_s, sp, nullptr, nullptr, 0, 0, ip, a.aev, lane, tw, 1 + cidx, env[cidx], team[cidx]);
  } else if (w < n_rows) {   // (k_small_front: warp <-> centre; warps beyond the centres wait at the next barrier)
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
  if (TW > 1) aev_forward_team<TW>(a.c, &g_s, &grp_s, sp, rowR_s[w], rowA_s[w], nR, nA, ip, a.aev, lane, 0, 1 + w, env[w], team[w]);
  else aev_forward_centre(a.c, &g_s, &grp_s, sp, rowR_s[w], rowA_s[w], nR, nA, ip, a.aev, lane, env[w]);
  }
}

__global__ void __launch_bounds__(SMALL_WARPS * 32, 1) k_small_front(SmallArgs a) {
  extern __shared__ __align__(16) uint8_t smraw[];
  SmallFrontSmemT<SMALL_WARPS>& sm = *reinterpret_cast<SmallFrontSmemT<SMALL_WARPS>*>(smraw);
  pdl_trigger();
  small_front<SMALL_WARPS, false>(a, sm, a.facc);
}

// ------------------------------------------------------------------------------------------------ the whole evaluation
// SURVEY.md section 8.f item 3 asks for "one cooperative/persistent kernel (or a single graph node) for n_ml <= ~300":
// PAPER.md lines 154 / 164 put the small-system cost into kernel launches and dispatch, and the ML regions of its ML/MM
// runs hold 14-107 atoms (lines 108, 140).  k_small_all is ONE launch without any grid-wide barrier, because every later
// stage of a centre needs only that centre's own data:
//   front    K0-K3 as above (per-CTA redundant ordering, rows and AEV of the CTA's centres: SA_R atoms of ONE species);
//   MLP      forward + backward of the CTA's centres on CUDA cores in fp32 (thread <-> neuron, the rows in registers,
//            activations in shared memory, weights streamed once per CTA from L2 through coalesced loads: transposed
//            copies for the forward layers) -- 2 x 10^5 MACs per atom is far too little for a tensor-core tile;
//   backward the AEV backward pass of the same centres (aev_backward_centre), fixed-point scatter into a private
//            accumulator that is zero between evaluations;
//   output   the last CTA to finish (ticket) converts the accumulators to forces, sums E in a fixed order and clears
//            the accumulator again.
// The MLP arithmetic of this path is plain fp32 (at least as accurate as the tensor-core modes).
constexpr int SA_R = 2;             // rows (centres) per CTA: the MLP phase is bound by the loads per FMA on ONE SM, so few rows, many CTAs
constexpr int SA_KSPLIT = 2;        // thread groups of 256 sharing the k loop of the MLP phase
static_assert(SA_R == 2 || SA_R % 4 == 0, "row vector loads");
constexpr int SA_THREADS = 256 * SA_KSPLIT;
constexpr int SA_TW = SA_THREADS / 32 / SA_R;   // warps per centre in the front end's AEV phase (a team: aev_forward.cuh)

struct SmallAllArgs {
  SmallArgs f;
  const NetTable* nets;             // DEVICE [n_members]
  int n_members;
  float* daev; float* e_atom;
  unsigned long long* acc;          // [SMALL_MAX * 3] fixed-point force accumulators, zero between evaluations
  unsigned int* ticket;
  float* forces; double* energy;
  double e_scale, f_scale;
  int zero_forces;                  // 1: an ML subset -- the rows of the other atoms are written as +0.0f here
};

__device__ __forceinline__ float celu_s(float x, float alpha) { return x > 0.f ? x : alpha * (__expf(x / alpha) - 1.0f); }
__device__ __forceinline__ float celu_grad_s(float a, float alpha) { return a > 0.f ? 1.0f : a / alpha + 1.0f; }

// out[n][r] = sum_k B(k, n) in[k][r] for the SA_R rows r, thread <-> n, B(k, n) = Bp[kidx(k) * sk + n]
// with consecutive n contiguous (coalesced).  in / out: [index][SA_R rows] in shared memory.  MAPK / MAPN: k / n runs over the
// compact AEV columns and the weight is addressed by the internal column.
template <bool MAPK, bool MAPN, class Epi>
__device__ __forceinline__ void dense_rows(const float* __restrict__ Bp, int sk, int K, int N, const float* __restrict__ in,
                                       const int* __restrict__ blkmap, float* __restrict__ part, int n0, Epi epi) {
  // Phase A: thread <-> (four consecutive n, k group): the 8 thread groups of 64 take four k of every 32-wide k block each,
  // weights as 128-bit loads (four neurons per load: a quarter of the load instructions of a thread-per-neuron mapping --
  // on ONE SM the phase is bound by load instructions, not by FMAs), two k blocks (8 loads) in flight per thread.
  // Phase B: the partial sums meet in shared memory (part[k group][n][row]); thread <-> n adds the 8 groups in order.
  static_assert(SA_R == 2 && SA_THREADS == 512, "dense_rows mapping");
  const int n4 = threadIdx.x & 63, kg = threadIdx.x >> 6;
  const int n = n0 + 4 * n4;
  float acc[4][SA_R];
#pragma unroll
  for (int j = 0; j < 4; ++j)
#pragma unroll
    for (int r = 0; r < SA_R; ++r) acc[j][r] = 0.f;
  if (n < N) {
    const int ncol = MAPN ? blkmap[n >> 5] * BLK + (n & 31) : n;
    for (int k0 = 0; k0 < K; k0 += 64) {     // K is a multiple of 32 (hidden widths, compact AEV blocks)
      float4 wv[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int k = k0 + 32 * (u >> 2) + 4 * kg + (u & 3);
        const int kr = MAPK ? blkmap[min(k, K - 1) >> 5] * BLK + (k & 31) : k;
        wv[u] = k < K ? __ldg(reinterpret_cast<const float4*>(Bp + (size_t)kr * sk + ncol)) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int k = min(k0 + 32 * (u >> 2) + 4 * kg + (u & 3), K - 1);
        const float2 x = *reinterpret_cast<const float2*>(in + k * SA_R);
        acc[0][0] = fmaf(wv[u].x, x.x, acc[0][0]); acc[0][1] = fmaf(wv[u].x, x.y, acc[0][1]);
        acc[1][0] = fmaf(wv[u].y, x.x, acc[1][0]); acc[1][1] = fmaf(wv[u].y, x.y, acc[1][1]);
        acc[2][0] = fmaf(wv[u].z, x.x, acc[2][0]); acc[2][1] = fmaf(wv[u].z, x.y, acc[2][1]);
        acc[3][0] = fmaf(wv[u].w, x.x, acc[3][0]); acc[3][1] = fmaf(wv[u].w, x.y, acc[3][1]);
      }
    }
#pragma unroll
    for (int j = 0; j < 4; ++j)
      *reinterpret_cast<float2*>(part + ((size_t)kg * 256 + 4 * n4 + j) * SA_R) = make_float2(acc[j][0], acc[j][1]);
  }
  __syncthreads();
  const int nl = threadIdx.x, nn = n0 + nl;
  if (nl < 256 && nn < N) {
    float o[SA_R] = {0.f, 0.f};
#pragma unroll
    for (int g8 = 0; g8 < 8; ++g8) {
      const float2 v = *reinterpret_cast<const float2*>(part + ((size_t)g8 * 256 + nl) * SA_R);
      o[0] += v.x; o[1] += v.y;
    }
    epi(nn, o);
  }
}

// forward + backward of the network of species s for the CTA's rows (centres ip_first .. ip_first + n_rows - 1).
// mb = shared-memory floats: x[Kc][R], h1..h3[HP][R], d3..d1[HP][R], red[warps][R], part[8][256][R]  (R = SA_R rows)
__device__ __forceinline__ void small_mlp(const SmallAllArgs& a, const GroupInfo& grp, int s, int ip_first, int n_rows, float* mb) {
  const int tid = threadIdx.x, lane = tid & 31, wp = tid >> 5;
  const int Kc = grp.Kc;
  float* xs = mb;
  float* h1 = xs + (size_t)Kc * SA_R;
  float* h2 = h1 + HP * SA_R;
  float* h3 = h2 + HP * SA_R;
  float* d3 = h3 + HP * SA_R;
  float* d2 = d3 + HP * SA_R;
  float* d1 = d2 + HP * SA_R;
  float* red = d1 + HP * SA_R;                 // [warps][8]
  float* part = red + (SA_THREADS / 32) * SA_R;   // [8 k groups][256][SA_R]
  const float escale = 1.0f / (float)a.n_members;
  {
    int rowof[SA_R];
#pragma unroll
    for (int r = 0; r < SA_R; ++r) rowof[r] = r < n_rows ? ip_first + r + grp.pad_shift[s] : -1;
    for (int mem = 0; mem < a.n_members; ++mem) {
      const Net& net = a.nets[mem].net[s];
      if (net.n_layers != 4) continue;    // (no network: the front end has flagged the species)
      const int N1 = net.dims[1], N2 = net.dims[2], N3 = net.dims[3], Kfull = net.dims[0];
      const float alpha = net.alpha;
      __syncthreads();
      // x = the rows' AEV, transposed to [k][row]; rows of other species are zero
      for (int idx = tid; idx < Kc * SA_R; idx += blockDim.x) {
        const int r = idx / Kc, k = idx - r * Kc;
        xs[k * SA_R + r] = rowof[r] >= 0 ? __ldcg(a.f.aev + (size_t)rowof[r] * Kc + k) : 0.f;
      }
      __syncthreads();
      dense_rows<true, false>(net.WT[0], N1, Kc, N1, xs, grp.blkmap, part, 0, [&](int nn, const float* acc) {
        const float b = __ldg(net.b[0] + nn);
#pragma unroll
        for (int r = 0; r < SA_R; ++r) h1[nn * SA_R + r] = celu_s(acc[r] + b, alpha);
      });
      __syncthreads();
      dense_rows<false, false>(net.WT[1], N2, N1, N2, h1, grp.blkmap, part, 0, [&](int nn, const float* acc) {
        const float b = __ldg(net.b[1] + nn);
#pragma unroll
        for (int r = 0; r < SA_R; ++r) h2[nn * SA_R + r] = celu_s(acc[r] + b, alpha);
      });
      __syncthreads();
      dense_rows<false, false>(net.WT[2], N3, N2, N3, h2, grp.blkmap, part, 0, [&](int nn, const float* acc) {
        const float b = __ldg(net.b[2] + nn);
#pragma unroll
        for (int r = 0; r < SA_R; ++r) h3[nn * SA_R + r] = celu_s(acc[r] + b, alpha);
      });
      __syncthreads();
      // output layer: E_r = w4 . h3[.][r] + b4 (fixed-order reduction: lane tree, then the warps in order);
      // d3 = escale w4 CELU'(h3)
      {
        float ep[SA_R];
#pragma unroll
        for (int r = 0; r < SA_R; ++r) ep[r] = 0.f;
        for (int nn = tid; nn < N3; nn += blockDim.x) {
          const float w4 = __ldg(net.W[3] + nn);
#pragma unroll
          for (int r = 0; r < SA_R; ++r) {
            const float h = h3[nn * SA_R + r];
            ep[r] = fmaf(w4, h, ep[r]);
            d3[nn * SA_R + r] = escale * w4 * celu_grad_s(h, alpha);
          }
        }
#pragma unroll
        for (int r = 0; r < SA_R; ++r) {
          for (int o = 16; o > 0; o >>= 1) ep[r] += __shfl_xor_sync(0xffffffffu, ep[r], o);
          if (lane == 0) red[wp * SA_R + r] = ep[r];
        }
        __syncthreads();
        if (tid < SA_R && rowof[tid] >= 0) {
          float e = 0.f;
          for (int w2 = 0; w2 < (int)(blockDim.x >> 5); ++w2) e += red[w2 * SA_R + tid];
          const float ev = escale * (e + __ldg(net.b[3]));
          a.e_atom[rowof[tid]] = mem > 0 ? a.e_atom[rowof[tid]] + ev : ev;
        }
      }
      // backward: d2 = (W3^T d3) * CELU'(h2), d1 = (W2^T d2) * CELU'(h1), g = W1^T d1
      dense_rows<false, false>(net.W[2], N2, N3, N2, d3, grp.blkmap, part, 0, [&](int kk, const float* acc) {
#pragma unroll
        for (int r = 0; r < SA_R; ++r) d2[kk * SA_R + r] = acc[r] * celu_grad_s(h2[kk * SA_R + r], alpha);
      });
      __syncthreads();
      dense_rows<false, false>(net.W[1], N1, N2, N1, d2, grp.blkmap, part, 0, [&](int kk, const float* acc) {
#pragma unroll
        for (int r = 0; r < SA_R; ++r) d1[kk * SA_R + r] = acc[r] * celu_grad_s(h1[kk * SA_R + r], alpha);
      });
      __syncthreads();
      for (int n0 = 0; n0 < Kc; n0 += 256) {   // the compact AEV may be wider than the 256 threads of a group
        dense_rows<false, true>(net.W[0], Kfull, N1, Kc, d1, grp.blkmap, part, n0, [&](int kk, const float* acc) {
#pragma unroll
          for (int r = 0; r < SA_R; ++r)
            if (rowof[r] >= 0) {
              float* o = a.daev + daev_off((size_t)rowof[r], kk, Kc);
              *o = mem > 0 ? *o + acc[r] : acc[r];
            }
        });
        __syncthreads();   // part is reused by the next chunk
      }
    }
  }
  __syncthreads();
}

struct SmallBwdSmem {
  BwdEnv env[SA_R];
  BwdTeam<SA_TW> team[SA_R];
  int pairoff[MAX_S * MAX_S];
};

__global__ void __launch_bounds__(SA_THREADS, 1) k_small_all(const __grid_constant__ SmallAllArgs a) {
  extern __shared__ __align__(16) uint8_t smraw[];
  using Front = SmallFrontSmemT<SA_R>;
  Front& sm = *reinterpret_cast<Front*>(smraw);
  float* mb = reinterpret_cast<float*>(smraw + ((sizeof(Front) + 15) & ~(size_t)15));   // MLP staging, then the backward staging
  __shared__ bool last;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int n = a.f.n_ml;
  // rows of the other atoms of an ML subset are +0.0f (sliced over the grid; the ML rows are written by the last CTA,
  // after every CTA's ticket -- i.e. after all of this)
  if (a.zero_forces)
    for (int k = blockIdx.x * blockDim.x + tid; k < 3 * a.f.n_atoms; k += gridDim.x * blockDim.x) a.forces[k] = 0.f;
  // (the teams' staging shares the MLP staging: the front end is over before the MLP phase starts)
  small_front<SA_R, true, SA_TW>(a.f, sm, nullptr, reinterpret_cast<FwdTeam<SA_TW>*>(mb));
  __syncthreads();
  int ip_first, n_rows;
  small_centres<SA_R, true>(sm.gs, a.f.c.S, n, ip_first, n_rows);
  if (n_rows > 0) small_mlp(a, sm.grp_s, (__float_as_int(sm.sp[ip_first].w) >> 28) & 7, ip_first, n_rows, mb);   // block-uniform
  // ---- AEV backward of the CTA's centres (the dE/dAEV rows were written by this CTA: visible after the barrier)
  SmallBwdSmem& sb = *reinterpret_cast<SmallBwdSmem*>(mb);
  fill_pairoff(a.f.c, &sm.grp_s, sb.pairoff);
  __syncthreads();
  // a team of SA_TW warps per centre, as in the front end: warp c < SA_R leads centre c
  const int cidx = (w < SA_R) ? w : (w - SA_R) / (SA_TW - 1), tw = (w < SA_R) ? 0 : 1 + (w - SA_R) % (SA_TW - 1);
  const int ip = ip_first + cidx;
  if (cidx < n_rows) {
    const int si = (__float_as_int(sm.sp[ip].w) >> 28) & 7;
    const int Kc = sm.grp_s.Kc;
    const float4* gb = reinterpret_cast<const float4*>(a.daev + daev_off((size_t)(ip + sm.grp_s.pad_shift[si]), 0, Kc));
    // (rows from global memory: the MLP staging has taken the place of the front end's shared copies)
    aev_backward_team<SA_TW>(a.f.c, &sm.g_s, &sm.grp_s, sm.sp, a.f.nbrR + (size_t)ip * a.f.rcap, a.f.nbrA + (size_t)ip * a.f.acap,
                             a.f.cntR[ip], a.f.cntA[ip], ip, gb, TILE_M, a.acc, lane, tw, 1 + cidx, sb.env[cidx], sb.team[cidx],
                             sb.pairoff);
  }
  // ---- output by the last CTA to get here
  __threadfence();
  __syncthreads();
  if (tid == 0) last = (atomicAdd(a.ticket, 1u) == gridDim.x - 1);
  __syncthreads();
  if (!last) return;
  __threadfence();
  const double sc = a.f_scale / 1099511627776.0;   // 2^-40 fixed point -> eV / Angstrom -> caller units
  for (int q = tid; q < n; q += blockDim.x) {
    const int wv = __float_as_int(sm.sp[q].w);
    const int al = wv & 0x0fffffff;
    const size_t o = a.f.ml ? (size_t)a.f.ml[al] : (size_t)al;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      a.forces[3 * o + d] = (float)((double)(long long)__ldcg(a.acc + 3 * (size_t)q + d) * sc);
      a.acc[3 * (size_t)q + d] = 0ull;             // zero again for the next evaluation
    }
  }
  if (w == 0) {   // E = sum of the per-atom energies in a fixed order (lane-strided partial sums, shuffle tree), fp64
    double e = 0.0;
    for (int q = lane; q < n; q += 32) {
      const int slot = (__float_as_int(sm.sp[q].w) >> 28) & 7;
      e += (double)__ldcg(a.e_atom + q + sm.grp_s.pad_shift[slot]);
    }
    for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    if (lane == 0) { *a.energy = e * a.e_scale; *a.ticket = 0u; }
  }
}

size_t small_all_smem(const nnp_model* m) {
  const size_t front = (sizeof(SmallFrontSmemT<SA_R>) + 15) & ~(size_t)15;
  const size_t mlp = ((size_t)m->Kfull * SA_R + 6 * (size_t)HP * SA_R + (SA_THREADS / 32) * SA_R + (size_t)8 * 256 * SA_R) * sizeof(float);
  return front + std::max(std::max(mlp, sizeof(SmallBwdSmem)), SA_R * sizeof(FwdTeam<SA_TW>));
}

// the single-kernel evaluation takes what the front end takes, with the tensor-core-shaped networks (four layers,
// widths multiples of 32), no virial output and no stage profiling (there are no stages to time)
bool small_all_applicable(const nnp_workspace* ws, const float* box, int pbc, int64_t n_ml) {
  return small_front_applicable(ws, box, pbc, n_ml) && ws->small_all && ws->model->tc && ws->model->d_nets && !ws->d_virial &&
         !ws->profiling && ws->small_acc != nullptr;
}

int launch_small_all(nnp_workspace* ws, const float* d_pos, const int32_t* d_Z, const float* box, const int32_t* d_ml,
                     int64_t n_atoms, int64_t n_ml, double* d_energy, float* d_forces) {
  const nnp_model* m = ws->model;
  SmallAllArgs a;
  SmallArgs& f = a.f;
  f.c = m->aev;
  f.grid = ws->grid; f.groups = ws->groups; f.tiles = ws->tiles;
  f.pos = d_pos; f.Z = d_Z; f.ml = d_ml;
  f.spos = ws->spos; f.scell = ws->scell; f.bstart = ws->bstart; f.facc = ws->facc;
  f.nbrR = ws->nbrR; f.nbrA = ws->nbrA; f.cntR = ws->cntR; f.cntA = ws->cntA;
  f.aev = ws->aev; f.flags = ws->flags;
  f.Lx = box[0]; f.Ly = box[4]; f.Lz = box[8];
  f.n_atoms = (int)n_atoms; f.n_ml = (int)n_ml; f.max_tiles = ws->max_tiles; f.dense_k = ws->dense_k;
  f.rcap = ws->rcap; f.acap = ws->acap;
  a.nets = m->d_nets; a.n_members = m->n_members;
  a.daev = ws->daev; a.e_atom = ws->e_atom; a.acc = ws->small_acc; a.ticket = ws->small_ticket;
  a.forces = d_forces; a.energy = d_energy;
  a.e_scale = ws->e_scale; a.f_scale = ws->e_scale * ws->len_scale;
  a.zero_forces = d_ml != nullptr;
  // one CTA per chunk of SA_R atoms of one species: at most n / SA_R + S chunks (the counts are only known on the device;
  // a CTA beyond the last chunk does the ordering and goes straight to the ticket)
  k_small_all<<<(unsigned)(n_ml / SA_R + m->aev.S), SA_THREADS, ws->small_all_smem, ws->stream>>>(a);
  return 1;
}

int small_all_prepare(nnp_workspace* ws) {
  ws->small_all_smem = small_all_smem(ws->model);
  return (cudaFuncSetAttribute(k_small_all, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ws->small_all_smem) == cudaSuccess &&
          cudaFuncSetAttribute(k_small_front, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SmallFrontSmemT<SMALL_WARPS>)) == cudaSuccess)
             ? NNP_OK : NNP_ERR_CUDA;
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
  k_small_front<<<(unsigned)((n_ml + SMALL_WARPS - 1) / SMALL_WARPS), SMALL_WARPS * 32, sizeof(SmallFrontSmemT<SMALL_WARPS>), ws->stream>>>(a);
  return 1;
}

}  // namespace nnp
