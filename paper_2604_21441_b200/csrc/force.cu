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
#include "aev_backward.cuh"

namespace nnp {

#ifndef BWD_ROUNDS
#define BWD_ROUNDS 2
#endif
constexpr int BWD_CENTRES = AEV_WARPS * BWD_ROUNDS;   // centres of a LONG block: BWD_ROUNDS per warp, one after the other
// Block shapes.  A block's start-up (launch, pair table, flag poll, two barriers: ~1.5 us) is a tenth of a centre's time, so
// the first BWD_LONG_PCT % of the centres go to long blocks that pay it once for BWD_ROUNDS centres per warp; the rest -- the
// end of the grid -- stays one centre per warp, because long blocks at the end stretch the drain.  cfg 2, kernel alone /
// whole step (us): one round everywhere 83.7 / 247.2; two rounds everywhere 79.9 / 248.6 (the drain eats the gain);
// two rounds for 80 %, one for the rest 77.7 / 241.0; 70 %: 76.9 / 241.5; 90 %: 77.3 / 241.5; three rounds for 75 %: 77.0 /
// 241.4; four for 60 %: 76.5 / 241.3.  (The same for k_aev_forward, whose blocks have no such start-up: 66.2 -> 67.8 us.)

template <bool VIRIAL>
// 7 blocks of 4 warps per SM: 72 registers, 32 bytes of spills outside the triplet loop.  Alone the kernel gains little over
// 6 blocks / 80 registers (84.2 -> 83.5 us), but the step gains 5 us (253.4 -> 248.4 us, same box, alternating runs): while the
// MLP's second wave holds 40 SMs, the extra warps on the other 108 hide more of the gather latency.  (8 blocks / 64
// registers spill ~250 bytes per thread inside the triplet loop -- local-memory loads are long-scoreboard stalls: 95 us.)
__global__ void __launch_bounds__(AEV_WARPS * 32, 7)
k_aev_backward(AevConst c, const GridInfo* __restrict__ g, const GroupInfo* __restrict__ grp,
               const float4* __restrict__ spos, const uint32_t* __restrict__ nbrR, const uint8_t* __restrict__ nbrA,
               const int* __restrict__ cntR, const int* __restrict__ cntA, int n_ml, int rcap, int acap,
               const float* daev, unsigned long long* __restrict__ facc, long long* __restrict__ wcentre,
               const int* tile_done, int done_target, int* __restrict__ flags, int nb_long) {
  __shared__ BwdEnv env[AEV_WARPS];
  __shared__ int timed_out;
  __shared__ float Pacc[AEV_WARPS][ACAP_MAX][3];
  __shared__ int pairoff[MAX_S * MAX_S];   // (s1, s2) -> first float4 piece of the pair's dE/dAEV block
  TL_SCOPE(0);
  pdl_trigger();
  if (!tile_done) pdl_wait();   // with per-tile flags the MLP kernel is NOT awaited as a whole (see below)
  if (threadIdx.x == 0) timed_out = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  fill_pairoff(c, grp, pairoff);
  // Overlap with the MLP kernel (programmatic dependent launch): this grid may start while the persistent MLP CTAs
  // are still on their last tiles; a centre only needs ITS OWN row of dE/dAEV, so the block waits for the completion
  // flags of its centres' 128-row tiles (released by the MLP epilogue after the tile's last store) instead of the
  // whole kernel.  Thread t looks after centre t and polls only where the tile changes (the rows of a block are
  // contiguous: one poller per block almost always -- thousands of polling warps saturate the L2 slice that holds
  // the flags and slow the MLP's weight stream down).  dE/dAEV is read through ordinary (coherent) loads.
  // the first nb_long blocks take BWD_ROUNDS centres per warp, the others (the end of the grid: a short drain) one
  const int rounds = (int)blockIdx.x < nb_long ? BWD_ROUNDS : 1;
  const int ip0 = (int)blockIdx.x < nb_long ? (int)blockIdx.x * BWD_CENTRES : nb_long * BWD_CENTRES + ((int)blockIdx.x - nb_long) * AEV_WARPS;
  if (tile_done && threadIdx.x < rounds * AEV_WARPS) {
    const int ipw = ip0 + threadIdx.x;
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
  TL_WAITED(0);   // (here: the block's tile flags are up)
  if (timed_out) return;
#pragma unroll 1
  for (int r = 0; r < rounds; ++r) {
  const int ip = ip0 + r * AEV_WARPS + w;
  if (ip >= n_ml) return;
  const float4 ci = spos[ip];
  const int si = (__float_as_int(ci.w) >> 28) & 7;
  const int Kc = grp->Kc;
  // row of dE/dAEV in the piece-major tile layout: float4 piece q of this row = gb[q * TILE_M].  (Read through L1 where it
  // is needed: staging the row in shared memory first was measured twice -- round 1 and again with the packed
  // arithmetic, 86 -> 92 us -- and lost both times: extra registers across the gather and bank conflicts between the
  // lanes' different species-pair blocks.)
  const float4* gb = reinterpret_cast<const float4*>(daev + daev_off((size_t)(ip + grp->pad_shift[si]), 0, Kc));
  aev_backward_centre<VIRIAL>(c, g, grp, spos, nbrR + (size_t)ip * rcap, nbrA + (size_t)ip * acap, cntR[ip], cntA[ip], ip, gb, TILE_M,
                              facc, wcentre, lane, env[w], Pacc[w], pairoff);
  __syncwarp();
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
            double* __restrict__ virial, double e_scale, double f_scale, const int* __restrict__ inv) {
  __shared__ double wsum[8];
  __shared__ float fst[3 * 256];
  __shared__ long long vsum[8][9];
  __shared__ bool last;
  TL_SCOPE(1);
  pdl_trigger();
  pdl_wait();
  TL_WAITED(1);
  const int ip = blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
  double e = 0.0;
  const double sc = f_scale / 1099511627776.0;   // fixed point -> eV/Angstrom -> caller units
  if (inv) {
    // all atoms are ML atoms and the inverse order is at hand (k_cell_sort): thread <-> atom in the CALLER's order, its
    // accumulators gathered through inv, the block's 768 floats staged in shared memory and written as whole 128-byte
    // lines.  `forces` may then be the caller's pinned host buffer (nnp_eval_host): coalesced stores go over PCIe at
    // full rate, where one 12-byte row per thread in sorted order did not (measured: 0.298 -> 0.352 ms per step).
    const int a = ip;
    float f3[3] = {0.f, 0.f, 0.f};
    if (a < n_ml) {
      const size_t q = (size_t)inv[a];
#pragma unroll
      for (int d = 0; d < 3; ++d) f3[d] = (float)((double)(long long)facc[3 * q + d] * sc);
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) fst[3 * threadIdx.x + d] = f3[d];
    __syncthreads();
    const size_t base = (size_t)blockIdx.x * 768, lim = 3 * (size_t)n_ml;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const size_t idx = base + threadIdx.x + 256 * k;
      if (idx < lim) forces[idx] = fst[threadIdx.x + 256 * k];
    }
  }
  if (ip < n_ml) {
    const int w = __float_as_int(spos[ip].w);
    const int a = w & 0x0fffffff, slot = (w >> 28) & 7;
    if (!inv) {
      const size_t o = ml ? (size_t)ml[a] : (size_t)a;
#pragma unroll
      for (int d = 0; d < 3; ++d) forces[3 * o + d] = (float)((double)(long long)facc[3 * (size_t)ip + d] * sc);
    }
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
#ifndef BWD_LONG_PCT
#define BWD_LONG_PCT 80
#endif
    // (only where one-round blocks would run several waves anyway -- 7 blocks x 148 SMs hold 4144 centres: at 3000 atoms long
    // blocks turned one wave into two rounds, 89 -> 94 us per evaluation)
    const int nb_long = n_ml >= 8192 ? (int)(n_ml * BWD_LONG_PCT / 100 / BWD_CENTRES) : 0;
    const int nb = nb_long + (int)((n_ml - (int64_t)nb_long * BWD_CENTRES + AEV_WARPS - 1) / AEV_WARPS);
    // after the tcgen05 MLP kernel the launch is a programmatic dependent launch: blocks start on the SMs the
    // persistent MLP CTAs have left and wait per tile (see the kernel); stage profiling keeps the stages apart
    const int* done = ws->profiling ? nullptr : ws->tile_done;
    if (ws->d_virial)
      launch_pdl(done != nullptr, ws->stream, k_aev_backward<true>, dim3(nb), dim3(AEV_WARPS * 32), 0, m->aev, ws->grid,
                 ws->groups, ws->spos, ws->nbrR, ws->nbrA, ws->cntR, ws->cntA, (int)n_ml, ws->rcap, ws->acap, ws->daev,
                 ws->facc, ws->wcentre, done, ws->tile_done_target, ws->flags, nb_long);
    else
      launch_pdl(done != nullptr, ws->stream, k_aev_backward<false>, dim3(nb), dim3(AEV_WARPS * 32), 0, m->aev, ws->grid,
                 ws->groups, ws->spos, ws->nbrR, ws->nbrA, ws->cntR, ws->cntA, (int)n_ml, ws->rcap, ws->acap, ws->daev,
                 ws->facc, nullptr, done, ws->tile_done_target, ws->flags, nb_long);
    prof_mark(ws, 4);
    // forces in the caller's order through the inverse map, straight into the caller's pinned host buffer (nnp_eval_host
    // sets forces_alias), where there is such a map and no index subset
    // (only then: into device memory the gather through inv costs 0.8 us more than the scattered rows)
    const int* inv = (ws->inv_valid && !d_ml && ws->forces_alias) ? ws->inv : nullptr;
    float* fdst = d_forces;
    if (inv) { fdst = ws->forces_alias; ws->forces_in_alias = 1; }
    launch_pdl(!ws->profiling, ws->stream, k_force_out, dim3((unsigned)((n_ml + 255) / 256)), dim3(256), 0, ws->spos, ws->facc,
               d_ml, (int)n_ml, fdst, ws->groups, ws->e_atom, ws->epart, ws->ticket, d_energy, ws->wcentre, ws->wblk,
               ws->d_virial, ws->e_scale, ws->e_scale * ws->len_scale, inv);
    nl += 2;
  } else {
    cudaMemsetAsync(d_energy, 0, sizeof(double), ws->stream);
    if (ws->d_virial) cudaMemsetAsync(ws->d_virial, 0, 9 * sizeof(double), ws->stream);
  }
  return nl;
}

}  // namespace nnp

TL_EXPORT(nnp_debug_step_timeline_force)
