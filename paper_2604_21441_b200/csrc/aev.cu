// aev.cu -- K3 of SURVEY.md section 8.a: radial + angular atomic environment vectors with cosine cut-offs
// (BASELINE.json north_star stage (2); formulas SURVEY.md Appendix A "Radial block", "Angular block").
//
// One warp per centre.  The neighbour row is sorted by species slot, so
//  * radial: lanes = 2 x 16 shifts, each half walks every other neighbour of one species segment;
//  * angular: every (s1 <= s2) species-pair block of triplets shares ONE 32-wide AEV block; lanes take
//    triplets, keep the 32 (ShfA x ShfZ) partial sums in registers, and one transposing butterfly reduces
//    them so that lane l ends with sub-feature l -> one coalesced 128-byte store per block.
// All summation orders are fixed by (row order, lane id): results are bitwise reproducible.
// Output rows are written in the compacted internal column order (nnp_internal.h GroupInfo).
#include "aev_forward.cuh"

namespace nnp {

__global__ void __launch_bounds__(AEV_FWD_WARPS * 32, 20)
k_aev_forward(AevConst c, const GridInfo* __restrict__ g, const GroupInfo* __restrict__ grp,
              const float4* __restrict__ spos, const uint32_t* __restrict__ nbrR, const uint8_t* __restrict__ nbrA,
              const int* __restrict__ cntR, const int* __restrict__ cntA, int n_ml, int rcap, int acap,
              float* __restrict__ aev) {
  __shared__ FwdEnv env[AEV_FWD_WARPS];
  TL_SCOPE(0);
  pdl_trigger();
  pdl_wait();
  TL_WAITED(0);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int ip = blockIdx.x * AEV_FWD_WARPS + w;
  if (ip >= n_ml) return;
  aev_forward_centre(c, g, grp, spos, nbrR + (size_t)ip * rcap, nbrA + (size_t)ip * acap, cntR[ip], cntA[ip], ip, aev, lane,
                     env[w]);
}

int launch_aev_forward(nnp_workspace* ws, int64_t n_ml) {
  if (n_ml <= 0) return 0;
  const nnp_model* m = ws->model;
  const int nb = (int)((n_ml + AEV_FWD_WARPS - 1) / AEV_FWD_WARPS);
  launch_pdl(!ws->profiling, ws->stream, k_aev_forward, dim3(nb), dim3(AEV_FWD_WARPS * 32), 0, m->aev, ws->grid, ws->groups,
             ws->spos, ws->nbrR, ws->nbrA, ws->cntR, ws->cntA, (int)n_ml, ws->rcap, ws->acap, ws->aev);
  return 1;
}

}  // namespace nnp

TL_EXPORT(nnp_debug_step_timeline_aev)
