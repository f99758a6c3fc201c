// neighbor_common.cuh -- the pinned neighbour predicate (reading #6) and small helpers
// shared by the cell-list search (neighbor.cu) and the small-system front end (small.cu).
#pragma once
#include "nnp_internal.h"

namespace nnp {

__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// minimum-image displacement r_oj - r_oi and its squared length, the pinned fp64 expression of reading #6
__device__ __forceinline__ double exact_disp(const float* __restrict__ pos, int oi, int oj, const GridInfo* g, double d[3]) {
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    double x = (double)pos[3 * (size_t)oj + a] - (double)pos[3 * (size_t)oi + a];
    if (g->pbc) x -= g->L_d[a] * rint(x / g->L_d[a]);
    d[a] = x;
  }
  return __fma_rn(d[2], d[2], __fma_rn(d[1], d[1], __dmul_rn(d[0], d[0])));
}
__device__ __noinline__ inline double exact_d2(const float* __restrict__ pos, int oi, int oj, const GridInfo* g) {
  double d[3];
  return exact_disp(pos, oi, oj, g, d);
}

constexpr float GUARD_BAND = 2.0e-3f;  // Angstrom^2; >> fp32 error of d2 (~1e-5), reading #6


}  // namespace nnp
