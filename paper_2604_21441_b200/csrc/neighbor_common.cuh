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

// Squared minimum-image distance |r_oj - r_oi|^2, the pinned fp64 expression of reading #6 (orthorhombic boxes and open
// boundaries).  Kept small: it is called out of line from the hot candidate sweeps, and a callee that needs many
// registers makes its callers spill around the call.
__device__ __noinline__ inline double exact_d2(const float* __restrict__ pos, int oi, int oj, const GridInfo* g) {
  double d[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    double x = (double)pos[3 * (size_t)oj + a] - (double)pos[3 * (size_t)oi + a];
    if (g->pbc) x = __dsub_rn(x, __dmul_rn(g->L_d[a], rint(x / g->L_d[a])));
    d[a] = x;
  }
  return __fma_rn(d[2], d[2], __fma_rn(d[1], d[1], __dmul_rn(d[0], d[0])));
}

// The same for a triclinic box (reading #35): row-by-row reduction c, b, a, then the nearest of the 27 surrounding
// images -- the operations of the oracle's disp() in the same order, no contraction.
__device__ __noinline__ inline double exact_d2_tric(const float* __restrict__ pos, int oi, int oj, const GridInfo* g) {
  double d[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) d[a] = (double)pos[3 * (size_t)oj + a] - (double)pos[3 * (size_t)oi + a];
  const double ax = g->H_d[0], by = g->H_d[1], cz = g->H_d[2], bx = g->H_d[3], cx = g->H_d[4], cy = g->H_d[5];
  double n = rint(d[2] / cz);
  d[2] = __dsub_rn(d[2], __dmul_rn(cz, n)); d[1] = __dsub_rn(d[1], __dmul_rn(cy, n)); d[0] = __dsub_rn(d[0], __dmul_rn(cx, n));
  n = rint(d[1] / by);
  d[1] = __dsub_rn(d[1], __dmul_rn(by, n)); d[0] = __dsub_rn(d[0], __dmul_rn(bx, n));
  n = rint(d[0] / ax);
  d[0] = __dsub_rn(d[0], __dmul_rn(ax, n));
  double best = __fma_rn(d[2], d[2], __fma_rn(d[1], d[1], __dmul_rn(d[0], d[0])));
  for (int nc = -1; nc <= 1; ++nc)
    for (int nb = -1; nb <= 1; ++nb)
      for (int na = -1; na <= 1; ++na) {
        double v0 = d[0], v1 = d[1], v2 = d[2];
        v2 = __dadd_rn(v2, __dmul_rn(cz, (double)nc)); v1 = __dadd_rn(v1, __dmul_rn(cy, (double)nc)); v0 = __dadd_rn(v0, __dmul_rn(cx, (double)nc));
        v1 = __dadd_rn(v1, __dmul_rn(by, (double)nb)); v0 = __dadd_rn(v0, __dmul_rn(bx, (double)nb));
        v0 = __dadd_rn(v0, __dmul_rn(ax, (double)na));
        const double q = __fma_rn(v2, v2, __fma_rn(v1, v1, __dmul_rn(v0, v0)));
        if (q < best) best = q;
      }
  return best;
}

// either, by the grid's box type (for the kernels that are not register-critical)
__device__ __forceinline__ double exact_d2_any(const float* __restrict__ pos, int oi, int oj, const GridInfo* g) {
  return g->tric ? exact_d2_tric(pos, oi, oj, g) : exact_d2(pos, oi, oj, g);
}

constexpr float GUARD_BAND = 2.0e-3f;  // Angstrom^2; >> fp32 error of d2 (~1e-5), reading #6


}  // namespace nnp
