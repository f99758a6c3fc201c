// link.cu -- link atoms at the ML/MM boundary (section 3, eq. 4): placement
//     r_L = r_ML + d (r_MM - r_ML) / |r_MM - r_ML|
// before the evaluation, and redistribution of the force on the link atom onto the two bonded atoms by the chain
// rule after it:  with l = |r_MM - r_ML|, u the unit bond vector,
//     F_ML += F_L - (d/l)(F_L - u (u.F_L)),   F_MM += (d/l)(F_L - u (u.F_L)).
// Link atoms occupy rows n_atoms .. n_atoms + n_links - 1 of the position / force arrays; the caller lists them in
// the ML index with the link element's atomic number (hydrogen by default).  Bond vectors take the minimum image in
// periodic boxes.  A handful of links per system: one thread per link for the placement; the spread walks the links
// in order in ONE thread, so that atoms bonded to several links accumulate in a fixed order (reproducible).
#include "nnp_internal.h"

namespace nnp {

// box rows a = (ax,0,0), b = (bx,by,0), c = (cx,cy,cz) (GROMACS; orthorhombic: bx = cx = cy = 0)
struct LinkBox { float ax, by, cz, bx, cx, cy; };

__device__ __forceinline__ bool link_bond(const float* __restrict__ pos, int a, int b, int pbc, LinkBox B, double* u, double& l) {
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < 3; ++k) u[k] = (double)pos[3 * (size_t)b + k] - (double)pos[3 * (size_t)a + k];
  if (pbc) {   // bond image: row-by-row reduction c, b, a (a bond is far shorter than half a box width)
    double n = rint(u[2] / (double)B.cz);
    u[2] -= (double)B.cz * n; u[1] -= (double)B.cy * n; u[0] -= (double)B.cx * n;
    n = rint(u[1] / (double)B.by);
    u[1] -= (double)B.by * n; u[0] -= (double)B.bx * n;
    n = rint(u[0] / (double)B.ax);
    u[0] -= (double)B.ax * n;
  }
#pragma unroll
  for (int k = 0; k < 3; ++k) s += u[k] * u[k];
  l = sqrt(s);
  if (!(l > 0.0)) return false;
#pragma unroll
  for (int k = 0; k < 3; ++k) u[k] /= l;
  return true;
}

__global__ void k_link_place(int n_atoms, int n_links, const int32_t* __restrict__ link_ml,
                             const int32_t* __restrict__ link_mm, double d, int pbc, LinkBox B,
                             float* __restrict__ pos) {
  const int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= n_links) return;
  const int a = link_ml[q], b = link_mm[q];
  if (a < 0 || a >= n_atoms || b < 0 || b >= n_atoms) return;   // validated on the host side of the caller
  double u[3], l;
  if (!link_bond(pos, a, b, pbc, B, u, l)) return;
#pragma unroll
  for (int k = 0; k < 3; ++k) pos[3 * (size_t)(n_atoms + q) + k] = (float)((double)pos[3 * (size_t)a + k] + d * u[k]);
}

__global__ void k_link_spread(int n_atoms, int n_links, const int32_t* __restrict__ link_ml,
                              const int32_t* __restrict__ link_mm, double d, int pbc, LinkBox B,
                              const float* __restrict__ pos, float* __restrict__ forces) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  for (int q = 0; q < n_links; ++q) {
    const int a = link_ml[q], b = link_mm[q];
    if (a < 0 || a >= n_atoms || b < 0 || b >= n_atoms) continue;
    double u[3], l;
    if (!link_bond(pos, a, b, pbc, B, u, l)) continue;
    float* FL = forces + 3 * (size_t)(n_atoms + q);
    const double f[3] = {(double)FL[0], (double)FL[1], (double)FL[2]};
    const double uf = u[0] * f[0] + u[1] * f[1] + u[2] * f[2];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const double perp = (d / l) * (f[k] - u[k] * uf);
      forces[3 * (size_t)a + k] = (float)((double)forces[3 * (size_t)a + k] + (f[k] - perp));
      forces[3 * (size_t)b + k] = (float)((double)forces[3 * (size_t)b + k] + perp);
      FL[k] = 0.f;
    }
  }
}

}  // namespace nnp

using namespace nnp;

static int link_args_ok(int64_t n_atoms, int64_t n_links, const void* a, const void* b, const float* box, int pbc,
                        const void* p, double d) {
  if (n_atoms < 0 || n_links < 0 || !(d > 0.0) || n_atoms + n_links >= (1ll << 31)) return NNP_ERR_INVALID_ARG;
  if (n_links > 0 && (!a || !b || !p)) return NNP_ERR_INVALID_ARG;
  if (pbc) {
    if (!box) return NNP_ERR_INVALID_ARG;
    for (int r = 0; r < 3; ++r)
      for (int c = 0; c < 3; ++c) {
        const float v = box[3 * r + c];
        if (r == c ? !(v > 0.f) : (c > r && v != 0.f)) return NNP_ERR_BOX_UNSUPPORTED;   // lower-triangular rows
      }
    if (fabsf(box[3]) > 0.5f * box[0] || fabsf(box[6]) > 0.5f * box[0] || fabsf(box[7]) > 0.5f * box[4]) return NNP_ERR_BOX_UNSUPPORTED;
  }
  return NNP_OK;
}
static LinkBox link_box(const float* box, int pbc) {
  if (!pbc) return LinkBox{1.f, 1.f, 1.f, 0.f, 0.f, 0.f};
  return LinkBox{box[0], box[4], box[8], box[3], box[6], box[7]};
}

extern "C" int nnp_link_place(void* cuda_stream, int64_t n_atoms, int64_t n_links, const int32_t* d_link_ml,
                              const int32_t* d_link_mm, double d, const float box[9], int32_t pbc, float* d_pos) {
  int rc = link_args_ok(n_atoms, n_links, d_link_ml, d_link_mm, box, pbc, d_pos, d);
  if (rc || n_links == 0) return rc;
  k_link_place<<<(int)((n_links + 127) / 128), 128, 0, (cudaStream_t)cuda_stream>>>(
      (int)n_atoms, (int)n_links, d_link_ml, d_link_mm, d, pbc ? 1 : 0, link_box(box, pbc), d_pos);
  return cudaGetLastError() == cudaSuccess ? NNP_OK : NNP_ERR_CUDA;
}

extern "C" int nnp_link_spread(void* cuda_stream, int64_t n_atoms, int64_t n_links, const int32_t* d_link_ml,
                               const int32_t* d_link_mm, double d, const float box[9], int32_t pbc, const float* d_pos,
                               float* d_forces) {
  int rc = link_args_ok(n_atoms, n_links, d_link_ml, d_link_mm, box, pbc, d_pos, d);
  if (rc || n_links == 0) return rc;
  if (!d_forces) return NNP_ERR_INVALID_ARG;
  k_link_spread<<<1, 32, 0, (cudaStream_t)cuda_stream>>>((int)n_atoms, (int)n_links, d_link_ml, d_link_mm, d, pbc ? 1 : 0,
                                                         link_box(box, pbc), d_pos, d_forces);
  return cudaGetLastError() == cudaSuccess ? NNP_OK : NNP_ERR_CUDA;
}
