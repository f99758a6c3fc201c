// mlp_simt.cu -- K5/K6 on CUDA cores in plain fp32 (NNP_MLP_FP32_SIMT): the reference rung of the precision
// ladder and the path for network shapes the tensor-core kernel does not take.
// Network and backward: SURVEY.md Appendix A "Network", "Backward"; CELU' is recovered from the activation
// (a > 0 -> 1, else a/alpha + 1).
//
// Rows are the element-grouped, tile-padded AEV rows (GroupInfo / TileInfo); one block = one 128-row tile of
// one element x 64 output columns.  Layer 0 reads / the last backward GEMM writes the compacted AEV column
// order; weights of layer 0 are stored in the internal full order, so columns go through blkmap.
#include "nnp_internal.h"

namespace nnp {

constexpr int SM_BM = 128, SM_BN = 64, SM_BK = 16;

__device__ __forceinline__ float celu_f(float x, float alpha) { return x > 0.f ? x : alpha * (__expf(x / alpha) - 1.0f); }
__device__ __forceinline__ float celu_grad_from_act(float a, float alpha) { return a > 0.f ? 1.0f : a / alpha + 1.0f; }

// out[r][n] = epilogue( sum_k in[r][k] * B(k,n) ),  B(k,n) = Bp[kmap(k)*sk + nmap(n)*sn]
//  mode 0: forward  hidden layer l : + bias, CELU                       (in = a_l, out = a_{l+1})
//  mode 1: backward hidden layer l : * CELU'(act[r][n])                 (in = dz_l, out = dz_{l-1})
//  mode 2: backward layer 0        : raw                                (in = dz_0, out = daev)
__global__ void __launch_bounds__(256)
k_dense(NetTable nets, const GroupInfo* __restrict__ grp, const TileInfo* __restrict__ tiles, int layer, int mode,
        const float* __restrict__ in, int ldin, float* __restrict__ out, int ldout, const float* __restrict__ act,
        int ldact, int accumulate) {
  if ((int)blockIdx.x >= grp->n_tiles) return;
  const TileInfo ti = tiles[blockIdx.x];
  const Net& net = nets.net[ti.slot];
  if (net.n_layers == 0) return;
  const bool kmap = (mode == 0 && layer == 0), nmap = (mode == 2);
  const float* __restrict__ Bp = net.W[layer];
  const int Kc = grp->Kc;
  if (ldin == 0) ldin = Kc;     // pitch 0 = "the compacted AEV pitch", only known on the device
  if (ldout == 0) ldout = Kc;
  const int wld = net.dims[layer];  // row stride of W[layer] ([out][in]; layer 0: internal padded width)
  int K, N, sk, sn;
  if (mode == 0) { K = (layer == 0) ? Kc : net.dims[layer]; N = net.dims[layer + 1]; sk = 1; sn = wld; }
  else { K = net.dims[layer + 1]; N = (layer == 0) ? Kc : net.dims[layer]; sk = wld; sn = 1; }
  const int n0 = blockIdx.y * SM_BN;
  if (n0 >= N) return;
  __shared__ float As[SM_BK][SM_BM + 4];
  __shared__ float Bs[SM_BK][SM_BN + 4];
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  float acc[8][4];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
  for (int k0 = 0; k0 < K; k0 += SM_BK) {
    // A tile: 128 rows x 16 k
    for (int idx = tid; idx < SM_BM * SM_BK; idx += 256) {
      const int r = idx / SM_BK, kk = idx % SM_BK;
      const int k = k0 + kk;
      As[kk][r] = (k < K && r < ti.nvalid) ? in[(size_t)(ti.row0 + r) * ldin + k] : 0.f;
    }
    for (int idx = tid; idx < SM_BN * SM_BK; idx += 256) {
      int kk, nn;
      if (mode == 0) { nn = idx / SM_BK; kk = idx % SM_BK; } else { kk = idx / SM_BN; nn = idx % SM_BN; }
      const int k = k0 + kk, n = n0 + nn;
      float v = 0.f;
      if (k < K && n < N) {
        const int km = kmap ? grp->blkmap[k >> 5] * BLK + (k & 31) : k;
        const int nm = nmap ? grp->blkmap[n >> 5] * BLK + (n & 31) : n;
        v = Bp[(size_t)km * sk + (size_t)nm * sn];
      }
      Bs[kk][nn] = v;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < SM_BK; ++kk) {
      float a[8], b[4];
#pragma unroll
      for (int i = 0; i < 8; ++i) a[i] = As[kk][ty * 8 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Bs[kk][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int r = ty * 8 + i;
    if (r >= ti.nvalid) continue;
    const size_t row = (size_t)(ti.row0 + r);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int n = n0 + tx * 4 + j;
      if (n >= N) continue;
      float v = acc[i][j];
      if (mode == 0) v = celu_f(v + net.b[layer][n], net.alpha);
      else if (mode == 1) v *= celu_grad_from_act(act[row * ldact + n], net.alpha);
      if (mode == 2) { float* o = out + daev_off(row, n, ldout); *o = accumulate ? *o + v : v; }   // ensemble: sum over members
      else out[row * ldout + n] = v;
    }
  }
}

// Last (linear) layer: E_i = w . a + b, and dz of the last hidden layer = w * CELU'(a).  One warp per row.
// n_layers == 1: the input is the AEV itself and dE/dAEV = w (mapped columns).
__global__ void __launch_bounds__(256)
k_last(NetTable nets, const GroupInfo* __restrict__ grp, const TileInfo* __restrict__ tiles,
       const float* __restrict__ in, int ldin, float* __restrict__ e_atom, float* __restrict__ dz, int lddz,
       float scale, int accumulate) {
  if ((int)blockIdx.x >= grp->n_tiles) return;
  const TileInfo ti = tiles[blockIdx.x];
  const Net& net = nets.net[ti.slot];
  const int nl = net.n_layers;
  if (nl == 0) return;
  const float* __restrict__ w = net.W[nl - 1];
  const int K = (nl == 1) ? grp->Kc : net.dims[nl - 1];
  const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
  if (ldin == 0) ldin = grp->Kc;
  if (lddz == 0) lddz = grp->Kc;
  for (int r = wp; r < TILE_M; r += 8) {
    const size_t row = (size_t)(ti.row0 + r);
    if (r >= ti.nvalid) { if (lane == 0 && !accumulate) e_atom[row] = 0.f; continue; }
    float s = 0.f;
    for (int k = lane; k < K; k += 32) {
      const int km = (nl == 1) ? grp->blkmap[k >> 5] * BLK + (k & 31) : k;
      const float a = in[row * ldin + k], wk = w[km];
      s = fmaf(a, wk, s);
      if (nl == 1) { float* o = dz + daev_off(row, k, lddz); *o = accumulate ? *o + scale * wk : scale * wk; }
      else dz[row * lddz + k] = scale * wk * celu_grad_from_act(a, net.alpha);
    }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) { const float ev = scale * (s + net.b[nl - 1][0]); e_atom[row] = accumulate ? e_atom[row] + ev : ev; }
  }
}

int launch_mlp_simt(nnp_workspace* ws, int64_t n_ml) {
  if (n_ml <= 0) return 0;
  const nnp_model* m = ws->model;
  const int nl = m->n_layers;
  cudaStream_t st = ws->stream;
  int launches = 0;
  const dim3 blk(256);
  const int nyh = (HP + SM_BN - 1) / SM_BN, nya = (m->Kfull + SM_BN - 1) / SM_BN;
  const float scale = 1.0f / (float)m->n_members;   // E = mean over the ensemble members; the 1/M rides on dz of the last layer
  for (int mem = 0; mem < m->n_members; ++mem) {
    const NetTable& nets = m->nets[mem];
    const int acc = mem > 0;
    // forward hidden layers: a_{l+1} = CELU(W_l a_l + b_l); a_0 = aev (pitch 0 = compacted pitch)
    for (int l = 0; l + 1 < nl; ++l) {
      k_dense<<<dim3(ws->max_tiles, nyh), blk, 0, st>>>(nets, ws->groups, ws->tiles, l, 0,
                                                        (l == 0) ? ws->aev : ws->hbuf[l - 1], (l == 0) ? 0 : HP,
                                                        ws->hbuf[l], HP, nullptr, 0, 0);
      ++launches;
    }
    // last layer: E_i and dz of the last hidden layer (or dE/dAEV itself for a one-layer network)
    if (nl == 1) k_last<<<ws->max_tiles, blk, 0, st>>>(nets, ws->groups, ws->tiles, ws->aev, 0, ws->e_atom, ws->daev, 0, scale, acc);
    else k_last<<<ws->max_tiles, blk, 0, st>>>(nets, ws->groups, ws->tiles, ws->hbuf[nl - 2], HP, ws->e_atom, ws->dbuf[0], HP, scale, acc);
    ++launches;
    // backward: dz_{l-1} = (W_l^T dz_l) * CELU'(a_l) for l = nl-2 .. 1, then dE/dAEV = W_0^T dz_0
    int cur = 0;
    for (int l = nl - 2; l >= 0; --l) {
      if (l > 0) {
        k_dense<<<dim3(ws->max_tiles, nyh), blk, 0, st>>>(nets, ws->groups, ws->tiles, l, 1, ws->dbuf[cur], HP,
                                                          ws->dbuf[cur ^ 1], HP, ws->hbuf[l - 1], HP, 0);
        cur ^= 1;
      } else {
        k_dense<<<dim3(ws->max_tiles, nya), blk, 0, st>>>(nets, ws->groups, ws->tiles, 0, 2, ws->dbuf[cur], HP,
                                                          ws->daev, 0, nullptr, 0, acc);
      }
      ++launches;
    }
  }
  return launches;
}

}  // namespace nnp
