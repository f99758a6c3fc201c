// api.cu -- the C-ABI boundary of include/nnp.h: model / workspace lifetime, nnp_eval (K0-K8 on one stream, no
// host synchronisation, no allocation), the host-buffer entry point, status and the debug exports.
// Interface: PAPER.md line 77 (inputs), lines 49-51 and 86 (outputs); SURVEY.md section 8.b.
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <algorithm>
#include <new>
#include <vector>
#include "nnp_internal.h"

using namespace nnp;

#define CU_OK(x) do { if ((x) != cudaSuccess) { cudaGetLastError(); return NNP_ERR_CUDA; } } while (0)

extern "C" const char* nnp_strerror(int code) {
  switch (code) {
    case NNP_OK: return "ok";
    case NNP_ERR_INVALID_ARG: return "invalid argument";
    case NNP_ERR_UNKNOWN_SPECIES: return "ML atom with an atomic number that has no species slot or no network";
    case NNP_ERR_BOX_UNSUPPORTED: return "box must be orthorhombic or GROMACS-style triclinic (lower triangular, within the shape limits, >= 3 cut-off wide cells per dimension when skewed) with positive lengths";
    case NNP_ERR_CAPACITY: return "neighbour row, cell buffer or tile capacity exceeded";
    case NNP_ERR_COINCIDENT: return "two ML atoms coincide";
    case NNP_ERR_CUDA: return "CUDA error or no CUDA device";
    case NNP_ERR_STATIC_LIMIT: return "size beyond the fixed maximum of a no-allocation entry point (NNP_STATIC_MAX_ATOMS)";
    case NNP_ERR_UNSUPPORTED: return "descriptor or network shape outside the kernels' range";
    case NNP_ERR_STALE: return "an atom left its cell by more than skin / 2 while the cell binning was being reused";
    default: return "unknown error";
  }
}

// ------------------------------------------------------------------------------------------------ model
extern "C" int nnp_model_create(const nnp_aev_params* p, const nnp_mlp_desc* nets, nnp_model** out) {
  return nnp_model_create_ensemble(p, nets, 1, out);
}

extern "C" int nnp_model_create_ensemble(const nnp_aev_params* p, const nnp_mlp_desc* nets_all, int32_t n_members,
                                         nnp_model** out) {
  if (!p || !nets_all || !out || n_members < 1 || n_members > MAX_MEMBERS) return NNP_ERR_INVALID_ARG;
  const nnp_mlp_desc* nets = nets_all;   // member 0 defines the architecture
  *out = nullptr;
  if (p->n_species < 1 || !p->species_Z || !p->ShfR || !p->ShfA || !p->ShfZ) return NNP_ERR_INVALID_ARG;
  if (!(p->Rcr > 0) || !(p->Rca > 0) || p->Rca > p->Rcr) return NNP_ERR_INVALID_ARG;
  if (p->n_species > MAX_S || p->nShfR != NSHFR || p->nShfA != NSHFA || p->nShfZ != NSHFZ) return NNP_ERR_UNSUPPORTED;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return NNP_ERR_CUDA; }
  const int S = p->n_species;
  const int L = S * NSHFR + S * (S + 1) / 2 * NSHFA * NSHFZ;
  nnp_model* m = new (std::nothrow) nnp_model();
  if (!m) return NNP_ERR_CUDA;
  memset(m, 0, sizeof(*m));
  AevConst& c = m->aev;
  c.Rcr = (float)p->Rcr; c.Rca = (float)p->Rca;
  c.Rcr2_d = p->Rcr * p->Rcr; c.Rca2_d = p->Rca * p->Rca;
  c.Rcr2 = (float)c.Rcr2_d; c.Rca2 = (float)c.Rca2_d;
  c.etaR = (float)p->EtaR; c.etaA = (float)p->EtaA;
  c.etaR_l2e = (float)(p->EtaR * 1.4426950408889634); c.etaA_l2e = (float)(p->EtaA * 1.4426950408889634);
  c.cR = (float)p->radial_prefactor; c.cTheta = (float)p->cos_scale; c.zeta = (float)p->Zeta;
  c.zeta_is_32 = (p->Zeta == 32.0);
  c.inv_Rcr = (float)(1.0 / p->Rcr); c.inv_Rca = (float)(1.0 / p->Rca);
  c.S = S; c.nRB = (S + 1) / 2; c.nblk_full = c.nRB + S * (S + 1) / 2; c.L = L;
  for (int i = 0; i < NSHFR; ++i) c.ShfR[i] = (float)p->ShfR[i];
  for (int i = 0; i < NSHFA; ++i) c.ShfA[i] = (float)p->ShfA[i];
  for (int i = 0; i < NSHFZ; ++i) { c.cosZ[i] = (float)cos(p->ShfZ[i]); c.sinZ[i] = (float)sin(p->ShfZ[i]); }
  for (int z = 0; z < 128; ++z) c.zlut[z] = -1;
  m->Kfull = c.nblk_full * BLK;

  // networks: validate, then pack all fp32 weights into one blob (layer 0 permuted to the internal column order)
  int nl_common = 0;
  size_t total = 0;
  for (int s = 0; s < S; ++s) {
    const nnp_mlp_desc& d = nets[s];
    if (d.n_layers == 0) continue;
    bool ok = d.n_layers >= 1 && d.n_layers <= MAX_LAYERS && d.dims && d.W && d.b && d.dims[d.n_layers] == 1;
    if (!ok) { delete m; return NNP_ERR_INVALID_ARG; }
    if (d.dims[0] != L) { delete m; return NNP_ERR_INVALID_ARG; }
    for (int l = 1; l < d.n_layers; ++l)
      if (d.dims[l] < 16 || d.dims[l] > HP || d.dims[l] % 16) { delete m; return NNP_ERR_UNSUPPORTED; }
    if (nl_common == 0) nl_common = d.n_layers;
    if (d.n_layers != nl_common) { delete m; return NNP_ERR_UNSUPPORTED; }
    const int z = p->species_Z[s];
    if (z < 0 || z >= 128) { delete m; return NNP_ERR_INVALID_ARG; }
    c.zlut[z] = (int8_t)s;
    for (int l = 0; l < d.n_layers; ++l) {
      const size_t in = (l == 0) ? (size_t)m->Kfull : (size_t)d.dims[l];
      total += 2 * in * d.dims[l + 1] + (size_t)d.dims[l + 1];   // W [out][in], its transpose [in][out], b
      total = (total + 7) & ~(size_t)7;
    }
  }
  if (nl_common == 0) { delete m; return NNP_ERR_INVALID_ARG; }
  m->n_layers = nl_common;
  m->n_members = n_members;
  for (int mem = 1; mem < n_members; ++mem)      // every member: same architecture as member 0
    for (int s = 0; s < S; ++s) {
      const nnp_mlp_desc &d0 = nets[s], &d = nets_all[(size_t)mem * S + s];
      bool same = d.n_layers == d0.n_layers && (d.n_layers == 0 || (d.dims && d.W && d.b));
      for (int l = 0; same && l <= d.n_layers && d.n_layers > 0; ++l) same = d.dims[l] == d0.dims[l];
      if (!same) { delete m; return NNP_ERR_UNSUPPORTED; }
    }
  total *= (size_t)n_members;
  std::vector<float> blob(total, 0.f);
  float* dbase = nullptr;
  if (cudaMalloc(&dbase, std::max<size_t>(total, 4) * sizeof(float)) != cudaSuccess) { cudaGetLastError(); delete m; return NNP_ERR_CUDA; }
  size_t off = 0;
  for (int mem = 0; mem < n_members; ++mem)
  for (int s = 0; s < S; ++s) {
    const nnp_mlp_desc& d = nets_all[(size_t)mem * S + s];
    Net& n = m->nets[mem].net[s];
    n.n_layers = d.n_layers;
    if (d.n_layers == 0) continue;
    n.alpha = (float)d.celu_alpha;
    for (int l = 0; l <= d.n_layers; ++l) n.dims[l] = d.dims[l];
    n.dims[0] = m->Kfull;  // device-side input width = internal padded column count
    for (int l = 0; l < d.n_layers; ++l) {
      const int in = d.dims[l], outw = d.dims[l + 1];
      const size_t ldw = (l == 0) ? (size_t)m->Kfull : (size_t)in;
      n.W[l] = dbase + off;
      for (int o = 0; o < outw; ++o)
        for (int i = 0; i < in; ++i) {
          size_t col = (size_t)i;
          if (l == 0 && i >= S * NSHFR) col = (size_t)c.nRB * BLK + (size_t)(i - S * NSHFR);
          blob[off + (size_t)o * ldw + col] = d.W[l][(size_t)o * in + i];
        }
      off += ldw * outw;
      n.b[l] = dbase + off;
      for (int o = 0; o < outw; ++o) blob[off + o] = d.b[l][o];
      off += outw;
      off = (off + 3) & ~(size_t)3;
      // transposed copy [in][out] (layer 0: [Kfull][out]): the single-kernel small-system path reads forward weights with
      // the output neuron on the thread index (coalesced), backward weights from W
      n.WT[l] = dbase + off;
      for (int o = 0; o < outw; ++o)
        for (int i = 0; i < in; ++i) {
          size_t col = (size_t)i;
          if (l == 0 && i >= S * NSHFR) col = (size_t)c.nRB * BLK + (size_t)(i - S * NSHFR);
          blob[off + col * outw + o] = d.W[l][(size_t)o * in + i];
        }
      off += ldw * outw;
      off = (off + 3) & ~(size_t)3;
    }
  }
  if (cudaMemcpy(dbase, blob.data(), total * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess) {
    cudaGetLastError(); cudaFree(dbase); delete m; return NNP_ERR_CUDA;
  }
  m->dev_blob = dbase; m->blob_bytes = total * sizeof(float);
  m->tc = nullptr;
  if (cudaMalloc((void**)&m->d_nets, sizeof(NetTable) * MAX_MEMBERS) != cudaSuccess ||
      cudaMemcpy(m->d_nets, m->nets, sizeof(NetTable) * MAX_MEMBERS, cudaMemcpyHostToDevice) != cudaSuccess) {
    cudaGetLastError(); if (m->d_nets) cudaFree(m->d_nets); cudaFree(dbase); delete m; return NNP_ERR_CUDA;
  }
  int rc = tc_model_create(m, nets_all);
  if (rc != NNP_OK) { cudaFree(m->d_nets); cudaFree(dbase); delete m; return rc; }
  *out = m;
  return NNP_OK;
}

extern "C" int nnp_model_destroy(nnp_model* m) {
  if (!m) return NNP_OK;
  tc_model_destroy(m);
  if (m->d_nets) cudaFree(m->d_nets);
  if (m->dev_blob) cudaFree(m->dev_blob);
  delete m;
  return NNP_OK;
}

extern "C" int nnp_model_aev_length(const nnp_model* m) { return m ? m->aev.L : NNP_ERR_INVALID_ARG; }

extern "C" int nnp_model_default_mlp_mode(const nnp_model* m) {
  if (!m) return NNP_ERR_INVALID_ARG;
  return m->tc ? NNP_MLP_F16X3 : NNP_MLP_FP32_SIMT;
}

// ------------------------------------------------------------------------------------------------ workspace
template <class T>
static bool dmalloc(T** p, size_t n) {
  *p = nullptr;
  if (cudaMalloc((void**)p, std::max<size_t>(n, 1) * sizeof(T)) != cudaSuccess) { cudaGetLastError(); return false; }
  return cudaMemset(*p, 0, std::max<size_t>(n, 1) * sizeof(T)) == cudaSuccess;
}

extern "C" int nnp_workspace_destroy(nnp_workspace* ws) {
  if (!ws) return NNP_OK;
  cudaStreamSynchronize(ws->stream);
  tc_workspace_destroy(ws);
  for (int i = 0; i < 6; ++i) if (ws->ev[i]) cudaEventDestroy(ws->ev[i]);
  void* ptrs[] = {ws->inv, ws->small_acc, ws->small_ticket, ws->wideR, ws->cntW, ws->spos_ref, ws->cellbuf, ws->cellfill, ws->present, ws->grid, ws->groups, ws->tiles, ws->flags, ws->cell_count, ws->bstart, ws->tmp4, ws->rank, ws->spos,
                  ws->scell, ws->nbrR, ws->nbrA, ws->cntR, ws->cntA, ws->aev, ws->daev, ws->hbuf[0], ws->hbuf[1],
                  ws->hbuf[2], ws->dbuf[0], ws->dbuf[1], ws->e_atom, ws->facc, ws->epart, ws->ticket, ws->wcentre, ws->wblk, ws->pos_scaled, ws->hd_pos, ws->hd_Z, ws->hd_ml,
                  ws->hd_forces};
  for (void* p : ptrs) if (p) cudaFree(p);
  if (ws->hd_energy) cudaFreeHost(ws->hd_energy);
  if (ws->hz_copy) cudaFreeHost(ws->hz_copy);
  if (ws->hml_copy) cudaFreeHost(ws->hml_copy);
  cudaGetLastError();
  delete ws;
  return NNP_OK;
}

extern "C" int nnp_workspace_create(const nnp_model* m, int64_t max_atoms, int64_t max_ml, void* stream,
                                    nnp_workspace** out) {
  if (!m || !out || max_atoms < 0 || max_ml < 0 || max_ml > max_atoms) return NNP_ERR_INVALID_ARG;
  if (max_ml >= (1ll << JBITS)) return NNP_ERR_UNSUPPORTED;
  *out = nullptr;
  nnp_workspace* ws = new (std::nothrow) nnp_workspace();
  if (!ws) return NNP_ERR_CUDA;
  memset(ws, 0, sizeof(*ws));
  ws->model = m; ws->stream = (cudaStream_t)stream; ws->max_atoms = max_atoms; ws->max_ml = max_ml;
  ws->rcap = RCAP_MAX; ws->acap = ACAP_MAX;
  ws->max_cells = (int)std::min<int64_t>(std::max<int64_t>(512, max_ml / 4), 1 << 21);
  ws->mlp_mode = m->tc ? NNP_MLP_F16X3 : NNP_MLP_FP32_SIMT;
  ws->dense_k = 0;
  ws->len_scale = 1.0; ws->e_scale = 1.0;
  {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
      cudaGetLastError(); delete ws; return NNP_ERR_CUDA;
    }
    ws->num_sms = sms;
    ws->prep_cluster = prep_cluster_size();
    ws->small_path = 1;
    ws->small_all = 1;
    ws->pack_done = 0;
    ws->inv_valid = 0; ws->forces_alias = nullptr; ws->forces_in_alias = 0;
    ws->pos_src_host = nullptr; ws->pos_src_dev = nullptr; ws->pos_src_bytes = 0;
    ws->prep_cluster_max = 8192;   // measured: 24 000 atoms run 4 us slower in one cluster than on the cooperative grid
  }
  ws->max_tiles = (int)(max_ml / TILE_M) + m->aev.S + 1;
  ws->max_rows = (int64_t)ws->max_tiles * TILE_M;
  const size_t nm = (size_t)max_ml, nr = (size_t)ws->max_rows, K = (size_t)m->Kfull;
  bool ok = dmalloc(&ws->grid, 1) && dmalloc(&ws->groups, 1) && dmalloc(&ws->tiles, (size_t)ws->max_tiles) &&
            dmalloc(&ws->flags, 1) && dmalloc(&ws->cell_count, (size_t)MAX_S * ws->max_cells + 1) &&
            dmalloc(&ws->bstart, (size_t)MAX_S * ws->max_cells + 1) && dmalloc(&ws->tmp4, nm) &&
            dmalloc(&ws->cellbuf, (size_t)ws->max_cells * cell_cap()) && dmalloc(&ws->cellfill, (size_t)ws->max_cells) && dmalloc(&ws->inv, nm) &&
            dmalloc(&ws->present, 1) &&
            dmalloc(&ws->rank, nm) && dmalloc(&ws->spos, nm) && dmalloc(&ws->scell, nm) &&
            dmalloc(&ws->nbrR, nm * ws->rcap) && dmalloc(&ws->nbrA, nm * ws->acap) && dmalloc(&ws->cntR, nm) &&
            dmalloc(&ws->cntA, nm) && dmalloc(&ws->aev, nr * K) && dmalloc(&ws->daev, nr * K) &&
            dmalloc(&ws->hbuf[0], nr * HP) && dmalloc(&ws->hbuf[1], nr * HP) && dmalloc(&ws->hbuf[2], nr * HP) &&
            dmalloc(&ws->dbuf[0], nr * HP) && dmalloc(&ws->dbuf[1], nr * HP) && dmalloc(&ws->e_atom, nr) &&
            dmalloc(&ws->facc, 3 * nm) && dmalloc(&ws->epart, nm / 256 + 2) && dmalloc(&ws->ticket, 1) && dmalloc(&ws->wcentre, 9 * nm) &&
            dmalloc(&ws->wblk, 9 * (nm / 256 + 2)) && dmalloc(&ws->pos_scaled, 3 * (size_t)max_atoms) && dmalloc(&ws->hd_pos, 3 * (size_t)max_atoms) &&
            dmalloc(&ws->hd_Z, (size_t)max_atoms) && dmalloc(&ws->hd_ml, nm) &&
            dmalloc(&ws->hd_forces, 3 * (size_t)max_atoms);
  if (ok) {   // host side of nnp_eval_host: the mapped energy word and the pinned copies of Z / ml_index of the last call
    ok = cudaHostAlloc((void**)&ws->hd_energy, sizeof(double), cudaHostAllocMapped) == cudaSuccess &&
         cudaHostGetDevicePointer((void**)&ws->hd_energy_dev, ws->hd_energy, 0) == cudaSuccess &&
         cudaHostAlloc((void**)&ws->hz_copy, sizeof(int32_t) * std::max<size_t>((size_t)max_atoms, 1), cudaHostAllocDefault) == cudaSuccess &&
         cudaHostAlloc((void**)&ws->hml_copy, sizeof(int32_t) * std::max<size_t>(nm, 1), cudaHostAllocDefault) == cudaSuccess;
    if (ok) *ws->hd_energy = 0.0;
  }
  if (ok) ok = dmalloc(&ws->small_acc, 3 * 256) && dmalloc(&ws->small_ticket, 1) && small_all_prepare(ws) == NNP_OK;
  if (ok) ok = (tc_workspace_create(ws) == NNP_OK);
  if (!ok || cudaDeviceSynchronize() != cudaSuccess) { cudaGetLastError(); nnp_workspace_destroy(ws); return NNP_ERR_CUDA; }
  *out = ws;
  return NNP_OK;
}

extern "C" int nnp_workspace_set_mlp_mode(nnp_workspace* ws, int32_t mode) {
  if (!ws) return NNP_ERR_INVALID_ARG;
  if (mode == NNP_MLP_FP32_SIMT) { ws->mlp_mode = mode; return NNP_OK; }
  if (mode == NNP_MLP_F16X3 || mode == NNP_MLP_F16X1) {
    if (!ws->model->tc) return NNP_ERR_UNSUPPORTED;
    ws->mlp_mode = mode;
    return NNP_OK;
  }
  return NNP_ERR_INVALID_ARG;
}

extern "C" int nnp_workspace_set_profiling(nnp_workspace* ws, int32_t on) {
  if (!ws) return NNP_ERR_INVALID_ARG;
  if (on && !ws->ev[0])
    for (int i = 0; i < 6; ++i) CU_OK(cudaEventCreate(&ws->ev[i]));
  ws->profiling = on ? 1 : 0;
  return NNP_OK;
}

extern "C" int nnp_debug_stage_times(nnp_workspace* ws, float* ms) {
  if (!ws || !ms || !ws->profiling) return NNP_ERR_INVALID_ARG;
  CU_OK(cudaEventSynchronize(ws->ev[5]));
  for (int i = 0; i < 5; ++i) CU_OK(cudaEventElapsedTime(&ms[i], ws->ev[i], ws->ev[i + 1]));
  return NNP_OK;
}

// positions in the caller's length unit -> Angstrom: converted in fp64 and rounded to fp32 ONCE; every later step
// (cell binning and the pinned fp64 neighbour predicate included) works on the converted fp32 coordinates.
__global__ void k_scale_pos(const float* __restrict__ in, float* __restrict__ out, long long n3, double s) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n3) out[i] = (float)((double)in[i] * s);
}

extern "C" int nnp_workspace_set_units(nnp_workspace* ws, double angstrom_per_length_unit, double energy_units_per_ev) {
  if (!ws || !(angstrom_per_length_unit > 0.0) || !(energy_units_per_ev > 0.0)) return NNP_ERR_INVALID_ARG;
  ws->len_scale = angstrom_per_length_unit;
  ws->e_scale = energy_units_per_ev;
  return NNP_OK;
}

extern "C" int nnp_workspace_set_virial_output(nnp_workspace* ws, double* d_virial9) {
  if (!ws) return NNP_ERR_INVALID_ARG;
  ws->d_virial = d_virial9;
  return NNP_OK;
}

extern "C" int nnp_workspace_set_pair_list(nnp_workspace* ws, const int32_t* d_pairs, int64_t n_pairs) {
  if (!ws || n_pairs < 0 || (n_pairs > 0 && !d_pairs)) return NNP_ERR_INVALID_ARG;
  ws->ext_pairs = d_pairs;
  ws->n_ext_pairs = d_pairs ? n_pairs : 0;
  return NNP_OK;
}

extern "C" int nnp_workspace_set_bin_reuse(nnp_workspace* ws, int32_t every_n, double skin) {
  if (!ws || (every_n > 1 && !(skin > 0.0))) return NNP_ERR_INVALID_ARG;
  if (every_n > 1 && !ws->wideR) {   // first use: the wide rows of the row reuse (allocated here, never inside nnp_eval)
    ws->wcap = 256;
    const size_t nm = (size_t)std::max<int64_t>(ws->max_ml, 1);
    if (cudaMalloc((void**)&ws->wideR, nm * ws->wcap * sizeof(uint32_t)) != cudaSuccess ||
        cudaMalloc((void**)&ws->cntW, nm * sizeof(int)) != cudaSuccess ||
        cudaMalloc((void**)&ws->spos_ref, nm * sizeof(float4)) != cudaSuccess) {
      cudaGetLastError();
      if (ws->wideR) cudaFree(ws->wideR);
      if (ws->cntW) cudaFree(ws->cntW);
      ws->wideR = nullptr; ws->cntW = nullptr; ws->spos_ref = nullptr;
      return NNP_ERR_CUDA;
    }
  }
  ws->reuse_every = every_n > 1 ? every_n : 0;
  ws->reuse_skin = every_n > 1 ? skin : 0.0;
  ws->reuse_left = 0;   // the next evaluation bins afresh (with the new cell width)
  return NNP_OK;
}

extern "C" int nnp_workspace_set_small_path(nnp_workspace* ws, int32_t on) {
  if (!ws) return NNP_ERR_INVALID_ARG;
  ws->small_path = on ? 1 : 0;
  ws->small_all = (on == 1) ? 0 : 1;   // 1: the front end only (five launches); any other non-zero value (default 2): one kernel
  return NNP_OK;
}

extern "C" int nnp_workspace_set_dense_k(nnp_workspace* ws, int32_t dense) {
  if (!ws) return NNP_ERR_INVALID_ARG;
  ws->dense_k = dense ? 1 : 0;
  return NNP_OK;
}

// ------------------------------------------------------------------------------------------------ evaluation
static int check_box(const float* box, int pbc) {
  if (!pbc) return NNP_OK;
  if (!box) return NNP_ERR_INVALID_ARG;
  for (int r = 0; r < 3; ++r)
    for (int c = 0; c < 3; ++c) {
      const float v = box[3 * r + c];
      if (r == c) { if (!(v > 0.f) || !isfinite(v)) return NNP_ERR_BOX_UNSUPPORTED; }
      else if (c > r ? v != 0.f : !isfinite(v)) return NNP_ERR_BOX_UNSUPPORTED;   // GROMACS rows: lower triangular
    }
  // triclinic shape limits of the minimum-image reduction (reading #35)
  if (fabsf(box[3]) > 0.5f * box[0] || fabsf(box[6]) > 0.5f * box[0] || fabsf(box[7]) > 0.5f * box[4]) return NNP_ERR_BOX_UNSUPPORTED;
  return NNP_OK;
}

void nnp::flush_pos_upload(nnp_workspace* ws) {
  if (!ws->pos_src_host) return;
  cudaMemcpyAsync(ws->hd_pos, ws->pos_src_host, ws->pos_src_bytes, cudaMemcpyHostToDevice, ws->stream);
  ws->pos_src_host = nullptr; ws->pos_src_dev = nullptr;
}

extern "C" int nnp_eval(nnp_workspace* ws, int64_t n_atoms, const float* d_pos, const int32_t* d_Z, const float box[9],
                        int32_t pbc, const int32_t* d_ml, int64_t n_ml, double* d_energy, float* d_forces) {
  if (!ws || n_atoms < 0 || !d_energy || (n_atoms > 0 && (!d_pos || !d_Z || !d_forces))) return NNP_ERR_INVALID_ARG;
  if (!d_ml) n_ml = n_atoms;
  if (n_ml < 0 || n_ml > n_atoms || n_atoms > ws->max_atoms || n_ml > ws->max_ml) return NNP_ERR_INVALID_ARG;
  int rc = check_box(box, pbc);
  if (rc) return rc;
  const float unit[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
  if (pbc) {   // a triclinic box must hold >= 3 cut-off wide cells between every pair of faces
    float bs[9];
    for (int i = 0; i < 9; ++i) bs[i] = (float)((double)box[i] * ws->len_scale);
    if (!neighbor_box_ok(ws, bs)) return NNP_ERR_BOX_UNSUPPORTED;
  }
  ws->n_atoms = n_atoms; ws->n_ml = n_ml; ws->d_ml_index = d_ml;
  prof_mark(ws, 0);
  int nl = 0;
  float box_a[9];
  ws->tile_done = nullptr;
  // small periodic ML region, everything in ONE kernel: no memset, no other launch
  if (ws->len_scale == 1.0 && small_all_applicable(ws, box, pbc, n_ml)) {
    flush_pos_upload(ws);
    ws->inv_valid = 0;   // (another sorted order from here on)
    ws->launches = launch_small_all(ws, d_pos, d_Z, box, d_ml, n_atoms, n_ml, d_energy, d_forces);
    if (cudaGetLastError() != cudaSuccess) return NNP_ERR_CUDA;
    return NNP_OK;
  }
  if (ws->len_scale != 1.0 || d_ml || n_ml <= 0 || small_front_applicable(ws, box, pbc, n_ml)) flush_pos_upload(ws);
  // rows of non-ML atoms are +0.0f; with no index subset every row is written by k_force_out
  if (n_atoms > 0 && (d_ml || n_ml <= 0)) cudaMemsetAsync(d_forces, 0, sizeof(float) * 3 * (size_t)n_atoms, ws->stream);
  if (ws->len_scale != 1.0) {   // unit conversion (GROMACS: nm -> Angstrom), see nnp_workspace_set_units
    if (n_atoms > 0) {
      k_scale_pos<<<(unsigned)((3 * n_atoms + 255) / 256), 256, 0, ws->stream>>>(d_pos, ws->pos_scaled, 3 * n_atoms, ws->len_scale);
      ++nl;
    }
    d_pos = ws->pos_scaled;
    if (pbc) { for (int i = 0; i < 9; ++i) box_a[i] = (float)((double)box[i] * ws->len_scale); box = box_a; }
  }
  if (small_front_applicable(ws, box, pbc, n_ml)) {
    // small periodic ML region: K0-K3 in one kernel (stage profiling books it under "neighbour", AEV forward = 0)
    ws->inv_valid = 0;
    nl += launch_small_front(ws, d_pos, d_Z, box, d_ml, n_atoms, n_ml);
    prof_mark(ws, 1);
    prof_mark(ws, 2);
  } else {
    nl += launch_neighbor_stage(ws, d_pos, d_Z, pbc ? box : unit, pbc ? 1 : 0, d_ml, n_atoms, n_ml);
    prof_mark(ws, 1);
    nl += launch_aev_forward(ws, n_ml);
    prof_mark(ws, 2);
  }
  nl += (ws->mlp_mode == NNP_MLP_FP32_SIMT) ? launch_mlp_simt(ws, n_ml) : launch_mlp_tc(ws, n_ml);
  prof_mark(ws, 3);
  if (n_ml <= 0) prof_mark(ws, 4);
  nl += launch_force_stage(ws, n_atoms, n_ml, d_ml, d_energy, d_forces);
  prof_mark(ws, 5);
  ws->launches = nl;
  if (cudaGetLastError() != cudaSuccess) return NNP_ERR_CUDA;
  return NNP_OK;
}

extern "C" int nnp_eval_host(nnp_workspace* ws, int64_t n_atoms, const float* h_pos, const int32_t* h_Z,
                             const float box[9], int32_t pbc, const int32_t* h_ml, int64_t n_ml, double* h_energy,
                             float* h_forces) {
  if (!ws || n_atoms < 0 || n_atoms > ws->max_atoms || !h_energy || (n_atoms > 0 && (!h_pos || !h_Z || !h_forces)))
    return NNP_ERR_INVALID_ARG;
  if (h_ml && (n_ml < 0 || n_ml > ws->max_ml)) return NNP_ERR_INVALID_ARG;
  cudaStream_t st = ws->stream;
  // Pinned (device-mapped) host buffers can be used by the kernels in place.  (Asked on every call -- ~1 us each: an
  // address may have been freed and handed out again as pageable memory since the last one.)
  auto device_alias = [](const void* h) -> void* {
    cudaPointerAttributes at;
    if (h && cudaPointerGetAttributes(&at, h) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer) return at.devicePointer;
    cudaGetLastError();
    return nullptr;
  };
  float* const f_alias = n_atoms > 0 ? static_cast<float*>(device_alias(h_forces)) : nullptr;
  // A small ML region inside a large system (ONE kernel, k_small_all; 14-107 ML atoms among
  // thousands): the kernel reads the few ML positions it needs from the caller's pinned buffer and writes the force rows
  // (zeros but for the ML atoms) into the caller's pinned buffer itself, instead of two copies of the whole arrays (cfg 4,
  // 64 of 9064 atoms: 69.1 -> 64.7 us per call).  Not below 2048 atoms (a 96-atom box: 55.7 -> 57.8 us, the PCIe round
  // trip inside the kernel costs more than two 1 KB copies), and not for the cell-list path's positions (read in place
  // by the binning kernel: e2e 271 -> 286 us at 24 000 atoms -- three 4-byte loads per atom do not stream over PCIe); its
  // forces go in place where the output kernel writes them coalesced (below).
  const bool small_direct = ws->len_scale == 1.0 && f_alias && n_atoms >= 2048 &&
                            small_all_applicable(ws, box, pbc, h_ml ? n_ml : n_atoms);
  const float* const p_alias = small_direct ? static_cast<const float*>(device_alias(h_pos)) : nullptr;
  const bool in_place = small_direct && p_alias;
  ws->pos_src_host = nullptr; ws->pos_src_dev = nullptr;
  if (!in_place) {
    // cell-list path with all atoms ML atoms and pinned positions: the upload is left to the binning kernel (pending here,
    // flush_pos_upload turns it into this copy on every other path)
    const float* up = (!h_ml && n_atoms >= 2048 && f_alias) ? static_cast<const float*>(device_alias(h_pos)) : nullptr;
    if (up) { ws->pos_src_host = h_pos; ws->pos_src_dev = up; ws->pos_src_bytes = sizeof(float) * 3 * (size_t)n_atoms; }
    else CU_OK(cudaMemcpyAsync(ws->hd_pos, h_pos, sizeof(float) * 3 * (size_t)n_atoms, cudaMemcpyHostToDevice, st));
  }
  // atomic numbers and the ML index rarely change between MD steps: they are compared with the host copy of the last
  // call and uploaded only when different (the comparison also makes binning reuse safe for this entry point: the
  // device buffers are always the same, so pointer identity alone would say "same atoms" -- a change bins afresh)
  const size_t zb = sizeof(int32_t) * (size_t)n_atoms, mb = h_ml ? sizeof(int32_t) * (size_t)n_ml : 0;
  const bool z_same = ws->hz_valid && ws->hz_n == n_atoms && (zb == 0 || memcmp(ws->hz_copy, h_Z, zb) == 0);
  const bool ml_same = ws->hml_valid && ws->hml_n == (h_ml ? n_ml : -1) && (mb == 0 || memcmp(ws->hml_copy, h_ml, mb) == 0);
  if (!z_same) {
    if (zb) { memcpy(ws->hz_copy, h_Z, zb); CU_OK(cudaMemcpyAsync(ws->hd_Z, ws->hz_copy, zb, cudaMemcpyHostToDevice, st)); }
    ws->hz_n = n_atoms; ws->hz_valid = 1;
  }
  if (!ml_same) {
    if (mb) { memcpy(ws->hml_copy, h_ml, mb); CU_OK(cudaMemcpyAsync(ws->hd_ml, ws->hml_copy, mb, cudaMemcpyHostToDevice, st)); }
    ws->hml_n = h_ml ? n_ml : -1; ws->hml_valid = 1;
  }
  if (!z_same || !ml_same) ws->reuse_left = 0;
  // A pinned force buffer of the caller is written by the output kernel itself where that kernel writes in the caller's
  // order (coalesced: force.cu k_force_out): no device-to-host copy then.
  ws->forces_alias = !h_ml ? f_alias : nullptr;
  ws->forces_in_alias = 0;
  int rc = nnp_eval(ws, n_atoms, in_place ? p_alias : ws->hd_pos, ws->hd_Z, box, pbc, h_ml ? ws->hd_ml : nullptr, n_ml,
                    ws->hd_energy_dev, in_place ? f_alias : ws->hd_forces);
  ws->forces_alias = nullptr;
  ws->pos_src_host = nullptr; ws->pos_src_dev = nullptr;   // (an evaluation that failed before its first launch)
  if (rc) return rc;
  if (!ws->forces_in_alias && !in_place)
    CU_OK(cudaMemcpyAsync(h_forces, ws->hd_forces, sizeof(float) * 3 * (size_t)n_atoms, cudaMemcpyDeviceToHost, st));
  CU_OK(cudaStreamSynchronize(st));
  *h_energy = *ws->hd_energy;   // mapped pinned word, written by the output kernel (or the memset of an empty subset)
  return NNP_OK;
}

extern "C" int nnp_status(nnp_workspace* ws) {
  if (!ws) return NNP_ERR_INVALID_ARG;
  if (cudaStreamSynchronize(ws->stream) != cudaSuccess) { cudaGetLastError(); return NNP_ERR_CUDA; }
  int f = 0;
  CU_OK(cudaMemcpy(&f, ws->flags, sizeof(int), cudaMemcpyDeviceToHost));
  CU_OK(cudaMemset(ws->flags, 0, sizeof(int)));
  if (f & FLAG_STALE) ws->reuse_left = 0;   // whatever else went wrong: the next evaluation bins afresh
  if (f & FLAG_CAP) ws->slow_prep = 1;      // (possibly) a cell beyond the fast binning's buffer: general binning from now on
  if (f & FLAG_TIMEOUT) return NNP_ERR_CUDA;   // a kernel gave up waiting for its producer (force.cu): outputs invalid
  if (f & FLAG_ARG) return NNP_ERR_INVALID_ARG;
  if (f & FLAG_SPECIES) return NNP_ERR_UNKNOWN_SPECIES;
  if (f & FLAG_CAP) return NNP_ERR_CAPACITY;
  if (f & FLAG_COINCIDENT) return NNP_ERR_COINCIDENT;
  if (f & FLAG_STALE) return NNP_ERR_STALE;
  return NNP_OK;
}

// ------------------------------------------------------------------------------------------------ debug exports
namespace {
struct Snapshot {
  std::vector<float4> spos;
  std::vector<int32_t> ml;
  GroupInfo grp;
};
int take_snapshot(nnp_workspace* ws, Snapshot& s) {
  if (cudaStreamSynchronize(ws->stream) != cudaSuccess) { cudaGetLastError(); return NNP_ERR_CUDA; }
  const size_t n = (size_t)ws->n_ml;
  s.spos.resize(n);
  if (n) CU_OK(cudaMemcpy(s.spos.data(), ws->spos, n * sizeof(float4), cudaMemcpyDeviceToHost));
  s.ml.clear();
  if (ws->d_ml_index && n) {
    s.ml.resize(n);
    CU_OK(cudaMemcpy(s.ml.data(), ws->d_ml_index, n * sizeof(int32_t), cudaMemcpyDeviceToHost));
  }
  CU_OK(cudaMemcpy(&s.grp, ws->groups, sizeof(GroupInfo), cudaMemcpyDeviceToHost));
  return NNP_OK;
}
inline int ml_local(const float4& v) { int w; memcpy(&w, &v.w, 4); return w & 0x0fffffff; }
inline int slot_of(const float4& v) { int w; memcpy(&w, &v.w, 4); return (w >> 28) & 7; }
}  // namespace

extern "C" int nnp_debug_neighbors(nnp_workspace* ws, int which, int64_t* n_pairs, int32_t* h_row_start,
                                   int32_t* h_col, int64_t col_cap) {
  if (!ws || !n_pairs || (which != 0 && which != 1)) return NNP_ERR_INVALID_ARG;
  Snapshot s;
  int rc = take_snapshot(ws, s);
  if (rc) return rc;
  const size_t n = (size_t)ws->n_ml;
  std::vector<int> cntR(n), cntA(n);
  std::vector<uint32_t> nbrR(n * ws->rcap);
  std::vector<uint8_t> nbrA(n * ws->acap);
  if (n) {
    CU_OK(cudaMemcpy(cntR.data(), ws->cntR, n * sizeof(int), cudaMemcpyDeviceToHost));
    CU_OK(cudaMemcpy(cntA.data(), ws->cntA, n * sizeof(int), cudaMemcpyDeviceToHost));
    CU_OK(cudaMemcpy(nbrR.data(), ws->nbrR, nbrR.size() * sizeof(uint32_t), cudaMemcpyDeviceToHost));
    CU_OK(cudaMemcpy(nbrA.data(), ws->nbrA, nbrA.size(), cudaMemcpyDeviceToHost));
  }
  std::vector<int> sorted_of(n);  // ml-local index -> sorted position
  for (size_t ip = 0; ip < n; ++ip) sorted_of[ml_local(s.spos[ip])] = (int)ip;
  int64_t tot = 0;
  for (size_t a = 0; a < n; ++a) tot += which ? cntA[sorted_of[a]] : cntR[sorted_of[a]];
  *n_pairs = tot;
  if (!h_col || !h_row_start || col_cap < tot) return NNP_OK;
  int64_t pos = 0;
  for (size_t a = 0; a < n; ++a) {
    const int ip = sorted_of[a];
    h_row_start[a] = (int32_t)pos;
    const int cnt = which ? cntA[ip] : cntR[ip];
    for (int q = 0; q < cnt; ++q) {
      const int pr = which ? nbrA[(size_t)ip * ws->acap + q] : q;
      const int jp = (int)(nbrR[(size_t)ip * ws->rcap + pr] & JMASK);
      const int aj = ml_local(s.spos[jp]);
      h_col[pos + q] = s.ml.empty() ? aj : s.ml[aj];
    }
    std::sort(h_col + pos, h_col + pos + cnt);
    pos += cnt;
  }
  h_row_start[n] = (int32_t)pos;
  return NNP_OK;
}

extern "C" int nnp_debug_aev(nnp_workspace* ws, float* h_aev) {
  if (!ws || !h_aev) return NNP_ERR_INVALID_ARG;
  Snapshot s;
  int rc = take_snapshot(ws, s);
  if (rc) return rc;
  const AevConst& c = ws->model->aev;
  const size_t n = (size_t)ws->n_ml, Kc = (size_t)s.grp.Kc;
  std::vector<float> buf((size_t)s.grp.n_rows * Kc);
  if (!buf.empty()) CU_OK(cudaMemcpy(buf.data(), ws->aev, buf.size() * sizeof(float), cudaMemcpyDeviceToHost));
  memset(h_aev, 0, n * (size_t)c.L * sizeof(float));
  for (size_t ip = 0; ip < n; ++ip) {
    const int a = ml_local(s.spos[ip]), sl = slot_of(s.spos[ip]);
    const float* row = buf.data() + (ip + s.grp.pad_shift[sl]) * Kc;
    float* dst = h_aev + (size_t)a * c.L;
    for (int b = 0; b < s.grp.nblk; ++b) {
      const int ib = s.grp.blkmap[b];
      for (int q = 0; q < BLK; ++q) {
        const int icol = ib * BLK + q;  // internal column -> public column
        int pub;
        if (ib < c.nRB) { if (icol >= c.S * NSHFR) continue; pub = icol; }
        else pub = c.S * NSHFR + (icol - c.nRB * BLK);
        dst[pub] = row[(size_t)b * BLK + q];
      }
    }
  }
  return NNP_OK;
}

static int export_rows(nnp_workspace* ws, const float* d_buf, float* h_out, bool piece_major) {
  Snapshot s;
  int rc = take_snapshot(ws, s);
  if (rc) return rc;
  const AevConst& c = ws->model->aev;
  const size_t n = (size_t)ws->n_ml, Kc = (size_t)s.grp.Kc;
  std::vector<float> buf((size_t)s.grp.n_rows * Kc);
  if (!buf.empty()) CU_OK(cudaMemcpy(buf.data(), d_buf, buf.size() * sizeof(float), cudaMemcpyDeviceToHost));
  memset(h_out, 0, n * (size_t)c.L * sizeof(float));
  for (size_t ip = 0; ip < n; ++ip) {
    const int a = ml_local(s.spos[ip]), sl = slot_of(s.spos[ip]);
    const float* row = buf.data() + (ip + s.grp.pad_shift[sl]) * Kc;
    float* dst = h_out + (size_t)a * c.L;
    for (int b = 0; b < s.grp.nblk; ++b) {
      const int ib = s.grp.blkmap[b];
      for (int q = 0; q < BLK; ++q) {
        const int icol = ib * BLK + q;  // internal column -> public column
        int pub;
        if (ib < c.nRB) { if (icol >= c.S * NSHFR) continue; pub = icol; }
        else pub = c.S * NSHFR + (icol - c.nRB * BLK);
        dst[pub] = piece_major ? buf[daev_off(ip + s.grp.pad_shift[sl], b * BLK + q, (int)Kc)] : row[(size_t)b * BLK + q];
      }
    }
  }
  return NNP_OK;
}

extern "C" int nnp_debug_daev(nnp_workspace* ws, float* h_daev) {
  if (!ws || !h_daev) return NNP_ERR_INVALID_ARG;
  return export_rows(ws, ws->daev, h_daev, true);
}

extern "C" int nnp_debug_atomic_energies(nnp_workspace* ws, float* h_e) {
  if (!ws || !h_e) return NNP_ERR_INVALID_ARG;
  Snapshot s;
  int rc = take_snapshot(ws, s);
  if (rc) return rc;
  std::vector<float> buf((size_t)s.grp.n_rows);
  if (!buf.empty()) CU_OK(cudaMemcpy(buf.data(), ws->e_atom, buf.size() * sizeof(float), cudaMemcpyDeviceToHost));
  for (size_t ip = 0; ip < (size_t)ws->n_ml; ++ip)
    h_e[ml_local(s.spos[ip])] = buf[ip + s.grp.pad_shift[slot_of(s.spos[ip])]];
  return NNP_OK;
}

extern "C" int nnp_debug_mlp_timeline(nnp_workspace* ws, int64_t* h_ticks) {
  if (!ws || !h_ticks) return NNP_ERR_INVALID_ARG;
  if (cudaStreamSynchronize(ws->stream) != cudaSuccess) { cudaGetLastError(); return NNP_ERR_CUDA; }
  static_assert(sizeof(long long) == sizeof(int64_t), "tick type");
  return tc_read_timeline(reinterpret_cast<long long*>(h_ticks));
}

extern "C" int nnp_debug_counters(nnp_workspace* ws, int64_t* launches) {
  if (!ws || !launches) return NNP_ERR_INVALID_ARG;
  launches[0] = ws->launches;
  return NNP_OK;
}
