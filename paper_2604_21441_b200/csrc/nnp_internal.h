// nnp_internal.h -- shared declarations of the CUDA path (not part of the C-ABI; never included by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/nnp.h"

namespace nnp {

constexpr int MAX_S = 8;          // species slots
constexpr int MAX_LAYERS = 4;
constexpr int MAX_MEMBERS = 8;    // networks per element in an ensemble (ANI-2x: 8)
constexpr int TILE_M = 128;       // MLP row tile (tcgen05 M)
constexpr int HP = 256;           // pitch of the hidden-activation / delta scratch rows (max hidden width)
constexpr int NSHFR = 16;         // radial shifts (fixed by the kernels)
constexpr int NSHFA = 4;          // angular radial shifts
constexpr int NSHFZ = 8;          // angular theta shifts
constexpr int BLK = 32;           // AEV column block: one angular pair (4x8) or two radial species (2x16)
constexpr int MAX_BLK = 40;       // ceil(8/2) + 8*9/2
constexpr int RCAP_MAX = 128;     // radial neighbour row capacity (positions fit a uint8 with room to spare)
constexpr int ACAP_MAX = 48;      // angular neighbour row capacity
constexpr int JBITS = 26;         // neighbour entry: sorted index in the low 26 bits, 3x2-bit cell offset above
constexpr uint32_t JMASK = (1u << JBITS) - 1u;
constexpr int FIX_SHIFT = 40;     // fixed-point scale 2^40 for the int64 force accumulators (K8)

// device-side sticky status bits
enum : int { FLAG_ARG = 1, FLAG_SPECIES = 2, FLAG_CAP = 4, FLAG_COINCIDENT = 8, FLAG_STALE = 16, FLAG_TIMEOUT = 32 };

// Descriptor constants, passed to kernels by value.
struct AevConst {
  float Rcr, Rca, Rcr2, Rca2;
  double Rcr2_d, Rca2_d;      // exact fp64 thresholds of the pinned neighbour predicate (reading #6)
  float etaR, etaA;
  float etaR_l2e, etaA_l2e;   // eta * log2(e): exp(-eta x^2) = exp2(-eta_l2e x^2)
  float cR, cTheta, zeta;
  int zeta_is_32;
  float inv_Rcr, inv_Rca;     // 1 / Rc
  int S;                      // species slots
  int nRB;                    // radial column blocks = ceil(S/2)
  int nblk_full;              // nRB + S(S+1)/2
  int L;                      // AEV length in the public (BASELINE.json) order
  float ShfR[NSHFR];
  float ShfA[NSHFA];
  float cosZ[NSHFZ], sinZ[NSHFZ];  // cos / sin of ShfZ
  int8_t zlut[128];           // atomic number -> slot (-1: none / no network)
};

// Cell grid of one evaluation (device resident; written by k_grid_setup).
struct GridInfo {
  int nc[3];
  int ncell;
  int pbc;
  float edge[3];       // cell edge per dimension
  double edge_d[3];
  double inv_edge_d[3];
  double origin_d[3];  // 0 for pbc; bounding-box minimum for open boundaries
  double L_d[3];       // box lengths (fp32 inputs promoted), for the exact predicate
  float L[3];
  // Triclinic boxes (GROMACS rows a = (ax,0,0), b = (bx,by,0), c = (cx,cy,cz); reading #35).  The cell of
  // index (i,j,k) has its origin at i ea + j eb + k ec with the edge VECTORS ea = a / nc[0], eb = b / nc[1],
  // ec = c / nc[2] (ev rows; orthorhombic: the diagonal holds edge[]), and the displacement of a stored neighbour is
  // (local_j - local_i) + ox ea + oy eb + oz ec.
  int tric;
  float ev[9];
  double ev_d[9];
  double H_d[6];       // {ax, by, cz, bx, cx, cy}
};

// Cartesian shift of a cell offset (ox, oy, oz)
__host__ __device__ inline void cell_shift(const float* __restrict__ ev, int ox, int oy, int oz, float& sx, float& sy, float& sz) {
  sx = (float)ox * ev[0] + (float)oy * ev[3] + (float)oz * ev[6];
  sy = (float)oy * ev[4] + (float)oz * ev[7];
  sz = (float)oz * ev[8];
}

// Species groups, MLP tiles and the compacted AEV column map of one evaluation (device resident; k_scan).
// Internal AEV column order: radial species s at s*16 (padded to nRB*32 columns), angular pair p at
// (nRB + p)*32.  Only column blocks that can be non-zero for the species present are materialised
// ("structural-zero compaction"): compact column = cpos[block]*32 + (col % 32).
struct GroupInfo {
  int count[MAX_S];      // atoms per slot
  int start[MAX_S + 1];  // first sorted index of the slot (sorted order is slot-major)
  int pad_shift[MAX_S];  // row = sorted index + pad_shift[slot]; group rows padded to TILE_M
  int n_tiles;
  int n_rows;            // padded row count
  int nblk;              // materialised column blocks
  int Kc;                // 32 * nblk = row pitch of aev / daev
  int blkmap[MAX_BLK];   // compact block -> internal block
  int cpos[MAX_BLK];     // internal block -> compact block, or -1
  int npres;             // species present in this evaluation, ascending
  int pres[MAX_S];
  unsigned long long colkey;  // bit 63 | bit mask of the materialised internal blocks (identifies the column set)
};

struct TileInfo { int slot, row0, nvalid, pad; };

// dE/dAEV is stored tile-wise "piece-major": within the 128-row tile of a row, the float4 piece q = col / 4 of all
// 128 rows is contiguous (2 KB).  The MLP epilogue (thread = row) then writes 512 contiguous bytes per warp store,
// and the AEV backward kernel, which only reads float4 pieces, finds the pieces of neighbouring rows in one line.
__host__ __device__ inline size_t daev_off(size_t row, int col, int Kc) {
  return (row >> 7) * ((size_t)Kc * TILE_M) + (size_t)(col >> 2) * (4 * TILE_M) + (row & (TILE_M - 1)) * 4 + (col & 3);
}

struct Net {             // device pointers, one per slot
  int n_layers;
  int dims[MAX_LAYERS + 1];
  const float* W[MAX_LAYERS];   // [out][in] fp32; layer 0 in the internal padded column order [out][Kfull]
  const float* WT[MAX_LAYERS];  // [in][out] fp32; layer 0 [Kfull][out]
  const float* b[MAX_LAYERS];
  float alpha;
};

struct NetTable { Net net[MAX_S]; };

}  // namespace nnp

struct nnp_model {
  nnp::AevConst aev;
  nnp::NetTable nets[nnp::MAX_MEMBERS];  // device pointers, one table per ensemble member
  int n_members;             // E = mean over the members' energies (1 = a single network per element)
  int n_layers;              // common to all networks
  int Kfull;                 // 32 * nblk_full
  void* dev_blob;            // single allocation holding all fp32 weights
  size_t blob_bytes;
  void* tc;                  // tensor-core weight images (mlp_tc.cu), or nullptr
  nnp::NetTable* d_nets;     // DEVICE copy of nets[] (the single-kernel small-system path reads the tables from global memory)
};

struct nnp_workspace {
  const nnp_model* model;
  cudaStream_t stream;
  int64_t max_atoms, max_ml;
  int rcap, acap;            // neighbour row capacities
  int max_cells;
  int num_sms;               // multiprocessor count of the device (cooperative grid size)
  int prep_cluster;          // CTAs of the single-cluster prep kernel (0: cooperative grid only)
  int prep_cluster_max;      // largest n_ml the single-cluster variant takes
  int mlp_mode;
  int dense_k;               // 1: materialise every column block (no structural-zero compaction)
  int small_path;            // 1 (default): small periodic ML regions take the single-kernel front end (small.cu)
  int small_all;             // 1 (default): ... and, where applicable, the whole evaluation as ONE kernel (k_small_all)
  unsigned long long* small_acc;   // [256 * 3] force accumulators of k_small_all (zero between evaluations)
  unsigned int* small_ticket;
  size_t small_all_smem;
  int* inv;                  // [max_ml] ML-local index -> sorted index (written by k_cell_sort)
  int inv_valid;             // inv matches the current sorted order
  float* forces_alias;       // nnp_eval_host: device alias of the caller's pinned force buffer, or NULL
  // nnp_eval_host with pinned positions: the upload into hd_pos is still pending when nnp_eval starts -- the binning
  // kernel of the cell-list path does it itself (coalesced, block by block), every other path asks for the copy first
  const float* pos_src_host; const float* pos_src_dev; size_t pos_src_bytes;
  int forces_in_alias;       // the last evaluation wrote its forces straight through forces_alias
  int pack_done;             // launch_tc_pack has run for this evaluation already (the cell-list path runs it early)
  int64_t max_rows;          // padded AEV rows
  int max_tiles;
  // last evaluation
  int64_t n_atoms, n_ml;
  const int32_t* d_ml_index;
  int64_t launches;
  // device buffers
  nnp::GridInfo* grid;
  nnp::GroupInfo* groups;
  nnp::TileInfo* tiles;
  int* flags;
  int* cell_count;           // [MAX_S*max_cells + 1]
  int* bstart;               // [MAX_S*max_cells + 1]
  float4* tmp4;              // [max_ml] local coords + key
  float4* cellbuf;           // [max_cells][CELL_CAP] per-cell append buffers of the fast binning (neighbor.cu)
  int* cellfill;             // [max_cells] fill counters of the above (zero between evaluations)
  int* present;              // [1] bit mask of the species slots seen by k_bin_cells (zero between evaluations)
  uint32_t* wideR;           // [max_ml][wcap] wide rows (everything within Rcr + skin at the last full build), row reuse only
  int* cntW;                 // [max_ml]
  float4* spos_ref;          // [max_ml] cell-local coordinates at the last full build
  int wcap;
  int slow_prep;             // 1: a cell overflowed its append buffer once; this workspace keeps to the general binning
  int* rank;                 // [max_ml]
  float4* spos;              // [max_ml] sorted: cell-local xyz, w = ml-local index | slot << 28
  int* scell;                // [max_ml]
  uint32_t* nbrR;            // [max_ml][rcap]
  uint8_t* nbrA;             // [max_ml][acap] positions into the radial row
  int* cntR; int* cntA;      // [max_ml]
  float* aev;                // [max_rows][Kc] fp32
  float* daev;               // [max_rows][Kc] fp32
  float* hbuf[3];            // hidden activations [max_rows][HP]
  float* dbuf[2];            // deltas [max_rows][HP]
  float* e_atom;             // [max_rows]
  unsigned long long* facc;  // [max_ml][3] int64 fixed point, indexed by sorted position
  double* epart;             // [ceil(max_ml/256)] block partial sums of E_i (K8)
  unsigned int* ticket;      // [1] last-block ticket of K8
  long long* wcentre;        // [max_ml][9] per-centre strain derivative, 2^-32 fixed point (virial output on)
  long long* wblk;           // [ceil(max_ml/256)][9] block partials of the above
  double* d_virial;          // caller's DEVICE [9] output, or nullptr = virial off
  float* pos_scaled;         // [max_atoms][3] positions converted to Angstrom (unit conversion on)
  double len_scale, e_scale; // Angstrom per caller length unit; caller energy units per eV (1, 1 = off)
  int reuse_every;           // > 1: the cell binning is reused for reuse_every - 1 evaluations after a full one
  double reuse_skin;         // Angstrom per caller length unit applied at use; cells are cut >= Rcr + skin wide
  int reuse_left;            // refresh-only evaluations left before the next full binning
  int64_t reuse_n_atoms, reuse_n_ml; float reuse_box[9]; const void* reuse_ml; const void* reuse_Z;   // what the stored order belongs to
  const int32_t* ext_pairs;  // caller's DEVICE [n_ext_pairs][2] candidate pair list, or nullptr = own cell search
  int64_t n_ext_pairs;
  void* tc_ws;               // tensor-core path scratch
  const int* tile_done;      // per-tile completion flags of the last MLP launch (tcgen05 path), or nullptr
  int tile_done_target;      // value a finished tile's flag holds (= ensemble members)
  int profiling;             // 1: record a CUDA event at every stage boundary of nnp_eval
  cudaEvent_t ev[8];         // 0 start, 1 after neighbour, 2 after AEV fwd, 3 after MLP, 4 after AEV bwd, 5 end
  // host-buffer entry point
  float* hd_pos; int32_t* hd_Z; int32_t* hd_ml; float* hd_forces;
  double* hd_energy;         // mapped pinned HOST word the output kernel writes the energy to (hd_energy_dev = its device alias)
  double* hd_energy_dev;
  int32_t* hz_copy; int32_t* hml_copy;   // pinned host copies of Z / ml_index as last uploaded
  int64_t hz_n, hml_n; int hz_valid, hml_valid;
};

namespace nnp {
// Programmatic dependent launch (PDL): every kernel of one evaluation after k_prep is launched with the
// programmatic-stream-serialization attribute, triggers its dependents at its top and then waits for its
// predecessor's completion (griddepcontrol.wait: full completion + memory flush), so launch latency and block
// scheduling of kernel n+1 overlap the tail of kernel n.  k_aev_backward alone does not wait for the whole MLP
// kernel but per tile (force.cu).  Stage profiling (events between the kernels) switches the attribute off.
#ifdef __CUDACC__
// Step timeline: where the kernels of ONE evaluation sit in time when they run as the PDL chain (ncu serialises them, stage
// profiling too).  Profiling scaffolding, compiled in only with -DNNP_STEP_TIMELINE (NNP_EXTRA_NVCC_FLAGS of build.py; read by
// `python -m paper_2604_21441_b200.step_timeline`): thread 0 of every block records %globaltimer into the slot of its kernel --
// {first block in, first block past griddepcontrol.wait, last block out, last block in, mark: first, mark: last}.  One array per
// translation unit (no relocatable device code), each with an export of its own.  The product build carries none of this.
#ifdef NNP_STEP_TIMELINE
static __device__ unsigned long long g_step_tl[4][6];
__device__ __forceinline__ unsigned long long tl_now() { unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
struct TlScope {
  int k;
  __device__ __forceinline__ explicit TlScope(int k_) : k(k_) {
    if (threadIdx.x == 0) { const unsigned long long t = tl_now(); atomicMin(&g_step_tl[k][0], t); atomicMax(&g_step_tl[k][3], t); }
  }
  __device__ __forceinline__ ~TlScope() { if (threadIdx.x == 0) atomicMax(&g_step_tl[k][2], tl_now()); }
};
#define TL_SCOPE(k) TlScope tl_scope_(k)
#define TL_WAITED(k) do { if (threadIdx.x == 0) atomicMin(&g_step_tl[k][1], tl_now()); } while (0)
#define TL_MARK(k) do { if (threadIdx.x == 0) { const unsigned long long t_ = tl_now(); atomicMin(&g_step_tl[k][4], t_); atomicMax(&g_step_tl[k][5], t_); } } while (0)
// host: copy the unit's slots out (h[24]) and re-arm them (minima to ~0, maxima to 0)
#define TL_EXPORT(name)                                                                                            \
  extern "C" int name(unsigned long long* h) {                                                                     \
    if (cudaMemcpyFromSymbol(h, nnp::g_step_tl, sizeof(nnp::g_step_tl)) != cudaSuccess) return NNP_ERR_CUDA;                  \
    unsigned long long z[4][6];                                                                                    \
    for (int k = 0; k < 4; ++k) { z[k][0] = z[k][1] = z[k][4] = ~0ull; z[k][2] = z[k][3] = z[k][5] = 0ull; }        \
    return cudaMemcpyToSymbol(nnp::g_step_tl, z, sizeof(z)) == cudaSuccess ? NNP_OK : NNP_ERR_CUDA;                      \
  }
#else
#define TL_SCOPE(k) do { } while (0)
#define TL_WAITED(k) do { } while (0)
#define TL_MARK(k) do { } while (0)
#define TL_EXPORT(name)
#endif
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
template <class... KArgs, class... Args>
inline void launch_pdl(bool pdl, cudaStream_t st, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
  cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}
#endif
inline void prof_mark(nnp_workspace* ws, int i) { if (ws->profiling) cudaEventRecord(ws->ev[i], ws->stream); }
// stage launchers (each returns the number of kernels it launched)
int launch_neighbor_stage(nnp_workspace* ws, const float* d_pos, const int32_t* d_Z, const float* box, int pbc,
                          const int32_t* d_ml, int64_t n_atoms, int64_t n_ml);
int prep_cluster_size();
int cell_cap();   // atoms per cell in the fast binning's append buffers
bool box_is_triclinic(const float* box);
bool neighbor_box_ok(const nnp_workspace* ws, const float* box);
int launch_aev_forward(nnp_workspace* ws, int64_t n_ml);
bool small_front_applicable(const nnp_workspace* ws, const float* box, int pbc, int64_t n_ml);
bool small_all_applicable(const nnp_workspace* ws, const float* box, int pbc, int64_t n_ml);
int launch_small_all(nnp_workspace* ws, const float* d_pos, const int32_t* d_Z, const float* box, const int32_t* d_ml,
                     int64_t n_atoms, int64_t n_ml, double* d_energy, float* d_forces);
int small_all_prepare(nnp_workspace* ws);
int launch_small_front(nnp_workspace* ws, const float* d_pos, const int32_t* d_Z, const float* box, const int32_t* d_ml,
                       int64_t n_atoms, int64_t n_ml);
int launch_mlp_simt(nnp_workspace* ws, int64_t n_ml);
int launch_mlp_tc(nnp_workspace* ws, int64_t n_ml);
// the layer-1 image check / repack + L2 prefetch of the MLP operands, ahead of the MLP kernel (see launch_tc_pack)
int launch_tc_pack(nnp_workspace* ws);
// the pending position upload of nnp_eval_host, as a copy (no-op when there is none)
void flush_pos_upload(nnp_workspace* ws);
int launch_force_stage(nnp_workspace* ws, int64_t n_atoms, int64_t n_ml, const int32_t* d_ml, double* d_energy,
                       float* d_forces);
int tc_model_create(nnp_model* m, const nnp_mlp_desc* nets /* [n_members][n_species] */);
void tc_model_destroy(nnp_model* m);
int tc_workspace_create(nnp_workspace* ws);
void tc_workspace_destroy(nnp_workspace* ws);
int tc_read_timeline(long long* h64);
}  // namespace nnp
