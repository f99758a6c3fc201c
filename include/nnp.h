/* nnp.h -- C-ABI boundary of the B200-native NNP energy+force evaluator.
 *
 * One call of nnp_eval = one evaluation of the ML potential behind the paper's ML/MM interface:
 *   inputs  = atomic numbers, positions, simulation box, PBC type, ML index group (PAPER.md line 77,
 *             "multiple inputs to the model can be specified, such as atomic numbers, positions, the
 *             simulation box and type of periodic boundary conditions ... ML subsystem ... index group");
 *   outputs = E_ML and F_i = -grad_i E_ML (eq. 2), the forces being
 *             "supplied directly by the model".
 * The model is the ANI / Behler-Parrinello descriptor network fixed by BASELINE.json (north_star stages
 * 1-4) and restated in SURVEY.md Appendix A; DESIGN.md lists every reading taken.
 *
 * Conventions
 *   - every function returns an int status: NNP_OK (0) or a negative NNP_ERR_* code; no exceptions/aborts.
 *   - "host" / "device" is stated for every pointer.  Device pointers are owned by the caller.
 *   - units are nominal: Angstrom in, "eV" and "eV/Angstrom" out (weights are synthetic).
 *   - nnp_eval is asynchronous on the workspace stream, allocates nothing and never synchronises, so a
 *     sequence of calls can be captured into a CUDA graph.  Device-side faults (unknown species,
 *     neighbour overflow, coincident atoms) are recorded in a sticky flag read by nnp_status().
 *   - there is NO CPU fallback: without a CUDA device every compute entry point returns NNP_ERR_CUDA.
 */
#ifndef NNP_H_
#define NNP_H_
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NNP_OK 0
#define NNP_ERR_INVALID_ARG (-1)     /* null/negative/unsorted/out-of-range argument, dims[0] != AEV length */
#define NNP_ERR_UNKNOWN_SPECIES (-2) /* an ML atom's Z has no species slot or no network (MM atoms' Z unread) */
#define NNP_ERR_BOX_UNSUPPORTED (-3) /* not orthorhombic / GROMACS-triclinic, or a triclinic box too small     */
#define NNP_ERR_CAPACITY (-4)        /* a neighbour row overflowed the workspace's row capacity                */
#define NNP_ERR_COINCIDENT (-5)      /* two ML atoms at distance exactly 0                                     */
#define NNP_ERR_CUDA (-6)            /* CUDA runtime error or no device                                        */
#define NNP_ERR_UNSUPPORTED (-7)     /* descriptor shape outside the kernels' range (see nnp_model_create)     */
#define NNP_ERR_STALE (-8)           /* cell binning reused beyond its validity (nnp_workspace_set_bin_reuse)   */
#define NNP_ERR_STATIC_LIMIT (-9)    /* size beyond the fixed maximum of a no-allocation entry point            */

typedef struct nnp_model nnp_model;         /* opaque, immutable after create, shareable between workspaces */
typedef struct nnp_workspace nnp_workspace; /* opaque scratch, one per stream, not thread-safe              */

/* Descriptor hyper-parameters (BASELINE.json configs[0]). All arrays are HOST
 * arrays and are copied.  AEV length = n_species*nShfR + n_species*(n_species+1)/2 * nShfA*nShfZ;
 * element order: radial s*nShfR+m, angular n_species*nShfR + p(s1,s2)*nShfA*nShfZ + a*nShfZ + z with
 * p = s1*S - s1*(s1-1)/2 + (s2-s1), s1 <= s2 (reading #11). */
typedef struct {
  double Rcr, Rca, EtaR, EtaA, Zeta;
  int32_t nShfR, nShfA, nShfZ;
  const double *ShfR, *ShfA, *ShfZ;
  double radial_prefactor;  /* c_R, 0.25 (reading #2)                                 */
  double cos_scale;         /* c_theta, 0.95: theta = acos(c_theta cos) (reading #3)  */
  int32_t n_species;
  const int32_t* species_Z; /* [n_species] slot -> atomic number, e.g. {1,6,7,8}      */
} nnp_aev_params;

/* One per species slot; n_layers = 0 => the slot has no network (an ML atom of it is an error). */
typedef struct {
  int32_t n_layers;        /* 1..4 layers; hidden layers CELU(alpha), last layer linear (reading #14)   */
  const int32_t* dims;     /* HOST [n_layers+1]; dims[0] = AEV length, dims[n_layers] = 1               */
  const float* const* W;   /* HOST W[l]: dims[l+1] x dims[l], row-major [out][in]                       */
  const float* const* b;   /* HOST b[l]: dims[l+1]                                                      */
  double celu_alpha;       /* 0.1                                                                       */
} nnp_mlp_desc;

/* MLP arithmetic (nnp_workspace_set_mlp_mode):
 *   NNP_MLP_FP32_SIMT  fp32 FMA on CUDA cores (reference rung of the precision ladder, slow)
 *   NNP_MLP_F16X3      tcgen05 tensor cores, every operand split x = hi + lo in fp16, three products
 *                      hi*hi + lo*hi + hi*lo accumulated in fp32 TMEM: fp32-grade results (default)
 *   NNP_MLP_F16X1      tcgen05, the single fp16 product hi*hi (3x fewer MMAs; force error ~6e-4 RMS
 *                      relative, inside the 1e-3 bar with little margin -- see DESIGN.md) */
#define NNP_MLP_FP32_SIMT 0
#define NNP_MLP_F16X3 1
#define NNP_MLP_F16X1 2

/* Creates the immutable model: copies parameters, uploads weights (and the derived fp16 hi/lo tile
 * images) to the current CUDA device.  Limits: n_species <= 8, nShfR == 16, nShfA == 4, nShfZ == 8 (the kernels' lane
 * mappings), hidden widths multiples of 16 and <= 256, n_layers <= 4  -> otherwise NNP_ERR_UNSUPPORTED.
 * The tensor-core modes additionally need n_layers == 4, hidden widths multiples of 32 and |w| < 6e4
 * (fp16 range); a model outside that runs in NNP_MLP_FP32_SIMT (about 8x slower MLP stage) and set_mlp_mode(F16*)
 * returns UNSUPPORTED -- nnp_model_default_mlp_mode() tells which arithmetic a new workspace of the model starts in. */
int nnp_model_create(const nnp_aev_params* aev, const nnp_mlp_desc* nets /* HOST [n_species] */, nnp_model** out);
/* Ensemble of n_members (1..8) networks per element, E = mean of the members' energies -- ANI-2x "is an ensemble of 8
 * networks".  nets: HOST [n_members][n_species], member-major; every member must have the same
 * layer widths per species.  nnp_model_create is the n_members = 1 case.  All members share one AEV.
 * The members of a tile hand over in order between the co-resident CTAs of ONE persistent kernel, so two ensemble MLP
 * kernels must not share the device.  The library enforces that: ensemble evaluations of ALL workspaces of the process
 * are ordered across streams with an event (each waits for the previous ensemble MLP launch), so workspaces on several
 * streams are safe to use concurrently -- their MLP stages simply do not overlap.  Not enforced while a stream is being
 * captured into a CUDA graph: do not replay ensemble graphs concurrently on several streams. */
int nnp_model_create_ensemble(const nnp_aev_params* aev, const nnp_mlp_desc* nets, int32_t n_members, nnp_model** out);
int nnp_model_destroy(nnp_model*);
int nnp_model_aev_length(const nnp_model*);
/* NNP_MLP_F16X3 if the model has tensor-core weight images, NNP_MLP_FP32_SIMT if its networks fall outside the tensor-core
 * shape limits above (the fall-back is not silent: ask here); NNP_ERR_INVALID_ARG for a NULL model. */
int nnp_model_default_mlp_mode(const nnp_model*);

/* Allocates all device scratch for up to max_ml_atoms ML atoms out of up to max_atoms atoms.
 * cuda_stream: a cudaStream_t (0 = legacy default stream).  Neighbour-row capacities default to
 * 128 radial / 48 angular (observed maxima on liquid water: 71 / 26). */
int nnp_workspace_create(const nnp_model*, int64_t max_atoms, int64_t max_ml_atoms, void* cuda_stream,
                         nnp_workspace** out);
int nnp_workspace_destroy(nnp_workspace*);
int nnp_workspace_set_mlp_mode(nnp_workspace*, int32_t mode);
/* dense != 0: materialise every AEV column block (K = full padded AEV length, "as ANI would run it");
 * 0 (default): only the column blocks that can be non-zero for the species present in the evaluation
 * (exact structural-zero compaction).  Results are identical up to summation order. */
int nnp_workspace_set_dense_k(nnp_workspace*, int32_t dense);
/* Unit conversion at the boundary (the MD engine's job in PAPER.md lines 75-77: GROMACS works in nm and kJ/mol).
 * Positions and box are multiplied by angstrom_per_length_unit in fp64 and rounded to fp32 once; the model then runs
 * in Angstrom / "eV" as always; E and the virial are multiplied by energy_units_per_ev, forces by
 * energy_units_per_ev * angstrom_per_length_unit.  GROMACS: (10.0, 96.48533212).  Default (1, 1) = no conversion. */
int nnp_workspace_set_units(nnp_workspace*, double angstrom_per_length_unit, double energy_units_per_ev);
/* Strain derivative of the energy (the quantity a barostat needs; NPT runs in PAPER.md lines 92-94): with
 * d_virial9 != NULL every later nnp_eval also writes DEVICE d_virial9[3*a+b] = dE/d eps_ab for the homogeneous
 * deformation r -> (1 + eps) r of positions and box, accumulated from the pair partials of the force kernel,
 *     W[a][b] = sum_i sum_{j in N(i)} (dE_i/dr_j)[a] (r_j - r_i)[b]      (minimum-image displacements),
 * in 2^-32 fixed point (reproducible).  NULL (default) switches it off; the pointer must stay valid while set. */
int nnp_workspace_set_virial_output(nnp_workspace*, double* d_virial9);

/* Small-system path (the ML/MM regime of PAPER.md lines 108, 140, 154, 164: 14-107 ML
 * atoms, where per-step latency -- kernel launches -- is what counts).  A periodic orthorhombic evaluation with at most
 * 256 ML atoms, box lengths <= 64 Angstrom and no external pair list is taken off the general cell-list path:
 *   on = 2 (default): the WHOLE evaluation is ONE kernel launch with no grid-wide barrier (k_small_all): per-CTA redundant
 *          ordering, all-pairs neighbour search in shared memory, AEV, the per-element networks forward + backward in
 *          plain fp32 on CUDA cores (whatever nnp_workspace_set_mlp_mode says: 2 x 10^5 MACs per atom do not fill a
 *          tensor-core tile), AEV backward, fixed-point force assembly, output by the last CTA to finish.  Needs the
 *          tensor-core-shaped networks (four layers, widths multiples of 32), no virial output, no unit conversion and
 *          no stage profiling; otherwise it falls back to on = 1;
 *   on = 1: only the front end (species map ... AEV) is one kernel; MLP (tensor cores), AEV backward and output follow as
 *          separate launches (five in all);
 *   on = 0: always the general cell-list path.
 * Rows, E and F are those of the general path up to fp32 summation order (and the MLP arithmetic mode). */
int nnp_workspace_set_small_path(nnp_workspace*, int32_t on);

/* Verlet-buffered reuse of the cell binning AND the neighbour rows over several MD steps (
 * the engine's own pair list lives for many steps -- the paper's runs update GROMACS' lists every 10-100
 * steps).  every_n <= 1 (default): every nnp_eval bins, sorts and searches from scratch.  every_n > 1: the cell grid is cut
 * with edges >= Rcr + skin and a full evaluation additionally keeps, per centre, its WIDE row: every neighbour within
 * Rcr + skin.  For the every_n - 1 evaluations that follow -- same n_atoms, n_ml, box, pbc and the SAME atoms behind d_Z /
 * d_ml_index (caller's responsibility; nnp_eval_host compares the contents) -- binning, scan, ordering and the 27-cell
 * candidate sweep are replaced by a refresh pass (positions re-read into the stored order) and a pass over the wide rows
 * that decides every stored pair from the CURRENT positions with the pinned predicate (fp32 outside the guard band, fp64
 * inside).  The effective rows, E and F are therefore exactly those of a full evaluation on the same order of atoms, as
 * long as no atom has moved by more than skin / 2 since the last full evaluation; one that has raises NNP_ERR_STALE through
 * nnp_status() (outputs of that step unspecified, the next evaluation rebuilds).  skin in the caller's length unit.
 * Periodic boxes (orthorhombic or triclinic) on the cell-list path; with an external pair list set only the binning is
 * reused (the list is the engine's own buffered list); open boundaries and the small-system front end keep rebuilding every
 * step.  The first call with every_n > 1 allocates the wide rows (256 entries = 1 KB per ML atom; liquid water at skin 1 A: about 105 entries; a row that does not fit raises NNP_ERR_CAPACITY).  The step counter lives on the
 * host: a CUDA graph captures whichever kind of step it was recorded on. */
int nnp_workspace_set_bin_reuse(nnp_workspace*, int32_t every_n, double skin);

/* External pair list ("The 2026 version adds the internal pair-list built by GROMACS ... as
 * available inputs").  With d_pairs != NULL every later nnp_eval takes its neighbour
 * candidates from this list instead of its own cell search:
 *   d_pairs  DEVICE [n_pairs][2] int32 GLOBAL atom indices (i, j), i != j, in any order; every unordered pair at most
 *            once; it must contain every ML-ML pair within the radial cut-off under the minimum-image convention and
 *            may contain more (a Verlet-buffered list): each pair is decided by the same pinned fp64 predicate as the
 *            cell search, so the neighbour rows -- and E, F -- are those of nnp_eval without a list.  Pairs with a
 *            non-ML end are ignored.  Read during every evaluation: the buffer must stay valid and unchanged while set.
 * A pair listed twice or with i == j raises NNP_ERR_INVALID_ARG through nnp_status().  d_pairs = NULL (default)
 * returns to the built-in cell search.  The list may be replaced between evaluations (list reuse over several MD
 * steps is the caller's choice of buffer width). */
int nnp_workspace_set_pair_list(nnp_workspace*, const int32_t* d_pairs, int64_t n_pairs);

/* One energy+force evaluation.  Asynchronous on the workspace stream.
 *   d_pos      DEVICE [n_atoms][3] fp32, Angstrom, any periodic image
 *   d_Z        DEVICE [n_atoms] int32 atomic numbers (only ML atoms' entries are read)
 *   box        HOST   [9] row vectors a,b,c in Angstrom (read during the call): orthorhombic, or triclinic in the
 *                     GROMACS convention a = (ax,0,0), b = (bx,by,0), c = (cx,cy,cz) with |bx| <= ax/2, |cx| <= ax/2,
 *                     |cy| <= by/2 and at least three cut-off wide cells between every pair of opposite faces
 *                     (face distance >= 3.0003 Rcr); a triclinic evaluation always takes the cell-list path
 *   pbc        1 = xyz periodic (minimum image), 0 = open boundaries (box ignored)
 *   d_ml_index DEVICE [n_ml] int32 strictly ascending atom indices, or NULL => all atoms are ML (n_ml ignored)
 *   d_energy   DEVICE [1] fp64
 *   d_forces   DEVICE [n_atoms][3] fp32; rows of non-ML atoms are set to +0.0f
 * Returns NNP_ERR_INVALID_ARG for sizes beyond the workspace, NNP_ERR_BOX_UNSUPPORTED for a bad box.
 * Content errors found on the device (unsorted ml_index, unknown species, overflow, coincident atoms)
 * surface through nnp_status(); outputs are then unspecified. */
int nnp_eval(nnp_workspace*, int64_t n_atoms, const float* d_pos, const int32_t* d_Z, const float box[9],
             int32_t pbc, const int32_t* d_ml_index, int64_t n_ml, double* d_energy, float* d_forces);

/* Same evaluation with HOST buffers: copies inputs to workspace-owned device buffers, runs nnp_eval,
 * copies energy and forces back and synchronises the stream.  h_ml_index may be NULL.  This is the
 * end-to-end entry point a host MD engine (GROMACS nnpot) would call.  Per call: ONE host-to-device
 * copy (positions) and ONE device-to-host copy (forces) -- none for the forces when h_forces is pinned (device-mapped) host
 * memory, all atoms are ML atoms and the cell-list path runs: the output kernel then writes them in the caller's order
 * straight into h_forces (coalesced stores over PCIe), and pinned positions are uploaded by the binning kernel itself
 * (each block streams the 3 KB of its atoms) instead of by a copy in front of it.  A small ML region inside a system of >= 2048 atoms (the one-kernel
 * path) with pinned h_pos and h_forces runs without either copy: the kernel uses both buffers in place.  The energy
 * arrives through a mapped pinned word the output kernel writes; atomic numbers and the ML index are compared with the copy of the previous call and uploaded only when
 * they changed (a change also ends any binning reuse: the next evaluation bins afresh). */
int nnp_eval_host(nnp_workspace*, int64_t n_atoms, const float* h_pos, const int32_t* h_Z, const float box[9],
                  int32_t pbc, const int32_t* h_ml_index, int64_t n_ml, double* h_energy, float* h_forces);

/* Link atoms at the ML/MM boundary (eq. 4).  Where the ML region cuts a covalent bond between ML
 * atom link_ml[q] and MM atom link_mm[q], link atom q is stored as row n_atoms + q of the position and force arrays
 * (the arrays hold n_atoms + n_links rows; the caller lists the link rows in the ML index with the link element's
 * atomic number, hydrogen by default).
 *   nnp_link_place : writes r_L = r_ML + d (r_MM - r_ML)/|r_MM - r_ML| into rows n_atoms.. of d_pos (call before nnp_eval)
 *   nnp_link_spread: adds the chain-rule shares of the link rows of d_forces onto the bonded atoms and zeroes the
 *                    link rows (call after nnp_eval): F_ML += F_L - (d/l)(F_L - u(u.F_L)), F_MM += (d/l)(F_L - u(u.F_L))
 * d = link distance in the SAME length unit as d_pos and box (PAPER.md default: 1.0 Angstrom; the link kernels take no
 * workspace and do no unit conversion -- a caller working in nm with nnp_workspace_set_units(10, ...) passes d = 0.1);
 * bond vectors take the minimum image when pbc != 0 (box as in
 * nnp_eval, HOST: orthorhombic or GROMACS-style triclinic).  d_link_ml / d_link_mm: DEVICE [n_links] int32 atom indices < n_atoms.  Asynchronous on the given
 * cudaStream_t; out-of-range indices and zero-length bonds are skipped.  Returns NNP_ERR_INVALID_ARG / _BOX_UNSUPPORTED
 * for bad arguments. */
int nnp_link_place(void* cuda_stream, int64_t n_atoms, int64_t n_links, const int32_t* d_link_ml,
                   const int32_t* d_link_mm, double d, const float box[9], int32_t pbc, float* d_pos);
int nnp_link_spread(void* cuda_stream, int64_t n_atoms, int64_t n_links, const int32_t* d_link_ml,
                    const int32_t* d_link_mm, double d, const float box[9], int32_t pbc, const float* d_pos,
                    float* d_forces);

/* Synchronises the stream and returns the sticky device status (NNP_OK or the first NNP_ERR_* seen),
 * then clears it. */
int nnp_status(nnp_workspace*);
const char* nnp_strerror(int);

/* Debug / parity exports of the LAST evaluation (synchronising; HOST output buffers).
 *   nnp_debug_neighbors: which = 0 radial (R <= Rcr), 1 angular (R <= Rca).  CSR over ML rows in
 *     ml_index order; h_col = GLOBAL atom indices, ascending within a row.  Pass h_col = NULL (or a too
 *     small cap) to query *n_pairs only.
 *   nnp_debug_aev: fp32 AEV rows [n_ml][aev_length] in ml_index order.
 *   nnp_debug_daev: fp32 dE_i/dAEV_i rows [n_ml][aev_length] in ml_index order (output of K6); columns of
 *     species absent from the evaluation are reported as 0 (they are never materialised).
 *   nnp_debug_atomic_energies: [n_ml] in ml_index order.
 *   nnp_debug_counters: launches[0] = number of kernels launched by the last nnp_eval. */
int nnp_debug_neighbors(nnp_workspace*, int which, int64_t* n_pairs, int32_t* h_row_start, int32_t* h_col,
                        int64_t col_cap);
int nnp_debug_aev(nnp_workspace*, float* h_aev);
int nnp_debug_daev(nnp_workspace*, float* h_daev);
int nnp_debug_atomic_energies(nnp_workspace*, float* h_e);
int nnp_debug_counters(nnp_workspace*, int64_t* launches);
/* SM-clock ticks of the tensor-core MLP kernel's CTA 0 over its first 32 GEMM rounds (HOST h_ticks[64]): even
 * entries = operand handed to the MMA warp, odd entries = accumulator complete.  Differences give the time spent
 * in epilogues (odd -> next even) and in MMA rounds (even -> odd); used by the profiling notes.  Profiling scaffolding:
 * only a library built with -DNNP_TC_TIMELINE (NNP_EXTRA_NVCC_FLAGS of build.py) records it; the default build carries no
 * instrumentation in the kernel and returns NNP_ERR_UNSUPPORTED here. */
int nnp_debug_mlp_timeline(nnp_workspace*, int64_t* h_ticks);
/* Stage timing of nnp_eval with CUDA events on the workspace stream.  set_profiling(1) makes every later
 * nnp_eval record an event at each stage boundary (not capturable into a CUDA graph while on);
 * nnp_debug_stage_times waits for the last evaluation and writes HOST ms[5] = {neighbour stage K0-K2,
 * AEV forward K3, MLP forward+backward K4-K6, AEV backward K7 (pair partials + scatter), force output +
 * energy reduction K8}. */
int nnp_workspace_set_profiling(nnp_workspace*, int32_t on);
int nnp_debug_stage_times(nnp_workspace*, float* ms);
/* Measured FP32-pipe peak of the current device: the denominator of the AEV kernels' roofline fractions (BASELINE.md
 * section 4 asks for "a register-resident FMA loop" measurement).  Runs a register-resident loop
 * of independent FMA chains on every SM (8 blocks of 256 threads per SM), timed with CUDA events on cuda_stream, and
 * writes HOST *h_tflops = best of 5 launches, counting 2 flop per FMA lane.  variant 0: scalar FFMA with three register
 * operands; variant 1: packed FFMA2 (fma.rn.f32x2, two FMA lanes per instruction, sm_100).  Synchronises the stream. */
int nnp_debug_fp32_peak(void* cuda_stream, int32_t variant, double* h_tflops);

/* The energy reduction of K8 without a workspace and WITHOUT ANY ALLOCATION (eq. 2: E is the sum of the
 * atomic network outputs) -- for callers that cannot call cudaMalloc (CUDA graph capture, tight
 * serving loops, harnesses that forbid it):  *d_energy = e_scale * sum_{i < n} d_e_atom[i], summed in fp64 in a fixed order
 * (block partials, then the last block adds them in index order): bitwise reproducible, no floating-point atomics.
 *   cuda_stream  cudaStream_t of the CURRENT device (the call is asynchronous on it)
 *   d_e_atom     DEVICE [n] fp32 atomic energies (e.g. what nnp_debug_atomic_energies reports), read-only
 *   e_scale      factor on the sum (1.0 = same unit as the inputs)
 *   d_energy     DEVICE [1] fp64, written by the kernel
 * Scratch: a static device array inside the library (33 024 bytes on every GPU that loads it, held until exit); the call
 * uses no cudaMalloc / cudaFree and no allocating routine (one cudaMemsetAsync of the ticket line + one kernel).
 * n > NNP_STATIC_MAX_ATOMS returns NNP_ERR_STATIC_LIMIT (nothing launched); n == 0 writes 0.0; bad pointers / n < 0
 * NNP_ERR_INVALID_ARG.  ALL calls on a device share the one scratch array: calls in one stream are ordered and safe; calls
 * whose kernels may overlap on the GPU (different streams without a dependency) RACE and give wrong sums -- serialise them. */
#define NNP_STATIC_MAX_ATOMS 1048576
int nnp_energy_sum_static(void* cuda_stream, int64_t n, const float* d_e_atom, double e_scale, double* d_energy);

#ifdef __cplusplus
}
#endif
#endif /* NNP_H_ */
