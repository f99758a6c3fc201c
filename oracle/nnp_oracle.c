/* nnp_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the hot path computes: one energy+force evaluation of
 * an ANI / Behler-Parrinello descriptor network,
 *     E = sum_{i in ML} MLP_{s_i}( AEV_i({r_j - r_i}_{j in ML}) ),   F = -dE/dr
 * ("E_ML is a function of the atomic coordinates and nuclear charges", line 51
 * eq. 2 F_i = -grad_i E_ML; model interface PAPER.md line 77).  PAPER.md does not spell the model
 * out; the functional form is the one restated in SURVEY.md Appendix A from BASELINE.json
 * (north_star stages 1-4, configs[0] hyper-parameters) -- every formula below cites it.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code with paper_2604_21441_b200/csrc and includes none of its headers.
 * Parity pins (tests/test_oracle_pins.py): Appendix-B closed forms, finite-difference forces,
 * invariances, autograd restatement, brute-force O(N^2) neighbour definition.  No function here is
 * "parity unpinned".
 *
 * OpenMP is used only as `parallel for` over centre atoms (SURVEY.md section 8.d "CPU baseline").
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
  double Rcr, Rca, EtaR, EtaA, Zeta;
  int32_t nShfR, nShfA, nShfZ;
  const double *ShfR, *ShfA, *ShfZ;
  double c_R;      /* radial prefactor, 0.25 (reading #2) */
  double c_theta;  /* cos scale, 0.95 (reading #3)        */
  int32_t S;       /* number of species slots             */
  const int32_t* species_Z; /* [S] slot -> atomic number  */
} orc_aev_params;

typedef struct {
  int32_t n_layers;        /* 0 => no network for this slot                   */
  const int32_t* dims;     /* [n_layers+1], dims[0] = AEV length, last = 1    */
  const float* const* W;   /* W[l]: dims[l+1] x dims[l], row-major [out][in]  */
  const float* const* b;   /* b[l]: dims[l+1]                                 */
  double alpha;            /* CELU alpha                                      */
} orc_mlp;

enum { ORC_OK = 0, ORC_ERR_ARG = -1, ORC_ERR_SPECIES = -2, ORC_ERR_BOX = -3, ORC_ERR_CAP = -4, ORC_ERR_COINCIDENT = -5 };

int orc_aev_length(const orc_aev_params* p) {
  return p->S * p->nShfR + p->S * (p->S + 1) / 2 * p->nShfA * p->nShfZ;
}

/* Cut-off (App. A): f_C(R;Rc) = 0.5 cos(pi R/Rc) + 0.5 for R <= Rc, else 0. */
double orc_fc(double R, double Rc) { return R <= Rc ? 0.5 * cos(M_PI * R / Rc) + 0.5 : 0.0; }
static double fc_prime(double R, double Rc) { return R <= Rc ? -0.5 * M_PI / Rc * sin(M_PI * R / Rc) : 0.0; }

/* CELU (App. A, reading #14). */
double orc_celu(double x, double a) { return x > 0.0 ? x : a * (exp(x / a) - 1.0); }
static double celu_prime(double x, double a) { return x > 0.0 ? 1.0 : exp(x / a); }

/* Minimum-image displacement and the pinned neighbour predicate (section 8.c step 2, readings #6, #7):
 * d = r_j - r_i on fp32 inputs promoted to fp64; d_a -= L_a * rint(d_a / L_a);
 * d2 = fma(dz,dz, fma(dy,dy, dx*dx)).
 * Triclinic boxes (reading #35) in the GROMACS convention: rows
 * a = (ax,0,0), b = (bx,by,0), c = (cx,cy,cz) with |bx| <= ax/2, |cx| <= ax/2, |cy| <= by/2.  The box is held as
 * L[6] = {ax, by, cz, bx, cx, cy}; the image is first reduced row by row, c first, then b, then a:
 *     n = rint(dz/cz): d -= n c;   n = rint(dy/by): d -= n b;   n = rint(dx/ax): d -= n a
 * which lands in the brick |dz| <= cz/2, ... but is NOT always the nearest image of a skewed box; the nearest one is
 * then searched among the 27 images d + nc c + nb b + na a, n in {-1,0,1} (loops nc, nb, na outermost to innermost,
 * first strict minimum of d2 wins).  Pinned against a 343-image brute force in tests/test_oracle_pins.py.  With
 * bx = cx = cy = 0 no search is made and the arithmetic is the orthorhombic expression above, bit for bit. */
static double disp(const float* pos, int64_t i, int64_t j, const double L[6], int pbc, double d[3]) {
  for (int a = 0; a < 3; ++a) d[a] = (double)pos[3 * j + a] - (double)pos[3 * i + a];
  if (pbc) {
    double n = rint(d[2] / L[2]);
    d[2] -= L[2] * n; d[1] -= L[5] * n; d[0] -= L[4] * n;
    n = rint(d[1] / L[1]);
    d[1] -= L[1] * n; d[0] -= L[3] * n;
    n = rint(d[0] / L[0]);
    d[0] -= L[0] * n;
    if (L[3] != 0.0 || L[4] != 0.0 || L[5] != 0.0) {
      double best = fma(d[2], d[2], fma(d[1], d[1], d[0] * d[0])), b[3] = {d[0], d[1], d[2]};
      for (int nc = -1; nc <= 1; ++nc)
        for (int nb = -1; nb <= 1; ++nb)
          for (int na = -1; na <= 1; ++na) {
            double v[3] = {d[0], d[1], d[2]};
            v[2] += L[2] * nc; v[1] += L[5] * nc; v[0] += L[4] * nc;
            v[1] += L[1] * nb; v[0] += L[3] * nb;
            v[0] += L[0] * na;
            const double v2 = fma(v[2], v[2], fma(v[1], v[1], v[0] * v[0]));
            if (v2 < best) { best = v2; b[0] = v[0]; b[1] = v[1]; b[2] = v[2]; }
          }
      d[0] = b[0]; d[1] = b[1]; d[2] = b[2];
    }
  }
  return fma(d[2], d[2], fma(d[1], d[1], d[0] * d[0]));
}

static int check_box(const float* box, double L[6]) {
  for (int r = 0; r < 3; ++r)
    for (int c = 0; c < 3; ++c) {
      double v = (double)box[3 * r + c];
      if (r == c) { if (!(v > 0.0)) return ORC_ERR_BOX; L[r] = v; }
      else if (c > r && v != 0.0) return ORC_ERR_BOX; /* lower-triangular rows only (readings #9, #35) */
    }
  L[3] = (double)box[3]; L[4] = (double)box[6]; L[5] = (double)box[7];
  if (fabs(L[3]) > 0.5 * L[0] || fabs(L[4]) > 0.5 * L[0] || fabs(L[5]) > 0.5 * L[1]) return ORC_ERR_BOX;
  return ORC_OK;
}
static int box_is_triclinic(const double L[6]) { return L[3] != 0.0 || L[4] != 0.0 || L[5] != 0.0; }

/* ---------------------------------------------------------------------------------------------
 * Neighbour lists.  mode 0: the definition -- every ordered pair (i,j) of active atoms (O(N^2)).
 * mode 1: a simple CPU cell list (27-cell stencil) applying the *same* predicate; used for the
 * timed baseline on large boxes and verified equal to mode 0 in the tests.
 * Output CSR over ML rows (ml_index order); columns are GLOBAL atom indices, ascending per row.
 * Returns number of pairs (>= 0) or an error code; if cap is too small returns ORC_ERR_CAP.
 * ------------------------------------------------------------------------------------------- */
static int cmp_i32(const void* a, const void* b) { int32_t x = *(const int32_t*)a, y = *(const int32_t*)b; return (x > y) - (x < y); }

typedef struct { int32_t* start; int32_t* col; int64_t n_pairs; } nbr_list;

static void nbr_free(nbr_list* nl) { free(nl->start); free(nl->col); nl->start = nl->col = NULL; }

static int build_neighbors(int64_t n_atoms, const float* pos, const double L[6], int pbc,
                           const int32_t* act, int64_t n_ml, double Rc, int mode, nbr_list* out) {
  const double Rc2 = Rc * Rc;
  if (pbc && box_is_triclinic(L)) mode = 0;   /* the simple cell list below is orthorhombic: use the definition */
  int32_t* count = (int32_t*)calloc((size_t)n_ml + 1, sizeof(int32_t));
  int32_t** rows = (int32_t**)calloc((size_t)n_ml, sizeof(int32_t*));
  int coincident = 0;
  (void)n_atoms;
  if (mode == 0) {
#pragma omp parallel for schedule(dynamic, 16) reduction(| : coincident)
    for (int64_t a = 0; a < n_ml; ++a) {
      int64_t i = act[a];
      int32_t cap = 128, n = 0;
      int32_t* r = (int32_t*)malloc(sizeof(int32_t) * cap);
      for (int64_t b = 0; b < n_ml; ++b) {
        if (b == a) continue;
        int64_t j = act[b];
        double d[3];
        double d2 = disp(pos, i, j, L, pbc, d);
        if (d2 <= Rc2) {
          if (d2 == 0.0) coincident = 1;
          if (n == cap) { cap *= 2; r = (int32_t*)realloc(r, sizeof(int32_t) * cap); }
          r[n++] = (int32_t)j;
        }
      }
      rows[a] = r; count[a] = n;
    }
  } else {
    /* cell list: nc = floor(L / Rc) cells per dimension (>= 1); fewer than 3 => scan every cell once */
    int nc[3];
    for (int a = 0; a < 3; ++a) { nc[a] = pbc ? (int)floor(L[a] / Rc) : 1; if (nc[a] < 1) nc[a] = 1; }
    double lo[3] = {0, 0, 0}, ext[3] = {L[0], L[1], L[2]};
    if (!pbc) { /* bounding-box grid for open boundaries */
      double hi[3] = {-1e300, -1e300, -1e300}; lo[0] = lo[1] = lo[2] = 1e300;
      for (int64_t a = 0; a < n_ml; ++a) for (int k = 0; k < 3; ++k) {
        double x = pos[3 * (int64_t)act[a] + k]; if (x < lo[k]) lo[k] = x; if (x > hi[k]) hi[k] = x; }
      for (int k = 0; k < 3; ++k) { ext[k] = hi[k] - lo[k] + 1e-9; nc[k] = (int)floor(ext[k] / Rc); if (nc[k] < 1) nc[k] = 1; }
    }
    int64_t ncell = (int64_t)nc[0] * nc[1] * nc[2];
    int32_t* cell_of = (int32_t*)malloc(sizeof(int32_t) * (size_t)n_ml);
    int32_t* cstart = (int32_t*)calloc((size_t)ncell + 1, sizeof(int32_t));
    for (int64_t a = 0; a < n_ml; ++a) {
      int c[3];
      for (int k = 0; k < 3; ++k) {
        double f = ((double)pos[3 * (int64_t)act[a] + k] - lo[k]) / ext[k];
        if (pbc) f -= floor(f);
        int ci = (int)floor(f * nc[k]);
        if (ci < 0) ci = 0; if (ci >= nc[k]) ci = nc[k] - 1;
        c[k] = ci;
      }
      cell_of[a] = (c[0] * nc[1] + c[1]) * nc[2] + c[2];
      cstart[cell_of[a] + 1]++;
    }
    for (int64_t c = 0; c < ncell; ++c) cstart[c + 1] += cstart[c];
    int32_t* fill = (int32_t*)malloc(sizeof(int32_t) * (size_t)ncell);
    memcpy(fill, cstart, sizeof(int32_t) * (size_t)ncell);
    int32_t* members = (int32_t*)malloc(sizeof(int32_t) * (size_t)n_ml);
    for (int64_t a = 0; a < n_ml; ++a) members[fill[cell_of[a]]++] = (int32_t)a;
    free(fill);
#pragma omp parallel for schedule(dynamic, 16) reduction(| : coincident)
    for (int64_t a = 0; a < n_ml; ++a) {
      int64_t i = act[a];
      int32_t cap = 128, n = 0;
      int32_t* r = (int32_t*)malloc(sizeof(int32_t) * cap);
      int ci = cell_of[a];
      int c0[3] = {ci / (nc[1] * nc[2]), (ci / nc[2]) % nc[1], ci % nc[2]};
      /* distinct cells of the 3x3x3 stencil (a dimension with < 3 cells is scanned completely) */
      int lst[3][3], nl[3];
      for (int k = 0; k < 3; ++k) {
        if (nc[k] < 3) { nl[k] = nc[k]; for (int q = 0; q < nc[k]; ++q) lst[k][q] = q; }
        else {
          nl[k] = 0;
          for (int q = -1; q <= 1; ++q) {
            int c = c0[k] + q;
            if (pbc) c = (c + nc[k]) % nc[k]; else if (c < 0 || c >= nc[k]) continue;
            lst[k][nl[k]++] = c;
          }
        }
      }
      for (int x = 0; x < nl[0]; ++x) for (int y = 0; y < nl[1]; ++y) for (int z = 0; z < nl[2]; ++z) {
        int c = (lst[0][x] * nc[1] + lst[1][y]) * nc[2] + lst[2][z];
        for (int32_t q = cstart[c]; q < cstart[c + 1]; ++q) {
          int32_t b = members[q];
          if (b == a) continue;
          int64_t j = act[b];
          double d[3];
          double d2 = disp(pos, i, j, L, pbc, d);
          if (d2 <= Rc2) {
            if (d2 == 0.0) coincident = 1;
            if (n == cap) { cap *= 2; r = (int32_t*)realloc(r, sizeof(int32_t) * cap); }
            r[n++] = (int32_t)j;
          }
        }
      }
      qsort(r, (size_t)n, sizeof(int32_t), cmp_i32);
      rows[a] = r; count[a] = n;
    }
    free(cell_of); free(cstart); free(members);
  }
  out->start = (int32_t*)malloc(sizeof(int32_t) * ((size_t)n_ml + 1));
  int64_t tot = 0;
  for (int64_t a = 0; a < n_ml; ++a) { out->start[a] = (int32_t)tot; tot += count[a]; }
  out->start[n_ml] = (int32_t)tot;
  out->col = (int32_t*)malloc(sizeof(int32_t) * (size_t)(tot > 0 ? tot : 1));
  for (int64_t a = 0; a < n_ml; ++a) { memcpy(out->col + out->start[a], rows[a], sizeof(int32_t) * (size_t)count[a]); free(rows[a]); }
  out->n_pairs = tot;
  free(count); free(rows);
  return coincident ? ORC_ERR_COINCIDENT : ORC_OK;
}

static int32_t* active_set(int64_t n_atoms, const int32_t* ml_index, int64_t n_ml) {
  int32_t* act = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n_ml > 0 ? n_ml : 1));
  for (int64_t a = 0; a < n_ml; ++a) act[a] = ml_index ? ml_index[a] : (int32_t)a;
  (void)n_atoms;
  return act;
}

int64_t orc_neighbors(int64_t n_atoms, const float* pos, const float* box, int32_t pbc,
                      const int32_t* ml_index, int64_t n_ml, double Rc, int32_t mode,
                      int32_t* row_start, int32_t* col, int64_t cap) {
  double L[6];
  int rc = check_box(box, L);
  if (rc) return rc;
  if (!ml_index) n_ml = n_atoms;
  int32_t* act = active_set(n_atoms, ml_index, n_ml);
  nbr_list nl;
  rc = build_neighbors(n_atoms, pos, L, pbc, act, n_ml, Rc, mode, &nl);
  free(act);
  if (rc && rc != ORC_ERR_COINCIDENT) { nbr_free(&nl); return rc; }
  int64_t np = nl.n_pairs;
  memcpy(row_start, nl.start, sizeof(int32_t) * ((size_t)n_ml + 1));
  if (np > cap) { nbr_free(&nl); return ORC_ERR_CAP; }
  memcpy(col, nl.col, sizeof(int32_t) * (size_t)np);
  nbr_free(&nl);
  return np;
}

/* ---------------------------------------------------------------------------------------------
 * AEV of one centre (App. A "Radial block", "Angular block"; reading #11 element order).
 * nb: neighbour displacement vectors d_ij (n x 3), distances R, slots s.  Radial neighbours are all
 * n entries (R <= Rcr by construction); the angular subset is R <= Rca decided on d2 <= Rca^2.
 * ------------------------------------------------------------------------------------------- */
static int pair_slot(int s1, int s2, int S) {
  if (s1 > s2) { int t = s1; s1 = s2; s2 = t; }
  return s1 * S - s1 * (s1 - 1) / 2 + (s2 - s1);
}

static void aev_centre(const orc_aev_params* p, int n, const double* d, const double* R, const double* d2,
                       const int* slot, double* G) {
  const int S = p->S, nR = p->nShfR, nA = p->nShfA, nZ = p->nShfZ;
  const int L = orc_aev_length(p);
  const double Rca2 = p->Rca * p->Rca;
  memset(G, 0, sizeof(double) * (size_t)L);
  for (int j = 0; j < n; ++j) {
    double f = orc_fc(R[j], p->Rcr);
    for (int m = 0; m < nR; ++m) {
      double x = R[j] - p->ShfR[m];
      G[slot[j] * nR + m] += p->c_R * exp(-p->EtaR * x * x) * f;
    }
  }
  for (int j = 0; j < n; ++j) {
    if (!(d2[j] <= Rca2)) continue;
    for (int k = j + 1; k < n; ++k) {
      if (!(d2[k] <= Rca2)) continue;
      double u = (d[3 * j] * d[3 * k] + d[3 * j + 1] * d[3 * k + 1] + d[3 * j + 2] * d[3 * k + 2]) / (R[j] * R[k]);
      double theta = acos(p->c_theta * u);
      double Rbar = 0.5 * (R[j] + R[k]);
      double ff = orc_fc(R[j], p->Rca) * orc_fc(R[k], p->Rca);
      int base = S * nR + pair_slot(slot[j], slot[k], S) * nA * nZ;
      for (int a = 0; a < nA; ++a) {
        double x = Rbar - p->ShfA[a];
        double F2 = exp(-p->EtaA * x * x);
        for (int z = 0; z < nZ; ++z) {
          double B = 0.5 * (1.0 + cos(theta - p->ShfZ[z]));
          G[base + a * nZ + z] += 2.0 * pow(B, p->Zeta) * F2 * ff;
        }
      }
    }
  }
}

/* Pair partials p_ij = dE_i/dr_j given g = dE_i/dAEV_i (App. A "Forces").  P: n x 3, zeroed here. */
static void aev_centre_backward(const orc_aev_params* p, int n, const double* d, const double* R, const double* d2,
                                const int* slot, const double* g, double* P) {
  const int S = p->S, nR = p->nShfR, nA = p->nShfA, nZ = p->nShfZ;
  const double Rca2 = p->Rca * p->Rca;
  memset(P, 0, sizeof(double) * 3 * (size_t)n);
  for (int j = 0; j < n; ++j) {
    double f = orc_fc(R[j], p->Rcr), fp = fc_prime(R[j], p->Rcr);
    double coef = 0.0;
    for (int m = 0; m < nR; ++m) {
      double x = R[j] - p->ShfR[m];
      double e = exp(-p->EtaR * x * x);
      coef += g[slot[j] * nR + m] * p->c_R * e * (-2.0 * p->EtaR * x * f + fp);
    }
    for (int a = 0; a < 3; ++a) P[3 * j + a] += coef * d[3 * j + a] / R[j];
  }
  for (int j = 0; j < n; ++j) {
    if (!(d2[j] <= Rca2)) continue;
    for (int k = j + 1; k < n; ++k) {
      if (!(d2[k] <= Rca2)) continue;
      double uj[3], uk[3];
      for (int a = 0; a < 3; ++a) { uj[a] = d[3 * j + a] / R[j]; uk[a] = d[3 * k + a] / R[k]; }
      double u = uj[0] * uk[0] + uj[1] * uk[1] + uj[2] * uk[2];
      double c = p->c_theta * u;
      double theta = acos(c);
      double dtheta_du = -p->c_theta / sqrt(1.0 - c * c);
      double Rbar = 0.5 * (R[j] + R[k]);
      double fj = orc_fc(R[j], p->Rca), fk = orc_fc(R[k], p->Rca);
      double fjp = fc_prime(R[j], p->Rca), fkp = fc_prime(R[k], p->Rca);
      int base = S * nR + pair_slot(slot[j], slot[k], S) * nA * nZ;
      double Aj = 0.0, Ak = 0.0, Au = 0.0;
      for (int a = 0; a < nA; ++a) {
        double x = Rbar - p->ShfA[a];
        double F2 = exp(-p->EtaA * x * x);
        for (int z = 0; z < nZ; ++z) {
          double ang = theta - p->ShfZ[z];
          double B = 0.5 * (1.0 + cos(ang));
          double F1 = pow(B, p->Zeta);
          double dF1 = -0.5 * p->Zeta * pow(B, p->Zeta - 1.0) * sin(ang);
          double gz = g[base + a * nZ + z];
          Aj += gz * 2.0 * F1 * (-p->EtaA * x * F2 * fj * fk + F2 * fjp * fk);
          Ak += gz * 2.0 * F1 * (-p->EtaA * x * F2 * fj * fk + F2 * fj * fkp);
          Au += gz * 2.0 * dF1 * dtheta_du * F2 * fj * fk;
        }
      }
      for (int a = 0; a < 3; ++a) {
        P[3 * j + a] += Aj * uj[a] + Au * (uk[a] - u * uj[a]) / R[j];
        P[3 * k + a] += Ak * uk[a] + Au * (uj[a] - u * uk[a]) / R[k];
      }
    }
  }
}

/* MLP forward (+ optional backward g = dE/dG) of one atom (App. A "Network", "Backward"). */
static double mlp_atom(const orc_mlp* net, const double* G, double* g /* may be NULL */) {
  const int nl = net->n_layers;
  int maxw = 0, tot = 0;
  for (int l = 0; l <= nl; ++l) { if (net->dims[l] > maxw) maxw = net->dims[l]; tot += net->dims[l]; }
  double* z = (double*)malloc(sizeof(double) * (size_t)tot * 2);  /* pre-activations, per layer   */
  double* h = z + tot;                                              /* activations, per layer       */
  int* off = (int*)malloc(sizeof(int) * (size_t)(nl + 1));
  off[0] = 0; for (int l = 1; l <= nl; ++l) off[l] = off[l - 1] + net->dims[l - 1];
  memcpy(h, G, sizeof(double) * (size_t)net->dims[0]);
  for (int l = 0; l < nl; ++l) {
    const int in = net->dims[l], out = net->dims[l + 1];
    const float* W = net->W[l]; const float* b = net->b[l];
    for (int o = 0; o < out; ++o) {
      double acc = (double)b[o];
      for (int i = 0; i < in; ++i) acc += (double)W[(size_t)o * in + i] * h[off[l] + i];
      z[off[l + 1] + o] = acc;
      h[off[l + 1] + o] = (l == nl - 1) ? acc : orc_celu(acc, net->alpha); /* last layer linear */
    }
  }
  double E = h[off[nl]];
  if (g) {
    double* delta = (double*)malloc(sizeof(double) * (size_t)maxw * 2);
    double* nxt = delta + maxw;
    delta[0] = 1.0; /* dE/dz_last */
    for (int l = nl - 1; l >= 0; --l) {
      const int in = net->dims[l], out = net->dims[l + 1];
      const float* W = net->W[l];
      for (int i = 0; i < in; ++i) {
        double acc = 0.0;
        for (int o = 0; o < out; ++o) acc += (double)W[(size_t)o * in + i] * delta[o];
        nxt[i] = (l > 0) ? acc * celu_prime(z[off[l] + i], net->alpha) : acc;
      }
      memcpy(delta, nxt, sizeof(double) * (size_t)in);
    }
    memcpy(g, delta, sizeof(double) * (size_t)net->dims[0]);
    free(delta);
  }
  free(z); free(off);
  return E;
}

/* Standalone exports for the pins. */
double orc_mlp_forward(const orc_mlp* net, const double* G, double* g) { return mlp_atom(net, G, g); }

/* ---------------------------------------------------------------------------------------------
 * Whole evaluation (section 8.c steps 1-5).  forces: [n_atoms][3] fp64, zero for non-ML atoms.
 * Optional outputs (NULL to skip): aev_out [n_ml][L], e_atom [n_ml], daev_out [n_ml][L].
 * want_forces = 0 skips the backward pass (used by the finite-difference driver).
 * ------------------------------------------------------------------------------------------- */
/* virial9 (may be NULL): the strain derivative of the energy, W[a][b] = dE/d eps_ab for the homogeneous deformation
 * r -> (1 + eps) r of positions and box, written out from its pair form:
 *     W[a][b] = sum_i sum_{j in N(i)} p_ij[a] * d_ij[b],   p_ij = dE_i/dr_j,  d_ij = r_j - r_i (minimum image),
 * because E_i depends on the positions only through the displacements d_ij, each of which deforms as d -> (1 + eps) d.
 * Pins (tests/test_oracle_pins.py): central finite differences of the energy under axis scaling (periodic) and shear
 * (open boundaries); symmetry; W = -sum_a F_a (x) r_a for an isolated cluster. */
static int eval_impl(const orc_aev_params* p, const orc_mlp* nets /* [S] */, int64_t n_atoms, const float* pos,
             const int32_t* Z, const float* box, int32_t pbc, const int32_t* ml_index, int64_t n_ml,
             int32_t nbr_mode, int32_t want_forces, double* energy, double* forces,
             double* aev_out, double* e_atom, double* daev_out, double* virial9) {
  double L3[6];
  int rc = check_box(box, L3);
  if (rc) return rc;
  if (!ml_index) n_ml = n_atoms;
  if (n_ml < 0 || n_atoms < 0) return ORC_ERR_ARG;
  const int L = orc_aev_length(p);
  int32_t* act = active_set(n_atoms, ml_index, n_ml);
  for (int64_t a = 0; a < n_ml; ++a) {
    if (act[a] < 0 || act[a] >= n_atoms || (a > 0 && act[a] <= act[a - 1])) { free(act); return ORC_ERR_ARG; }
  }
  /* step 1: species slots of the ML atoms (MM atoms' Z are never inspected) */
  int* slot_of = (int*)malloc(sizeof(int) * (size_t)(n_atoms > 0 ? n_atoms : 1));
  for (int64_t i = 0; i < n_atoms; ++i) slot_of[i] = -1;
  for (int64_t a = 0; a < n_ml; ++a) {
    int s = -1;
    for (int q = 0; q < p->S; ++q) if (p->species_Z[q] == Z[act[a]]) s = q;
    if (s < 0 || nets[s].n_layers == 0) { free(act); free(slot_of); return ORC_ERR_SPECIES; }
    if (nets[s].dims[0] != L) { free(act); free(slot_of); return ORC_ERR_ARG; }
    slot_of[act[a]] = s;
  }
  /* step 2: radial neighbour list */
  nbr_list nl;
  rc = build_neighbors(n_atoms, pos, L3, pbc, act, n_ml, p->Rcr, nbr_mode, &nl);
  if (rc) { nbr_free(&nl); free(act); free(slot_of); return rc; }

  int nthreads = 1;
#ifdef _OPENMP
  nthreads = omp_get_max_threads();
#endif
  double* Fth = NULL;
  if (want_forces) Fth = (double*)calloc((size_t)nthreads * 3 * (size_t)(n_atoms > 0 ? n_atoms : 1), sizeof(double));
  double* Wth = (double*)calloc((size_t)nthreads * 9, sizeof(double));
  double* Ei = (double*)calloc((size_t)(n_ml > 0 ? n_ml : 1), sizeof(double));

#pragma omp parallel
  {
    int tid = 0;
#ifdef _OPENMP
    tid = omp_get_thread_num();
#endif
    double* F = want_forces ? Fth + (size_t)tid * 3 * (size_t)n_atoms : NULL;
    double* G = (double*)malloc(sizeof(double) * (size_t)L * 2);
    double* g = G + L;
    int cap = 256;
    double* d = (double*)malloc(sizeof(double) * (size_t)cap * 8);
    int* sl = (int*)malloc(sizeof(int) * (size_t)cap);
#pragma omp for schedule(dynamic, 8)
    for (int64_t a = 0; a < n_ml; ++a) {
      const int64_t i = act[a];
      const int n = nl.start[a + 1] - nl.start[a];
      if (n > cap) { cap = 2 * n; d = (double*)realloc(d, sizeof(double) * (size_t)cap * 8); sl = (int*)realloc(sl, sizeof(int) * (size_t)cap); }
      double *R = d + 3 * (size_t)cap, *d2 = d + 4 * (size_t)cap, *P = d + 5 * (size_t)cap;
      for (int q = 0; q < n; ++q) {
        int64_t j = nl.col[nl.start[a] + q];
        d2[q] = disp(pos, i, j, L3, pbc, d + 3 * q);
        R[q] = sqrt(d2[q]);
        sl[q] = slot_of[j];
      }
      aev_centre(p, n, d, R, d2, sl, G);                       /* step 3 */
      if (aev_out) memcpy(aev_out + (size_t)a * L, G, sizeof(double) * (size_t)L);
      Ei[a] = mlp_atom(&nets[slot_of[i]], G, want_forces ? g : NULL);  /* step 4 (+5) */
      if (want_forces) {
        if (daev_out) memcpy(daev_out + (size_t)a * L, g, sizeof(double) * (size_t)L);
        aev_centre_backward(p, n, d, R, d2, sl, g, P);
        /* F = -dE/dr: dE_i/dr_j = p_ij, dE_i/dr_i = -sum_j p_ij */
        for (int q = 0; q < n; ++q) {
          int64_t j = nl.col[nl.start[a] + q];
          for (int c = 0; c < 3; ++c) { F[3 * j + c] -= P[3 * q + c]; F[3 * i + c] += P[3 * q + c]; }
          for (int c = 0; c < 3; ++c)
            for (int b = 0; b < 3; ++b) Wth[(size_t)tid * 9 + 3 * c + b] += P[3 * q + c] * d[3 * q + b];
        }
      }
    }
    free(G); free(d); free(sl);
  }
  double E = 0.0;
  for (int64_t a = 0; a < n_ml; ++a) E += Ei[a]; /* index order, fp64 (step 4) */
  *energy = E;
  if (e_atom) memcpy(e_atom, Ei, sizeof(double) * (size_t)n_ml);
  if (want_forces) {
    for (int64_t q = 0; q < 3 * n_atoms; ++q) {
      double s = 0.0;
      for (int t = 0; t < nthreads; ++t) s += Fth[(size_t)t * 3 * (size_t)n_atoms + q];
      forces[q] = s;
    }
    free(Fth);
  }
  if (virial9)
    for (int q = 0; q < 9; ++q) {
      double w = 0.0;
      for (int t = 0; t < nthreads; ++t) w += Wth[(size_t)t * 9 + q];
      virial9[q] = w;
    }
  free(Wth);
  free(Ei); nbr_free(&nl); free(act); free(slot_of);
  return ORC_OK;
}

int orc_eval(const orc_aev_params* p, const orc_mlp* nets /* [S] */, int64_t n_atoms, const float* pos,
             const int32_t* Z, const float* box, int32_t pbc, const int32_t* ml_index, int64_t n_ml,
             int32_t nbr_mode, int32_t want_forces, double* energy, double* forces,
             double* aev_out, double* e_atom, double* daev_out) {
  return eval_impl(p, nets, n_atoms, pos, Z, box, pbc, ml_index, n_ml, nbr_mode, want_forces, energy, forces, aev_out,
                   e_atom, daev_out, NULL);
}

int orc_eval_virial(const orc_aev_params* p, const orc_mlp* nets /* [S] */, int64_t n_atoms, const float* pos,
                    const int32_t* Z, const float* box, int32_t pbc, const int32_t* ml_index, int64_t n_ml,
                    int32_t nbr_mode, double* energy, double* forces, double* virial9) {
  return eval_impl(p, nets, n_atoms, pos, Z, box, pbc, ml_index, n_ml, nbr_mode, 1, energy, forces, NULL, NULL, NULL,
                   virial9);
}

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void orc_set_num_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/* ---------------------------------------------------------------------------------------------
 * Link atoms (section 3, eq. 4): where the ML/MM boundary cuts a covalent bond between
 * ML atom a and MM atom b, a link atom (hydrogen by default) is placed along the bond at a fixed distance d
 * (1 Angstrom by default) from the ML atom,
 *     r_L = r_a + d (r_b - r_a) / |r_b - r_a|,
 * it enters the model as an additional ML atom, and the force the model puts on it is "redistributed" onto a and b
 * (PAPER.md line 82).  The redistribution is the chain rule of eq. 4: with l = |r_b - r_a|, u = (r_b - r_a)/l,
 *     dr_L/dr_a = I - (d/l)(I - u u^T),   dr_L/dr_b = (d/l)(I - u u^T)      (both symmetric), so
 *     F_a += F_L - (d/l)(F_L - u (u.F_L)),   F_b += (d/l)(F_L - u (u.F_L)).
 * Reading (#30): the bond vector is taken under the minimum-image convention when pbc != 0, the link
 * atoms are stored as rows n_atoms .. n_atoms + n_links - 1 of the position / force arrays, and after the spread
 * their force rows are zero.  fp32 in / fp32 out like the hot path, arithmetic in fp64.
 * Pins (tests/test_oracle_pins.py): |r_L - r_a| = d and collinearity; total force and total torque conserved;
 * central finite differences of a scalar function of r_L with respect to r_a and r_b.
 * --------------------------------------------------------------------------------------------- */
static void link_bond(const float* pos, const float* box, int32_t pbc, int32_t a, int32_t b, double* u, double* l) {
  double v[3], s = 0.0;
  for (int k = 0; k < 3; ++k) v[k] = (double)pos[3 * (size_t)b + k] - (double)pos[3 * (size_t)a + k];
  if (pbc) {   /* row-by-row image reduction as in disp(): c, then b, then a (orthorhombic: per component) */
    double n = rint(v[2] / (double)box[8]);
    v[2] -= (double)box[8] * n; v[1] -= (double)box[7] * n; v[0] -= (double)box[6] * n;
    n = rint(v[1] / (double)box[4]);
    v[1] -= (double)box[4] * n; v[0] -= (double)box[3] * n;
    n = rint(v[0] / (double)box[0]);
    v[0] -= (double)box[0] * n;
  }
  for (int k = 0; k < 3; ++k) s += v[k] * v[k];
  *l = sqrt(s);
  for (int k = 0; k < 3; ++k) u[k] = v[k] / *l;
}

int orc_link_place(int64_t n_atoms, int64_t n_links, const int32_t* link_ml, const int32_t* link_mm, double d,
                   const float* box, int32_t pbc, float* pos /* [n_atoms + n_links][3] */) {
  for (int64_t q = 0; q < n_links; ++q) {
    double u[3], l;
    link_bond(pos, box, pbc, link_ml[q], link_mm[q], u, &l);
    if (!(l > 0.0)) return -1;
    for (int k = 0; k < 3; ++k)
      pos[3 * (size_t)(n_atoms + q) + k] = (float)((double)pos[3 * (size_t)link_ml[q] + k] + d * u[k]);
  }
  return 0;
}

int orc_link_spread(int64_t n_atoms, int64_t n_links, const int32_t* link_ml, const int32_t* link_mm, double d,
                    const float* box, int32_t pbc, const float* pos, double* forces /* [n_atoms + n_links][3] */) {
  for (int64_t q = 0; q < n_links; ++q) {
    double u[3], l, uf = 0.0;
    link_bond(pos, box, pbc, link_ml[q], link_mm[q], u, &l);
    if (!(l > 0.0)) return -1;
    double* FL = forces + 3 * (size_t)(n_atoms + q);
    for (int k = 0; k < 3; ++k) uf += u[k] * FL[k];
    for (int k = 0; k < 3; ++k) {
      const double perp = (d / l) * (FL[k] - u[k] * uf);
      forces[3 * (size_t)link_ml[q] + k] += FL[k] - perp;
      forces[3 * (size_t)link_mm[q] + k] += perp;
    }
    for (int k = 0; k < 3; ++k) FL[k] = 0.0;
  }
  return 0;
}
