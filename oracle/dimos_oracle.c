/*
 * dimos_oracle.c -- CPU fp64 ORACLE for the DIMOS neighbour-list + short-range nonbonded hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header, table
 * or helper with the CUDA path under paper_2503_20541_b200/csrc/, and never will.
 *
 * What it is: the plain definition of what the method computes (the method reaches exactly the
 * plain result, faster -- SURVEY.md §8(c)), written out in fp64:
 *   - an O(N^2) brute-force minimum-image pair sum (orc_nonbonded_bruteforce,
 *     orc_neighbor_pairs_bruteforce), and
 *   - a SEPARATE naive cell list (cells of edge >= range, 27-stencil with periodic wrap,
 *     PAPER.md:177) that must reproduce the brute force (orc_nonbonded_celllist,
 *     orc_neighbor_pairs_celllist).
 * No blocking, no fusion, no reordering beyond the definition.  OpenMP only distributes the outer
 * loop over atoms i; every per-atom result is computed by one thread in a fixed order, so results
 * do not depend on the thread count.
 *
 * Passages followed (PAPER.md = /root/reference/PAPER.md, arXiv 2503.20541):
 *   Verlet list radius r_nl = r_c + r_g .................. PAPER.md:173  (§III A 2 a)
 *   rebuild criterion d > r_g/2 ........................... PAPER.md:175
 *   cell list, cells >= r_nl, neighbouring cells .......... PAPER.md:177
 *   Lennard-Jones 12-6, Eq. (4) ........................... PAPER.md:189-191
 *   Lorentz-Berthelot combining rules, Eq. (5) ............ PAPER.md:193-196
 *   LJ switching function S(x), Eq. (6) (optional, r_switch) PAPER.md:198-202
 *   Coulomb, Eq. (7) ...................................... PAPER.md:204-206
 *   reaction field, Eq. (8) with k_RFA, c_RFA ............. PAPER.md:208-213
 *   Ewald direct-space term, Eq. (10), n = 0 image only ... PAPER.md:215-223
 *   exclusions filtered at neighbour-list level ........... PAPER.md:243
 * Readings of silent/garbled points (restated in DESIGN.md):
 *   C-1  eps == eps_s == eps_rf in k_RFA, c_RFA (the only reading with U_RFA(r_c) = 0)
 *   C-3  component-wise nearest image, d_a <- d_a - L_a * nearbyint(d_a / L_a)
 *   C-4  strict r^2 < r_c^2 and r^2 < r_nl^2
 *   C-5  strict max |dr| > skin/2, raw (unwrapped) coordinate difference
 *   C-7  virial W_ab = sum_pairs d_a f_ij,b, d = r_i - r_j (min image), f_ij = force on i from j
 *   C-8  plain truncation of LJ at r_c (no switch)
 *   C-14 Ewald real space: nearest image only, unordered pairs once, multiplied by k_e
 *   C-15 exclusion correction -k_e q_i q_j erf(alpha r)/r over ALL excluded pairs (no cutoff);
 *        no self term, no reciprocal term
 *
 * Parity pins (tests/test_oracle_*.py, run with -m "not gpu"): two-particle closed forms, LJ
 * textbook points (U(sigma)=0, U(2^(1/6) sigma) = -eps, F = 0 there), U_RFA(r_c) = 0,
 * erfc + erf = 1 identity, forces = -finite-difference gradient of the energy, Newton III,
 * virial = -dE/dlambda under uniform scaling, translation / periodic-image invariance,
 * exclusion special cases, cell list == brute force, neighbour set == scipy cKDTree.
 * Nothing here is "parity unpinned" except absolute agreement with DIMOS/OpenMM themselves,
 * which the paper gives no numbers for.
 *
 * Units: nm, kJ/mol, e; forces kJ mol^-1 nm^-1.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_METHOD_RF 0
#define ORC_METHOD_EWALD_REAL 1

typedef struct {
    double r_cut;
    double eps_rf;
    double alpha;
    double coulomb_const; /* k_e = 1/(4 pi eps0) in kJ mol^-1 nm e^-2 */
    int32_t method;
    double r_switch;      /* LJ switching distance r_s of Eq. 6; <= 0 or >= r_cut: plain truncation */
} orc_params;

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Eq. (5): eps_ij = sqrt(eps_i eps_j), sigma_ij = (sigma_i + sigma_j)/2.
 * table[(a*ntypes+b)*2 + 0] = sigma_ab, [..+1] = eps_ab. */
void orc_lorentz_berthelot(const double* sigma, const double* eps, int32_t ntypes, double* table)
{
    for (int a = 0; a < ntypes; ++a)
        for (int b = 0; b < ntypes; ++b) {
            table[(a * ntypes + b) * 2 + 0] = 0.5 * (sigma[a] + sigma[b]);
            table[(a * ntypes + b) * 2 + 1] = sqrt(eps[a] * eps[b]);
        }
}

/* Reading C-3: component-wise nearest image. */
static double min_image(double d, double L) { return d - L * nearbyint(d / L); }

/* Reaction-field constants, Eq. (8) / PAPER.md:213 with reading C-1. */
static void rf_constants(const orc_params* p, double* k_rf, double* c_rf)
{
    double rc = p->r_cut;
    *k_rf = (p->eps_rf - 1.0) / ((2.0 * p->eps_rf + 1.0) * rc * rc * rc);
    *c_rf = 3.0 * p->eps_rf / ((2.0 * p->eps_rf + 1.0) * rc);
}

/* Energy and (force on i)/d for one non-excluded pair at squared distance r2 < r_c^2.
 *   LJ  (Eq. 4):  U = 4 eps [(s/r)^12 - (s/r)^6];      -dU/dr / r = 24 eps [2 (s/r)^12 - (s/r)^6] / r^2
 *   RF  (Eq. 8):  U = k_e qq (1/r + k_rf r^2 - c_rf);  -dU/dr / r = k_e qq (1/r^3 - 2 k_rf)
 *   Ewald real (Eq. 10, n=0): U = k_e qq erfc(a r)/r;
 *                 -dU/dr / r = k_e qq [erfc(a r)/r + (2a/sqrt(pi)) exp(-a^2 r^2)] / r^2
 * The force on i from j is  f_over_r * d  with d = r_i - r_j. */
static void pair_terms(double r2, double qq, double sigma, double eps, const orc_params* p,
                       double* e_lj, double* e_coul, double* f_over_r)
{
    double r = sqrt(r2);
    double sr = sigma / r;
    double sr2 = sr * sr;
    double sr6 = sr2 * sr2 * sr2;
    double sr12 = sr6 * sr6;
    double ke_qq = p->coulomb_const * qq;
    *e_lj = 4.0 * eps * (sr12 - sr6);
    double f = 24.0 * eps * (2.0 * sr12 - sr6) / r2;
    if (p->r_switch > 0.0 && p->r_switch < p->r_cut && r > p->r_switch) {
        /* Eq. 6: U_LJ -> S(x) U_LJ, x = (r - r_s)/(r_c - r_s), S = 1 - 6x^5 + 15x^4 - 10x^3;
         * -d(S U)/dr = S (-U') - S'(x) U / (r_c - r_s), S'(x) = -30x^4 + 60x^3 - 30x^2 */
        double w = p->r_cut - p->r_switch;
        double x = (r - p->r_switch) / w;
        double S = 1.0 - 6.0 * x * x * x * x * x + 15.0 * x * x * x * x - 10.0 * x * x * x;
        double dS = -30.0 * x * x * x * x + 60.0 * x * x * x - 30.0 * x * x;
        f = S * f - dS / w * (*e_lj) / r;
        *e_lj = S * (*e_lj);
    }
    if (p->method == ORC_METHOD_RF) {
        double k_rf, c_rf;
        rf_constants(p, &k_rf, &c_rf);
        *e_coul = ke_qq * (1.0 / r + k_rf * r2 - c_rf);
        f += ke_qq * (1.0 / (r2 * r) - 2.0 * k_rf);
    } else {
        double a = p->alpha;
        double two_a_sqrtpi = 2.0 * a / sqrt(M_PI);
        *e_coul = ke_qq * erfc(a * r) / r;
        f += ke_qq * (erfc(a * r) / r + two_a_sqrtpi * exp(-a * a * r2)) / r2;
    }
    *f_over_r = f;
}

/* Ewald exclusion correction for one excluded pair (reading C-15):
 *   U = -k_e qq erf(a r)/r;   -dU/dr / r = k_e qq [(2a/sqrt(pi)) exp(-a^2 r^2) - erf(a r)/r] / r^2 */
static void excl_correction_terms(double r2, double qq, const orc_params* p, double* e, double* f_over_r)
{
    double r = sqrt(r2);
    double a = p->alpha;
    double ke_qq = p->coulomb_const * qq;
    *e = -ke_qq * erf(a * r) / r;
    *f_over_r = ke_qq * (2.0 * a / sqrt(M_PI) * exp(-a * a * r2) - erf(a * r) / r) / r2;
}

/* ---- exclusion set as adjacency (CSR over both directions) ---------------------------------- */
typedef struct {
    int64_t* start; /* N+1 */
    int32_t* adj;   /* 2*n_excl */
} excl_csr;

static int excl_build(excl_csr* x, int64_t N, const int32_t* pairs, int64_t n_excl)
{
    x->start = (int64_t*)calloc((size_t)N + 1, sizeof(int64_t));
    x->adj = (int32_t*)malloc(sizeof(int32_t) * (size_t)(2 * n_excl > 0 ? 2 * n_excl : 1));
    if (!x->start || !x->adj) return -1;
    for (int64_t k = 0; k < n_excl; ++k) {
        x->start[pairs[2 * k] + 1]++;
        x->start[pairs[2 * k + 1] + 1]++;
    }
    for (int64_t i = 0; i < N; ++i) x->start[i + 1] += x->start[i];
    int64_t* fill = (int64_t*)malloc(sizeof(int64_t) * (size_t)(N > 0 ? N : 1));
    if (!fill) return -1;
    memcpy(fill, x->start, sizeof(int64_t) * (size_t)N);
    for (int64_t k = 0; k < n_excl; ++k) {
        int32_t a = pairs[2 * k], b = pairs[2 * k + 1];
        x->adj[fill[a]++] = b;
        x->adj[fill[b]++] = a;
    }
    free(fill);
    return 0;
}
static void excl_free(excl_csr* x) { free(x->start); free(x->adj); }
static int is_excluded(const excl_csr* x, int64_t i, int64_t j)
{
    for (int64_t k = x->start[i]; k < x->start[i + 1]; ++k)
        if (x->adj[k] == j) return 1;
    return 0;
}

/* ---- the naive cell list ------------------------------------------------------
 * n_a = max(1, floor(L_a / range)) cells per axis, so every cell edge >= range (reading C-18).
 * Atoms are wrapped into [0,L) only to find their cell; distances always use min_image on the
 * raw coordinates.  Linked list: head[cell], next[atom]. */
typedef struct {
    int n[3];
    int64_t ncell;
    int64_t* head;
    int64_t* next;
} cell_list;

static int cell_coord(double x, double L, int n)
{
    double f = x / L - floor(x / L); /* fractional coordinate in [0,1) */
    int c = (int)floor(f * n);
    if (c >= n) c = n - 1; /* f rounded up to 1.0 */
    if (c < 0) c = 0;
    return c;
}

static int cells_build(cell_list* cl, const double* pos, int64_t N, const double* box, double range)
{
    for (int a = 0; a < 3; ++a) {
        int n = (int)floor(box[a] / range);
        cl->n[a] = n < 1 ? 1 : n;
    }
    cl->ncell = (int64_t)cl->n[0] * cl->n[1] * cl->n[2];
    cl->head = (int64_t*)malloc(sizeof(int64_t) * (size_t)cl->ncell);
    cl->next = (int64_t*)malloc(sizeof(int64_t) * (size_t)(N > 0 ? N : 1));
    if (!cl->head || !cl->next) return -1;
    for (int64_t c = 0; c < cl->ncell; ++c) cl->head[c] = -1;
    for (int64_t i = N - 1; i >= 0; --i) { /* reverse so each list is in ascending atom order */
        int cx = cell_coord(pos[3 * i + 0], box[0], cl->n[0]);
        int cy = cell_coord(pos[3 * i + 1], box[1], cl->n[1]);
        int cz = cell_coord(pos[3 * i + 2], box[2], cl->n[2]);
        int64_t c = ((int64_t)cx * cl->n[1] + cy) * cl->n[2] + cz;
        cl->next[i] = cl->head[c];
        cl->head[c] = i;
    }
    return 0;
}
static void cells_free(cell_list* cl) { free(cl->head); free(cl->next); }

/* Unique neighbour cells of cell (cx,cy,cz): the 27-stencil with periodic wrap, de-duplicated
 * when an axis has fewer than 3 cells (reading C-18).  Returns the count, fills out[27]. */
static int neighbour_cells(const cell_list* cl, int cx, int cy, int cz, int64_t* out)
{
    int cnt = 0;
    for (int dx = -1; dx <= 1; ++dx)
        for (int dy = -1; dy <= 1; ++dy)
            for (int dz = -1; dz <= 1; ++dz) {
                int x = ((cx + dx) % cl->n[0] + cl->n[0]) % cl->n[0];
                int y = ((cy + dy) % cl->n[1] + cl->n[1]) % cl->n[1];
                int z = ((cz + dz) % cl->n[2] + cl->n[2]) % cl->n[2];
                int64_t c = ((int64_t)x * cl->n[1] + y) * cl->n[2] + z;
                int dup = 0;
                for (int k = 0; k < cnt; ++k)
                    if (out[k] == c) dup = 1;
                if (!dup) out[cnt++] = c;
            }
    return cnt;
}

/* ---- per-atom work shared by both enumerations: add pair (i,j) to atom i's sums ---------------
 * Called for every ordered pair (i, j != i) that the enumeration proposes; it applies the
 * exclusion filter, the minimum image (C-3) and the strict cutoff (C-4) itself.
 * Forces: F_i = sum_{j != i} f_ij.  Energies/virial/pair count are taken from the j > i half so
 * each unordered pair counts once.  allow_i accumulates |f_ij| for pairs inside the cutoff band
 * |r - r_c| < band (reading C-10), evaluated with the in-cutoff expression. */
typedef struct {
    double f[3];
    double e_lj, e_coul;
    double w[9];
    double allow;
    int64_t npairs;
} atom_acc;

static void visit_pair(int64_t i, int64_t j, const double* pos, const double* charge, const int32_t* type,
                       const double* lj_table, int32_t ntypes, const double* box, const orc_params* p,
                       const excl_csr* x, double band, atom_acc* acc)
{
    if (is_excluded(x, i, j)) return;
    double d[3];
    for (int a = 0; a < 3; ++a) d[a] = min_image(pos[3 * i + a] - pos[3 * j + a], box[a]);
    double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    double rc = p->r_cut;
    int in_cut = r2 < rc * rc;
    int in_band = 0;
    if (band > 0.0) {
        double r = sqrt(r2);
        in_band = fabs(r - rc) < band;
    }
    if (!in_cut && !in_band) return;
    const double* sp = &lj_table[((int64_t)type[i] * ntypes + type[j]) * 2];
    double e_lj, e_coul, f_over_r;
    pair_terms(r2, charge[i] * charge[j], sp[0], sp[1], p, &e_lj, &e_coul, &f_over_r);
    if (in_band) acc->allow += fabs(f_over_r) * sqrt(r2);
    if (!in_cut) return;
    for (int a = 0; a < 3; ++a) acc->f[a] += f_over_r * d[a];
    if (j > i) {
        acc->e_lj += e_lj;
        acc->e_coul += e_coul;
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) acc->w[3 * a + b] += d[a] * (f_over_r * d[b]);
        acc->npairs++;
    }
}

/* Sum per-atom accumulators in atom order (fixed order => thread-count independent). */
static void finish(int64_t N, const atom_acc* acc, double* F, double* E, double* W, double* allow,
                   int64_t* npairs)
{
    double e_lj = 0, e_coul = 0, w[9] = {0};
    int64_t np = 0;
    for (int64_t i = 0; i < N; ++i) {
        for (int a = 0; a < 3; ++a) F[3 * i + a] = acc[i].f[a];
        e_lj += acc[i].e_lj;
        e_coul += acc[i].e_coul;
        for (int k = 0; k < 9; ++k) w[k] += acc[i].w[k];
        np += acc[i].npairs;
        if (allow) allow[i] = acc[i].allow;
    }
    E[1] = e_lj;
    E[2] = e_coul;
    for (int k = 0; k < 9; ++k) W[k] = w[k];
    *npairs = np;
}

/* Ewald exclusion correction over the excluded-pair list (reading C-15); adds into F, W, E[3]. */
static void add_exclusion_correction(int64_t N, const double* pos, const double* charge, const double* box,
                                     const orc_params* p, const int32_t* excl_pairs, int64_t n_excl,
                                     double* F, double* E, double* W)
{
    (void)N;
    double e_sum = 0;
    for (int64_t k = 0; k < n_excl; ++k) {
        int64_t i = excl_pairs[2 * k], j = excl_pairs[2 * k + 1];
        double d[3];
        for (int a = 0; a < 3; ++a) d[a] = min_image(pos[3 * i + a] - pos[3 * j + a], box[a]);
        double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
        double e, f_over_r;
        excl_correction_terms(r2, charge[i] * charge[j], p, &e, &f_over_r);
        e_sum += e;
        for (int a = 0; a < 3; ++a) {
            F[3 * i + a] += f_over_r * d[a];
            F[3 * j + a] -= f_over_r * d[a];
            for (int b = 0; b < 3; ++b) W[3 * a + b] += d[a] * (f_over_r * d[b]);
        }
    }
    E[3] = e_sum;
}

/* 1-4 exceptions ("scale the strength of the non-bonded interactions by some common factor", or an
 * individual factor per pair; "handled explicitly by the non-bonded interaction method").  Reading C-21 (the paper
 * gives no formula): every exception pair is also an excluded pair, so the sums above skip it; it contributes
 *   U = s_lj * 4 eps [(s/r)^12 - (s/r)^6]  (Eq. 4)  +  s_c * k_e q_i q_j / r  (Eq. 7)
 * at its minimum-image distance, without cutoff, switch, reaction field or Ewald modification.
 *   exc_pairs n_exc x 2 (i<j), exc_scale n_exc x 2 = (s_c, s_lj).  Adds into F, W, E[0], E[1] (LJ), E[2] (Coulomb). */
int orc_add_exceptions(int64_t N, const double* pos, const double* charge, const int32_t* type, const double* lj_table,
                       int32_t ntypes, const double* box, double coulomb_const, const int32_t* exc_pairs,
                       const double* exc_scale, int64_t n_exc, double* F, double* E, double* W)
{
    (void)N;
    for (int64_t k = 0; k < n_exc; ++k) {
        int64_t i = exc_pairs[2 * k], j = exc_pairs[2 * k + 1];
        double d[3];
        for (int a = 0; a < 3; ++a) d[a] = min_image(pos[3 * i + a] - pos[3 * j + a], box[a]);
        double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
        double r = sqrt(r2);
        const double* sp = &lj_table[((int64_t)type[i] * ntypes + type[j]) * 2];
        double sr = sp[0] / r, sr2 = sr * sr, sr6 = sr2 * sr2 * sr2, sr12 = sr6 * sr6;
        double s_c = exc_scale[2 * k], s_lj = exc_scale[2 * k + 1];
        double e_lj = s_lj * 4.0 * sp[1] * (sr12 - sr6);
        double e_c = s_c * coulomb_const * charge[i] * charge[j] / r;
        double f_over_r = s_lj * 24.0 * sp[1] * (2.0 * sr12 - sr6) / r2 + e_c / r2;
        E[1] += e_lj;
        E[2] += e_c;
        E[0] += e_lj + e_c;
        for (int a = 0; a < 3; ++a) {
            F[3 * i + a] += f_over_r * d[a];
            F[3 * j + a] -= f_over_r * d[a];
            for (int b = 0; b < 3; ++b) W[3 * a + b] += d[a] * (f_over_r * d[b]);
        }
    }
    return 0;
}

/* O(N^2) brute force: THE definition.
 *   pos N x 3, charge N, type N, lj_table ntypes x ntypes x 2 = (sigma_ab, eps_ab), box[3],
 *   excl_pairs n_excl x 2 (i<j, unique).
 * Outputs: F N x 3; E[4] = {total, lj, coul_pair, coul_excl_corr}; W[9] row-major;
 *   allow (N, may be NULL) per-atom cutoff-band allowance with half-width `band` (C-10);
 *   *npairs = number of unordered in-cutoff pairs.  Returns 0, or -1 on allocation failure. */
int orc_nonbonded_bruteforce(int64_t N, const double* pos, const double* charge, const int32_t* type,
                             const double* lj_table, int32_t ntypes, const double* box, const orc_params* p,
                             const int32_t* excl_pairs, int64_t n_excl, double band,
                             double* F, double* E, double* W, double* allow, int64_t* npairs)
{
    excl_csr x;
    if (excl_build(&x, N, excl_pairs, n_excl)) return -1;
    atom_acc* acc = (atom_acc*)calloc((size_t)(N > 0 ? N : 1), sizeof(atom_acc));
    if (!acc) return -1;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < N; ++i)
        for (int64_t j = 0; j < N; ++j)
            if (j != i) visit_pair(i, j, pos, charge, type, lj_table, ntypes, box, p, &x, band, &acc[i]);
    finish(N, acc, F, E, W, allow, npairs);
    E[3] = 0.0;
    if (p->method == ORC_METHOD_EWALD_REAL)
        add_exclusion_correction(N, pos, charge, box, p, excl_pairs, n_excl, F, E, W);
    E[0] = E[1] + E[2] + E[3];
    free(acc);
    excl_free(&x);
    return 0;
}

/* The same sums, enumerated through the naive cell list with cells of edge >= r_cut. */
int orc_nonbonded_celllist(int64_t N, const double* pos, const double* charge, const int32_t* type,
                           const double* lj_table, int32_t ntypes, const double* box, const orc_params* p,
                           const int32_t* excl_pairs, int64_t n_excl, double band,
                           double* F, double* E, double* W, double* allow, int64_t* npairs)
{
    excl_csr x;
    cell_list cl;
    if (excl_build(&x, N, excl_pairs, n_excl)) return -1;
    if (cells_build(&cl, pos, N, box, p->r_cut + (band > 0 ? band : 0))) return -1;
    atom_acc* acc = (atom_acc*)calloc((size_t)(N > 0 ? N : 1), sizeof(atom_acc));
    if (!acc) return -1;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < N; ++i) {
        int cx = cell_coord(pos[3 * i + 0], box[0], cl.n[0]);
        int cy = cell_coord(pos[3 * i + 1], box[1], cl.n[1]);
        int cz = cell_coord(pos[3 * i + 2], box[2], cl.n[2]);
        int64_t nb[27];
        int nnb = neighbour_cells(&cl, cx, cy, cz, nb);
        for (int k = 0; k < nnb; ++k)
            for (int64_t j = cl.head[nb[k]]; j >= 0; j = cl.next[j])
                if (j != i) visit_pair(i, j, pos, charge, type, lj_table, ntypes, box, p, &x, band, &acc[i]);
    }
    finish(N, acc, F, E, W, allow, npairs);
    E[3] = 0.0;
    if (p->method == ORC_METHOD_EWALD_REAL)
        add_exclusion_correction(N, pos, charge, box, p, excl_pairs, n_excl, F, E, W);
    E[0] = E[1] + E[2] + E[3];
    free(acc);
    cells_free(&cl);
    excl_free(&x);
    return 0;
}

/* ---- neighbour pair set P(r_list) = { i<j : (i,j) not excluded, min-image r^2 < r_list^2 } ----
 * (PAPER.md:173, 243).  Two passes: count per i, prefix, fill; rows are in ascending j, so the
 * output is lexicographically sorted.  Call with pairs == NULL to get the count only.
 * Returns the number of pairs, or -1 on allocation failure, or -2 if cap is too small. */
static int in_list(int64_t i, int64_t j, const double* pos, const double* box, double r_list, const excl_csr* x)
{
    if (is_excluded(x, i, j)) return 0;
    double r2 = 0;
    for (int a = 0; a < 3; ++a) {
        double d = min_image(pos[3 * i + a] - pos[3 * j + a], box[a]);
        r2 += d * d;
    }
    return r2 < r_list * r_list;
}

int64_t orc_neighbor_pairs_bruteforce(int64_t N, const double* pos, const double* box, double r_list,
                                      const int32_t* excl_pairs, int64_t n_excl, int32_t* pairs, int64_t cap)
{
    excl_csr x;
    if (excl_build(&x, N, excl_pairs, n_excl)) return -1;
    int64_t* row = (int64_t*)calloc((size_t)N + 1, sizeof(int64_t));
    if (!row) return -1;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < N; ++i) {
        int64_t c = 0;
        for (int64_t j = i + 1; j < N; ++j) c += in_list(i, j, pos, box, r_list, &x);
        row[i + 1] = c;
    }
    for (int64_t i = 0; i < N; ++i) row[i + 1] += row[i];
    int64_t total = row[N];
    if (pairs) {
        if (total > cap) { free(row); excl_free(&x); return -2; }
#pragma omp parallel for schedule(dynamic, 16)
        for (int64_t i = 0; i < N; ++i) {
            int64_t k = row[i];
            for (int64_t j = i + 1; j < N; ++j)
                if (in_list(i, j, pos, box, r_list, &x)) {
                    pairs[2 * k] = (int32_t)i;
                    pairs[2 * k + 1] = (int32_t)j;
                    ++k;
                }
        }
    }
    free(row);
    excl_free(&x);
    return total;
}

static int cmp_i64(const void* a, const void* b)
{
    int64_t x = *(const int64_t*)a, y = *(const int64_t*)b;
    return (x > y) - (x < y);
}

/* Collect the j > i neighbours of atom i through the cell list, sorted ascending, into buf. */
static int64_t cell_row(const cell_list* cl, int64_t i, const double* pos, const double* box, double r_list,
                        const excl_csr* x, int64_t* buf, int64_t bufcap)
{
    int cx = cell_coord(pos[3 * i + 0], box[0], cl->n[0]);
    int cy = cell_coord(pos[3 * i + 1], box[1], cl->n[1]);
    int cz = cell_coord(pos[3 * i + 2], box[2], cl->n[2]);
    int64_t nb[27];
    int nnb = neighbour_cells(cl, cx, cy, cz, nb);
    int64_t c = 0;
    for (int k = 0; k < nnb; ++k)
        for (int64_t j = cl->head[nb[k]]; j >= 0; j = cl->next[j])
            if (j > i && in_list(i, j, pos, box, r_list, x)) {
                if (buf && c < bufcap) buf[c] = j;
                ++c;
            }
    if (buf) qsort(buf, (size_t)(c < bufcap ? c : bufcap), sizeof(int64_t), cmp_i64);
    return c;
}

int64_t orc_neighbor_pairs_celllist(int64_t N, const double* pos, const double* box, double r_list,
                                    const int32_t* excl_pairs, int64_t n_excl, int32_t* pairs, int64_t cap)
{
    excl_csr x;
    cell_list cl;
    if (excl_build(&x, N, excl_pairs, n_excl)) return -1;
    if (cells_build(&cl, pos, N, box, r_list)) return -1;
    int64_t* row = (int64_t*)calloc((size_t)N + 1, sizeof(int64_t));
    if (!row) return -1;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < N; ++i) row[i + 1] = cell_row(&cl, i, pos, box, r_list, &x, NULL, 0);
    for (int64_t i = 0; i < N; ++i) row[i + 1] += row[i];
    int64_t total = row[N];
    int fail = 0;
    if (pairs) {
        if (total > cap) { free(row); cells_free(&cl); excl_free(&x); return -2; }
#pragma omp parallel for schedule(dynamic, 16)
        for (int64_t i = 0; i < N; ++i) {
            int64_t n = row[i + 1] - row[i];
            if (n == 0) continue;
            int64_t* buf = (int64_t*)malloc(sizeof(int64_t) * (size_t)n);
            if (!buf) { fail = 1; continue; }
            cell_row(&cl, i, pos, box, r_list, &x, buf, n);
            for (int64_t k = 0; k < n; ++k) {
                pairs[2 * (row[i] + k)] = (int32_t)i;
                pairs[2 * (row[i] + k) + 1] = (int32_t)buf[k];
            }
            free(buf);
        }
    }
    free(row);
    cells_free(&cl);
    excl_free(&x);
    return fail ? -1 : total;
}

/* Rebuild trigger, PAPER.md:175 with reading C-5: flag = [ max_i |pos_i - pos_at_build_i| > skin/2 ],
 * raw coordinates, strict.  *max_disp (may be NULL) receives the maximum displacement. */
int orc_needs_rebuild(int64_t N, const double* pos, const double* pos_at_build, double skin, double* max_disp)
{
    double m2 = 0;
    for (int64_t i = 0; i < N; ++i) {
        double s = 0;
        for (int a = 0; a < 3; ++a) {
            double d = pos[3 * i + a] - pos_at_build[3 * i + a];
            s += d * d;
        }
        if (s > m2) m2 = s;
    }
    if (max_disp) *max_disp = sqrt(m2);
    return m2 > (0.5 * skin) * (0.5 * skin);
}
