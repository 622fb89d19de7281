/*
 * dimos.h -- C ABI of libdimos_b200: the per-step hot path of the DIMOS method (arXiv 2503.20541)
 * as hand-written CUDA for sm_100a (NVIDIA B200).
 *
 * What the library computes (PAPER.md = /root/reference/PAPER.md, section III A 2):
 *   - the Verlet neighbour list of radius r_nl = r_c + r_g built in O(N) from a cell list
 *     (PAPER.md:173-177), with excluded pairs filtered at list level;
 *   - the rebuild trigger "any atom moved more than r_g/2 since construction";
 *   - the short-range nonbonded pair sum over that list: Lennard-Jones 12-6 (Eq. 4)
 *     plus reaction-field electrostatics (Eq. 8) or the Ewald direct-space term
 *     erfc(alpha r)/r (Eq. 10) with its intramolecular exclusion correction,
 *     under the minimum-image convention, returning per-atom forces, energy
 *     components and the virial.
 * Readings of points the paper leaves open are listed in DESIGN.md (C-1 ... C-20).
 *
 * Conventions
 *   Units: nm, ps, amu, e, kJ/mol; forces kJ mol^-1 nm^-1.
 *   "dev" pointers are CUDA device pointers on the context's device, "host" pointers are host
 *   memory.  All arrays are contiguous, row-major.  The element type of pos / charge / F is
 *   `float` for DIMOS_F32 and DIMOS_MIXED contexts and `double` for DIMOS_F64 contexts.
 *   The caller owns every array it passes in; the library owns only its opaque handles and the
 *   workspace they hold (obtained through the dimos_allocator callbacks when given, so that the
 *   caller's framework -- torch's caching allocator in the Python binding -- owns device memory).
 *   All device work is enqueued on the `stream` argument (a cudaStream_t passed as void*; NULL is
 *   the legacy default stream).  A call does not synchronise with the host unless stated.
 *   Every call returns a dimos_status (0 = DIMOS_OK, negative = error); on error no output array
 *   is guaranteed to be written.  dimos_last_error(ctx) gives a human-readable message.
 *   Host calls on one context must not overlap in time (no internal locking).  Their device work may: calls may use
 *   different streams and several lists, and up to 64 rebuild-trigger evaluations (dimos_nl_needs_rebuild and the
 *   integrator steps that fuse it) may be in flight at once, each with its own reduction state.
 *   Every call that touches the device makes the context's device the calling thread's current CUDA device
 *   (cudaSetDevice) and leaves it current on return; `stream` must belong to that device.
 *   CUDA graphs: dimos_nl_needs_rebuild_static, dimos_nl_needs_rebuild with flag_host = NULL, the integrator calls
 *   without a host flag, dimos_pme_recip (once a call with the same mesh, order, alpha and box has made its plans), and
 *   dimos_nonbonded (once an ordinary call on the same list has created its per-step workspace)
 *   enqueue only kernels and memsets, allocate nothing and do not synchronise: they may be recorded by a stream capture
 *   and replayed.  The recorded arguments include the list's buffers and sizes, so capture again after every
 *   dimos_nl_build; dimos_nb_params.skip_flag lets the recorded force kernels return at once on the step that needs one.
 *   A recorded trigger keeps the reduction-state slot (one of the 64) it was recorded with: replay it on one stream, and
 *   do not run other trigger calls of the same context on another stream at the same time.
 *   There is no CPU fallback: without a usable CUDA device every compute call fails with
 *   DIMOS_ECUDA.
 */
#ifndef DIMOS_H_
#define DIMOS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define DIMOS_API __attribute__((visibility("default")))
#else
#define DIMOS_API
#endif

typedef struct dimos_ctx dimos_ctx; /* opaque, library-owned */
typedef struct dimos_nl dimos_nl;   /* opaque neighbour list, library-owned, tied to its ctx */

typedef enum {
    DIMOS_OK = 0,
    DIMOS_EINVAL = -1,    /* bad argument (NULL pointer, N <= 0, non-finite box, unsupported value) */
    DIMOS_EBOX = -2,      /* r_cut > min(box)/2: more than one image inside the cutoff (reading C-3) */
    DIMOS_ENOMEM = -3,    /* host or device allocation failed */
    DIMOS_EOVERFLOW = -4, /* an internal capacity was exceeded even after growing (see message) */
    DIMOS_ECUDA = -5,     /* CUDA runtime error, or no CUDA device */
    DIMOS_ESTALE = -6     /* N, box or r_cut differ from the values the list was built with */
} dimos_status;

/* Element type of pos/charge/F and arithmetic of the pair kernel (reading C-11):
 *   DIMOS_F32   float in/out, float pair math, per-thread float partial sums, fp64 final reduction.
 *               Exception: boxes with fewer than three cells per axis (N of a few thousand at most; the per-pair
 *               minimum-image kernel) evaluate the pair ENERGY in fp64 from the same fp32 inputs, because their
 *               total is a ~1e-4 remainder of cancelling terms that fp32 pair energies cannot resolve to 1e-5
 *               (DESIGN.md section 3); forces and virial stay fp32.  Larger boxes are fp32 throughout.
 *   DIMOS_F64   double everywhere
 *   DIMOS_MIXED float in/out, float pair math, energy and virial accumulated in fp64 from the
 *               first add */
typedef enum { DIMOS_F32 = 0, DIMOS_F64 = 1, DIMOS_MIXED = 2 } dimos_precision;

/* Electrostatics of the pair sum: reaction field (Eq. 8) or Ewald direct space (Eq. 10, nearest
 * image only, reading C-14) plus the exclusion correction (reading C-15). */
typedef enum { DIMOS_RF = 0, DIMOS_EWALD_REAL = 1 } dimos_method;

/* Device-memory callbacks.  alloc returns a device pointer aligned to >= 256 bytes, or NULL;
 * free_ releases a pointer returned by alloc.  Both are called from the thread that calls the
 * library, only from dimos_nl_build / dimos_create / dimos_destroy / dimos_nl_destroy, never
 * while a kernel of this library that uses the block is pending on a stream other than the
 * one given to alloc.  Pass NULL instead of a dimos_allocator to use cudaMalloc/cudaFree. */
typedef struct {
    void* (*alloc)(size_t bytes, void* stream, void* user);
    void (*free_)(void* ptr, void* user);
    void* user;
} dimos_allocator;

typedef struct {
    double r_cut;         /* r_c, nm; must equal the r_cut the list was built with */
    double eps_rf;        /* reaction-field dielectric (DIMOS_RF); reading C-1 */
    double alpha;         /* Ewald splitting parameter, nm^-1 (DIMOS_EWALD_REAL) */
    double coulomb_const; /* k_e = 1/(4 pi eps0), kJ mol^-1 nm e^-2 (138.935456, reading C-2) */
    int32_t method;       /* dimos_method */
    double r_switch;      /* LJ switching distance r_s of Eq. 6: for r_s < r < r_c the LJ term is
                           * multiplied by S(x) = 1 - 6x^5 + 15x^4 - 10x^3, x = (r - r_s)/(r_c - r_s); Coulomb terms are
                           * not switched.  <= 0 or >= r_cut: plain truncation at r_cut (reading C-8).  NaN: EINVAL */
    const int32_t* skip_flag; /* NULL, or a DEVICE word (e.g. the flag_dev of dimos_nl_needs_rebuild): if it is
                           * non-zero when the kernels of dimos_nonbonded run, they do nothing -- F, E and virial keep their
                           * old contents -- so that the force call can be enqueued behind the trigger without waiting for the
                           * host to read the flag; a caller that then finds the flag set rebuilds the list and calls again
                           * with skip_flag = NULL.  Must be NULL for the *_host entry points (DIMOS_EINVAL otherwise). */
} dimos_nb_params;

typedef struct {
    int64_t n_atoms;
    int64_t n_units;         /* i-clusters of DIMOS_UNIT atoms (incl. one partial unit per cell) */
    int64_t n_slots;         /* n_units * DIMOS_UNIT (sorted atom slots incl. padding) */
    int64_t n_entries;       /* (unit, j-atom) list entries, excluding chunk padding */
    int64_t n_entries_padded;/* entries incl. padding to 32-wide chunks (what the kernel streams) */
    int64_t n_pair_slots;    /* n_entries_padded * DIMOS_UNIT pair evaluations per force call */
    int64_t list_bytes;      /* bytes of list data streamed per force call */
    int64_t workspace_bytes; /* device bytes held by the list */
    int32_t n_cells[3];
    int32_t pbc_mode;        /* 0 = image shift from cell offsets, 1 = per-pair minimum image */
    int32_t row_capacity;    /* entries per unit row */
    int32_t n_rebuild_grow;  /* times the build was repeated with a larger capacity */
} dimos_nl_stats_t;

#define DIMOS_UNIT 8 /* atoms per i-cluster ("unit") of the cluster-pair list */

/* Create a context bound to CUDA device `device` with the given precision.
 * allocator may be NULL.  *out receives the handle. */
DIMOS_API int dimos_create(dimos_ctx** out, int device, int precision, const dimos_allocator* allocator);

/* Destroy a context and every list built with it (the caller must have synchronised the streams
 * that used it). */
DIMOS_API int dimos_destroy(dimos_ctx* ctx);

/* dimos_nl_build -- PAPER.md:173-177, 243.
 * Bins the N atoms into cells of edge >= r_cut + skin by counting sort (periodic wrap, positions
 * need not lie inside [0,L)), forms compact units of DIMOS_UNIT atoms inside each cell, and builds
 * for every unit the list of j-atoms that have at least one atom of the unit within
 * r_nl = r_cut + skin (strict <, reading C-4), each unordered atom pair being owned by exactly
 * one unit, with a per-entry bitmask that removes excluded pairs, the i >= j half of
 * intra-unit pairs and padding atoms.
 *   pos           dev, N x 3, float or double per the context precision; read
 *   N             number of atoms, 1 .. 2^31-1
 *   box           host, 3 doubles: orthorhombic box edges in nm
 *   r_cut, skin   nm; r_cut > 0, skin >= 0, r_cut <= min(box)/2 else DIMOS_EBOX
 *   excl_pairs    dev, n_excl x 2 int32, each row (i, j) with i < j, rows unique (reading C-17);
 *                 may be NULL when n_excl == 0.  At most 32 exclusion partners per atom.  Rows out of range, with i >= j,
 *                 or listed twice, and atoms with more partners, are reported as DIMOS_EINVAL.
 *   pos_at_build  dev, N x 3, same type as pos, caller-owned; written with a copy of pos (the
 *                 reference positions of the rebuild trigger)
 *   stream        cudaStream_t
 *   inout         *inout == NULL: a new list is created and returned; otherwise the given list
 *                 (built with the same ctx) is rebuilt in place, reusing its workspace.
 * Synchronises the stream once (to read the list size / overflow flag), and again per capacity
 * growth.  Also retains a device copy of excl_pairs for the Ewald exclusion correction. */
DIMOS_API int dimos_nl_build(dimos_ctx* ctx, const void* pos, int64_t N, const double* box, double r_cut,
                             double skin, const int32_t* excl_pairs, int64_t n_excl, void* pos_at_build,
                             void* stream, dimos_nl** inout);

/* Free one list (optional; dimos_destroy frees all lists of a context). */
DIMOS_API int dimos_nl_destroy(dimos_ctx* ctx, dimos_nl* nl);

/* dimos_nl_needs_rebuild -- PAPER.md:175, reading C-5.
 * flag = [ max_i |pos_i - pos_at_build_i| > skin/2 ], Euclidean norm of the raw (unwrapped)
 * coordinate difference, strict >, compared as squares in the context's element type.
 *   pos, pos_at_build  dev, N x 3
 *   flag_dev           dev, one int32, written with 0 or 1 (required)
 *   flag_host          host, one int32; if non-NULL the stream is synchronised and the flag copied
 *                      there, if NULL the call does not synchronise. */
DIMOS_API int dimos_nl_needs_rebuild(dimos_ctx* ctx, const void* pos, const void* pos_at_build, int64_t N,
                                     double skin, int32_t* flag_dev, int32_t* flag_host, void* stream);

/* dimos_nl_needs_rebuild_static -- the same trigger (reading C-5) for callers that must not allocate: code
 * under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The call allocates nothing (no
 * cudaMalloc / cudaFree, no dimos_allocator callback, no allocating library routine) and does not synchronise: its whole
 * scratch -- one block maximum per 1024 atoms and a ticket -- is a fixed __device__ array of 64.25 KiB inside the library,
 * held by every GPU that loads the library until the process exits.  The first call on a device looks the array's device
 * address up (cudaGetSymbolAddress; make one call outside any capture).
 *   pos, pos_at_build  dev, N x 3, element type of the context
 *   N                  1 .. DIMOS_STATIC_MAX_ATOMS; beyond it the call returns DIMOS_EOVERFLOW and launches nothing
 *   flag_dev           dev, one int32, written with 0 or 1 (required): the flag dimos_nl_needs_rebuild writes
 *   max_disp2_dev      dev, one double, may be NULL: receives max_i |pos_i - pos_at_build_i|^2 as computed in the context's
 *                      element type (+inf if a coordinate is NaN)
 * Enqueues one memset of the ticket and one kernel on `stream`.  ALL calls of a process on one GPU share the array, which
 * keeps the last call's contents: two calls that overlap on the GPU (different streams, or different contexts on the same
 * device) race and may both write wrong flags -- order them on one stream or with events. */
#define DIMOS_STATIC_MAX_ATOMS 8388608 /* 8192 blocks x 1024 atoms */
DIMOS_API int dimos_nl_needs_rebuild_static(dimos_ctx* ctx, const void* pos, const void* pos_at_build, int64_t N,
                                            double skin, int32_t* flag_dev, double* max_disp2_dev, void* stream);

/* dimos_nonbonded -- PAPER.md:189-213, 222, 243; SURVEY/DESIGN reading C-7 for the virial.
 * Evaluates, over the pairs of the list that are not excluded and have minimum-image r < r_cut
 * (strict, fp32 r^2 in F32/MIXED contexts), the Lennard-Jones energy (Eq. 4) and the Coulomb
 * energy by the chosen method, and their forces.  The list must be valid for `pos` (no atom moved
 * more than skin/2 since dimos_nl_build), which the caller checks with dimos_nl_needs_rebuild.
 *   pos      dev, N x 3
 *   charge   dev, N (e)
 *   type     dev, N int32 in [0, ntypes); an index outside that range is evaluated as type 0 and reported as DIMOS_EINVAL by
 *            the next call on this list that synchronises (dimos_nonbonded_host, dimos_step_host)
 *   lj_table dev, ntypes x ntypes x 2 doubles = (sigma_ab, eps_ab), symmetric (Eq. 5 filled by the
 *            caller, reading C-16); ntypes <= 64
 *   box      host, 3 doubles, must equal the build box (else DIMOS_ESTALE)
 *   params   host
 *   F        dev, N x 3, overwritten: F_i = sum_j f_ij (plus the exclusion-correction forces)
 *   E        dev, 4 doubles, overwritten: {total, lj, coul_pair, coul_excl_corr}; the 1-4 exceptions set with
 *            dimos_nl_set_exceptions add their LJ part to lj and their Coulomb part to coul_pair
 *   virial   dev, 9 doubles row-major, overwritten: W_ab = sum_pairs d_a f_ij,b with
 *            d = r_i - r_j (minimum image), including exclusion-correction pairs; may be NULL
 * Does not synchronise. */
DIMOS_API int dimos_nonbonded(dimos_ctx* ctx, const dimos_nl* nl, const void* pos, const void* charge,
                              const int32_t* type, const double* lj_table, int32_t ntypes, const double* box,
                              const dimos_nb_params* params, void* F, double* E, double* virial, void* stream);

/* dimos_nonbonded_host -- the same call with HOST arrays (pinned memory recommended): copies
 * pos/charge/type/lj_table to the device, runs dimos_nonbonded, copies F, E[4] and virial[9]
 * back and synchronises the stream before returning.  Staging buffers live in the list. */
DIMOS_API int dimos_nonbonded_host(dimos_ctx* ctx, dimos_nl* nl, const void* pos_host, const void* charge_host,
                                   const int32_t* type_host, const double* lj_table_host, int32_t ntypes,
                                   const double* box, const dimos_nb_params* params, void* F_host,
                                   double* E_host, double* virial_host, void* stream);

/* dimos_step_host -- one whole pass of the hot path for a caller whose arrays live in HOST memory
 * (pinned recommended): uploads pos (and charge/type/lj_table), evaluates the rebuild trigger
 * against the reference positions kept inside the list, rebuilds the list in place
 * when it fired, runs dimos_nonbonded and copies F, E[4] and virial[9] back.
 *   inout         *inout == NULL (or a list whose N / box / r_cut / skin / n_excl differ): the list is
 *                 built from pos_host and returned; otherwise reused / rebuilt in place
 *   excl_pairs_host  host, n_excl x 2 int32 (read only when the list is first built; the list keeps
 *                 its device copy for later rebuilds)
 *   charge_host, type_host, lj_table_host   each may be NULL once a call on this list has passed it: the device copy
 *                 kept in the list is used again, so that only what changed travels (positions travel every step)
 *   rebuilt_host  host, may be NULL: receives 1 if this call (re)built the list, else 0
 * Other arguments as in dimos_nonbonded_host.  Synchronises with the host: on a step that keeps the list the force
 * kernels are enqueued behind the trigger, conditional on its device flag, the host waits for the flag alone while they
 * run, then for the results; otherwise once to read the trigger, inside the rebuild, and once at the end. */
DIMOS_API int dimos_step_host(dimos_ctx* ctx, dimos_nl** inout, const void* pos_host, const void* charge_host,
                              const int32_t* type_host, const double* lj_table_host, int32_t ntypes, int64_t N,
                              const double* box, double skin, const int32_t* excl_pairs_host, int64_t n_excl,
                              const dimos_nb_params* params, void* F_host, double* E_host, double* virial_host,
                              int32_t* rebuilt_host, void* stream);

/* dimos_nl_export_pairs -- the neighbour set the list represents, for parity checks and for
 * consumers that want a plain edge list.
 * Writes every unordered pair (i < j, original atom indices) that is not excluded and has
 * minimum-image r < r_cut + skin at the build positions, in unspecified order (reading C-6).
 *   pairs         dev, cap x 2 int32; may be NULL when cap == 0 (count only)
 *   n_pairs_host  host, receives the number of pairs in the list; if it exceeds cap only the first
 *                 cap pairs found were written and the call returns DIMOS_EOVERFLOW.
 * Synchronises the stream. */
DIMOS_API int dimos_nl_export_pairs(dimos_ctx* ctx, const dimos_nl* nl, int32_t* pairs, int64_t cap,
                                    int64_t* n_pairs_host, void* stream);

/* dimos_pme_recip -- reciprocal-space electrostatics by smooth particle-mesh Ewald ("we implement smooth
 * PME ... B-splines based on the recursive definition") and the self energy, i.e. the two terms of Eq. 9
 * that dimos_nonbonded with DIMOS_EWALD_REAL does not return:
 *   U_recip = k_e / (2 pi V) sum_{k != 0} exp(-(pi k / alpha)^2) / k^2 |sum_j q_j exp(2 pi i k . r_j)|^2
 *             (Eq. 11, with the charges and the imaginary unit the printed formula lost: reading C-25),
 *             approximated on a K1 x K2 x K3 mesh with cardinal B-splines of the given order (Essmann et al. 1995);
 *   U_self  = -k_e alpha / sqrt(pi) sum_i q_i^2   (Eq. 12).
 * Steps: charge spreading (hand-written kernel), 3-D real-to-complex FFT (cuFFT), influence function B(m) C(m) with energy
 * and virial (hand-written), inverse FFT (cuFFT), force interpolation (hand-written).
 *   pos, charge  dev, N x 3 and N (element type of the context; positions need not be wrapped)
 *   box          host, 3 doubles;   alpha  Ewald splitting parameter (nm^-1), the one given to dimos_nonbonded
 *   mesh         host, 3 int32: mesh points per axis, each in [2 * order, 4096] with prime factors 2, 3, 5, 7
 *                (dimos_pme_mesh_size gives the paper's heuristic);   order  spline order n, 3..6 (OpenMM's 5)
 *   F            dev, N x 3 or NULL (energy only): reciprocal forces, ADDED to F when accumulate != 0, else overwriting
 *   E            dev, 2 doubles, overwritten: {U_recip, U_self};   virial  dev, 9 doubles or NULL: the reciprocal-space
 *                virial W_ab = -dU_recip/d(strain_ab) (reading C-7; the self term has none)
 * F32/MIXED contexts spread, transform and interpolate in fp32 and reduce energy/virial in fp64; F64 contexts are fp64
 * throughout.  The mesh, the cuFFT plans and their work area are kept in the context and re-made when mesh or order
 * change (that first call synchronises the stream); otherwise the call does not synchronise. */
DIMOS_API int dimos_pme_recip(dimos_ctx* ctx, const void* pos, const void* charge, int64_t N, const double* box, double alpha,
                              const int32_t* mesh, int32_t order, double coulomb_const, void* F, int32_t accumulate, double* E,
                              double* virial, void* stream);

/* dimos_pme_mesh_size -- the paper's mesh heuristic n_mesh = 2 alpha d / (3 delta^(1/5)) per box edge d,
 * rounded up to the next size with prime factors 2, 3, 5, 7.  Host only; mesh_out receives 3 int32. */
DIMOS_API int dimos_pme_mesh_size(double alpha, const double* box, double delta, int32_t* mesh_out);

/* dimos_lj_table_fill -- Lorentz-Berthelot combining rules, Eq. 5: sigma_ab = (sigma_a + sigma_b) / 2,
 * eps_ab = sqrt(eps_a eps_b), written as the ntypes x ntypes x 2 table (sigma_ab, eps_ab) that dimos_nonbonded takes
 * (reading C-16).  Host only: sigma, eps host arrays of ntypes doubles, table_out host array of 2 ntypes^2 doubles. */
DIMOS_API int dimos_lj_table_fill(const double* sigma, const double* eps, int32_t ntypes, double* table_out);

/* dimos_dispersion_correction -- PAPER.md:202 ("long-range dispersion corrections that approximate the contributions
 * beyond r_c"; the paper gives no formula: reading C-22).  The homogeneous-fluid tail of the 12-6 potential that the
 * truncated (and, with r_switch, switched) pair sum leaves out:
 *   E = (2 pi / V) sum_a sum_b N_a N_b  integral [1 - S(r)] U_ab(r) r^2 dr,   S = 1 below r_s, Eq. 6 up to r_c, 0 beyond
 * A constant for a given composition, box, r_cut and r_switch; the type histogram is taken on the device, the
 * integrals in closed form (tail) and by Gauss-Legendre quadrature (switching interval) on the host.
 *   type      dev, N int32;   lj_table  dev, ntypes x ntypes x 2 doubles (sigma_ab, eps_ab) as for dimos_nonbonded
 *   box       host, 3 doubles;   r_switch <= 0 or >= r_cut: plain truncation
 *   E_host    host, 1 double, written;   virial_host  host, 9 doubles or NULL: E * identity (E ~ 1/V; reading C-7)
 * Synchronises the stream. */
DIMOS_API int dimos_dispersion_correction(dimos_ctx* ctx, const int32_t* type, int64_t N, const double* lj_table,
                                          int32_t ntypes, const double* box, double r_cut, double r_switch, double* E_host,
                                          double* virial_host, void* stream);

/* dimos_virtual_box -- non-periodic systems ("the system is ... embedded into a non-periodic box" for the
 * neighbour-list computation).  Returns the edges of a virtual periodic box around the current positions that is large
 * enough for the periodic routines to reproduce open boundaries exactly: box[a] = extent[a] + r_cut + 2 skin (at least
 * 2 r_cut), so the periodic images of the system are farther apart than r_cut + skin and stay so while no atom has
 * moved more than skin/2 since (the rebuild trigger).  Use the returned box in dimos_nl_build and dimos_nonbonded (positions
 * need no shift: the routines wrap consistently), and call it again before every rebuild.  Meaningful with DIMOS_RF
 * (or eps_rf = 1 for a plain shifted cutoff); the Ewald variant presumes a real periodic system.
 *   pos        dev, N x 3, float or double per the context precision
 *   box_host   host, 3 doubles, written (fp32-representable values)
 *   lo_host    host, 3 doubles, written if not NULL: the lower corner of the bounding box
 * Synchronises the stream.  DIMOS_EINVAL for a non-finite coordinate. */
DIMOS_API int dimos_virtual_box(dimos_ctx* ctx, const void* pos, int64_t N, double r_cut, double skin, double* box_host,
                                double* lo_host, void* stream);

/* dimos_vv_kick_drift / dimos_vv_kick -- velocity Verlet, PAPER.md:281-292 (steps 1 + 2, and step 5; steps 3 and 6 for rigid water are
 * dimos_settle and dimos_settle_velocities; step 7 is dimos_berendsen).  Units nm, ps, amu, kJ mol^-1 nm^-1: a = F / m needs no conversion factor.
 *   kick_drift:  v <- v + (dt/2) F / m;  x <- x + dt v      (in place)
 *   kick:        v <- v + (dt/2) F / m                      (in place, with the forces at the new positions)
 *   pos, vel, F   dev, N x 3, float or double per the context precision
 *   inv_mass      dev, N, same type: 1 / m_i
 *   pos_at_build, skin, flag_dev, flag_host (kick_drift only; pos_at_build and flag_dev both NULL to skip): the rebuild
 *                 trigger of dimos_nl_needs_rebuild evaluated on the NEW positions in the same pass.
 *                 A non-NULL flag_host synchronises the stream.
 *   skip_flag     (kick only) NULL, or a device word as in dimos_nb_params.skip_flag: if it is non-zero when the kernel runs,
 *                 vel is left untouched.  With it a whole step -- kick_drift (sets the flag), dimos_nonbonded and this kick, all
 *                 given the same word -- can be enqueued or recorded in a CUDA graph without the host knowing the flag: on
 *                 the step where it fires the forces and the second kick do nothing, and the host finishes that step
 *                 (dimos_nl_build, dimos_nonbonded, this kick, all without skip_flag). */
DIMOS_API int dimos_vv_kick_drift(dimos_ctx* ctx, void* pos, void* vel, const void* F, const void* inv_mass, int64_t N,
                                  double dt, const void* pos_at_build, double skin, int32_t* flag_dev, int32_t* flag_host,
                                  void* stream);
DIMOS_API int dimos_vv_kick(dimos_ctx* ctx, void* vel, const void* F, const void* inv_mass, int64_t N, double dt,
                            const int32_t* skip_flag, void* stream);

/* dimos_settle -- step 3 of velocity Verlet for rigid three-site water: the SETTLE closed form that
 * PAPER.md:327 names, i.e. the positions the three distance constraints |O-H1| = |O-H2| = d_OH, |H1-H2| = d_HH admit when
 * the correction of every pair acts along its OLD bond vector, weighted by inverse mass (the converged SHAKE solution).
 *   pos_old   dev, N x 3: positions before the drift; they must satisfy the constraints
 *   pos       dev, N x 3: positions after the unconstrained drift, corrected in place
 *   vel       dev, N x 3 or NULL: if given, v += (x_constrained - x_unconstrained) / dt, the half-step velocity that goes
 *             with the constrained positions (step 6 is dimos_settle_velocities)
 *   water     dev, n_w x 3 int32: atom indices (O, H1, H2) of each molecule; molecules must be whole (no atom of a molecule
 *             wrapped into another periodic image), which dimos_vv_kick_drift preserves since it never wraps.  Every index
 *             must be a valid row of pos / vel and no atom may belong to two molecules; the call does not receive N, so
 *             neither is checked (this holds for every call that takes `water`)
 *   m_O, m_H  masses; d_OH, d_HH the constraint lengths (0 < d_HH < 2 d_OH)
 * float or double per the context precision (coordinates enter only as differences to the old oxygen).  Asynchronous on
 * the stream; n_w = 0 is a no-op.  DIMOS_EINVAL for bad lengths, masses or dt. */
DIMOS_API int dimos_settle(dimos_ctx* ctx, const void* pos_old, void* pos, void* vel, const int32_t* water, int64_t n_w,
                           double m_O, double m_H, double d_OH, double d_HH, double dt, void* stream);

/* dimos_settle_velocities -- step 6 of velocity Verlet for rigid three-site water: after the second
 * kick, remove the component of every relative velocity along its bond, (v_i - v_j) . (x_i - x_j) = 0 for the three bonds,
 * by impulses along the bonds shared by inverse mass (the converged RATTLE velocity stage); the three multipliers of a
 * molecule come from one direct 3 x 3 solve.  Linear and angular momentum of each molecule are unchanged.
 *   pos     dev, N x 3: the (constrained) positions of the step
 *   vel     dev, N x 3: corrected in place
 *   water   dev, n_w x 3 int32 (O, H1, H2), molecules whole, as for dimos_settle
 * Asynchronous on the stream; n_w = 0 is a no-op. */
DIMOS_API int dimos_settle_velocities(dimos_ctx* ctx, const void* pos, void* vel, const int32_t* water, int64_t n_w,
                                      double m_O, double m_H, void* stream);

/* dimos_kinetic_energy / dimos_berendsen -- step 7 of velocity Verlet with the Berendsen thermostat,
 * the velocity-rescaling thermostat of PAPER.md:306.  Units nm, ps, amu, kJ/mol, K; k_B = 8.314462618e-3 kJ mol^-1 K^-1.
 *   kinetic_energy:  K = 1/2 sum_i m_i |v_i|^2  -> *ke_dev (and *ke_host if not NULL, which synchronises the stream)
 *   berendsen:       T = 2 K / (n_dof k_B);  v <- v sqrt(1 + (dt/tau) (T0/T - 1))  in place, lambda taken from the
 *                    device-resident K (no host round trip); *ke_dev holds K BEFORE the scaling, *T_host (if not NULL,
 *                    synchronises) the temperature before the scaling
 *   vel        dev, N x 3, float or double per the context precision;  inv_mass  dev, N, same type: 1 / m_i
 *   n_dof      degrees of freedom, e.g. 3 N - 3 or, with rigid water, 6 n_w - 3
 *   ke_dev     dev, one double, written (the caller owns it)
 * The sum is accumulated in fp64 with one atomic per thread block: its last bits depend on the block order.
 * DIMOS_EINVAL unless T0 >= 0 and 0 < dt <= tau.  A system at rest (K = 0) has no temperature to rescale: its
 * velocities are left as they are (lambda = 1).  Atoms with inv_mass = 0 (frozen) carry no kinetic energy. */
DIMOS_API int dimos_kinetic_energy(dimos_ctx* ctx, const void* vel, const void* inv_mass, int64_t N, double* ke_dev,
                                   double* ke_host, void* stream);
DIMOS_API int dimos_berendsen(dimos_ctx* ctx, void* vel, const void* inv_mass, int64_t N, int64_t n_dof, double T0, double tau,
                              double dt, double* ke_dev, double* T_host, void* stream);
/* dimos_langevin_ou -- Langevin dynamics (PAPER.md:309 names it and gives no formula: reading C-26): the friction + noise
 * part of dv = -gamma v dt + sqrt(2 gamma k_B T / m) dW integrated exactly over one time step, applied where velocity Verlet
 * has its step 7:   v <- a v + sqrt((1 - a^2) k_B T / m) xi,   a = exp(-gamma dt).
 *   vel       dev, N x 3, in place;   inv_mass  dev, N (1 / m_i; 0 = frozen atom: its velocity only decays)
 *   xi        dev, N x 3 standard normal numbers supplied by the caller (e.g. torch.randn on the device), same type
 *   gamma     friction in ps^-1 (0: no-op up to rounding);   T in K;   k_B = 8.314462618e-3 kJ mol^-1 K^-1
 * With rigid water the velocity constraints (dimos_settle_velocities) must be applied again afterwards. */
DIMOS_API int dimos_langevin_ou(dimos_ctx* ctx, void* vel, const void* inv_mass, const void* xi, int64_t N, double gamma, double dt,
                                double T, void* stream);
/* dimos_berendsen_scale -- the rescaling half of dimos_berendsen with the kinetic energy taken from *ke_dev as some earlier
 * call on the same stream left it (dimos_kinetic_energy, dimos_water_kick_settle_velocities): one pass over vel, no sum. */
DIMOS_API int dimos_berendsen_scale(dimos_ctx* ctx, void* vel, int64_t N, int64_t n_dof, double T0, double tau, double dt,
                                    const double* ke_dev, void* stream);

/* dimos_water_kick_drift_settle / dimos_water_kick_settle_velocities -- the velocity-Verlet loop of PAPER.md:281-292 for a
 * system of rigid three-site waters in two passes instead of five: each thread holds one molecule in registers.
 *   kick_drift_settle:       steps 1 + 2 + 3 = dimos_vv_kick_drift, then dimos_settle with vel and the pre-drift positions
 *                            (no copy of the old positions is needed), then the rebuild trigger of dimos_nl_needs_rebuild
 *                            on the CONSTRAINED positions (pos_at_build, skin, flag_dev, flag_host as in dimos_vv_kick_drift)
 *   kick_settle_velocities:  steps 5 + 6 = dimos_vv_kick, then dimos_settle_velocities; if ke_dev is not NULL it receives
 *                            the kinetic energy of the constrained velocities (step 8; one double, fp64 accumulation)
 * Same arithmetic as the separate calls, in the same order.  Only atoms listed in `water` (dev, n_w x 3 int32: O, H1, H2)
 * are moved; masses come from m_O, m_H.  pos must satisfy the constraints on entry to kick_drift_settle.  Asynchronous on
 * the stream unless flag_host is given.  kick_settle_velocities takes skip_flag as dimos_vv_kick does (vel untouched, and
 * *ke_dev = 0, when the word is non-zero). */
DIMOS_API int dimos_water_kick_drift_settle(dimos_ctx* ctx, void* pos, void* vel, const void* F, const int32_t* water,
                                            int64_t n_w, double m_O, double m_H, double d_OH, double d_HH, double dt,
                                            const void* pos_at_build, double skin, int32_t* flag_dev, int32_t* flag_host,
                                            void* stream);
DIMOS_API int dimos_water_kick_settle_velocities(dimos_ctx* ctx, const void* pos, void* vel, const void* F, const int32_t* water,
                                                 int64_t n_w, double m_O, double m_H, double dt, double* ke_dev,
                                                 const int32_t* skip_flag, void* stream);

/* dimos_nl_set_exceptions -- PAPER.md:243 ("1-4 exceptions ... scale the strength of the non-bonded interactions by
 * some common factor", or an individual factor per pair; "handled explicitly by the non-bonded interaction method").
 * Reading C-21 (the paper gives no formula): every exception pair must ALSO be one of the excluded pairs the list was
 * built with, so the pair sums skip it (under DIMOS_EWALD_REAL it keeps the exclusion correction); dimos_nonbonded
 * then adds, for every exception, s_lj * U_LJ(r) (Eq. 4) + s_c * k_e q_i q_j / r (Eq. 7) at the minimum-image distance,
 * without cutoff, switch, reaction-field or Ewald modification, and the matching forces and virial.  The LJ part goes
 * into E[1], the Coulomb part into E[2].
 *   pairs   dev, n_exc x 2 int32, (i, j) with i < j, original atom indices, each pair once (a repeated row is applied
 *           repeatedly; not checked); read (copied into the list)
 *   scale   dev, n_exc x 2 double, (s_c, s_lj) per pair; read (copied)
 *   n_exc   >= 0; 0 removes the exceptions.  The copy belongs to the list and survives rebuilds in place.
 * The list is checked here (indices in range, i < j, every pair among the list's excluded pairs: DIMOS_EINVAL
 * otherwise); the call synchronises the stream.  Every later dimos_nl_build into the same handle repeats the check against
 * the atom count and the exclusion list it is given: if the stored exceptions no longer fit, that build removes them and
 * returns DIMOS_EINVAL (build again, then set the exceptions that belong to the new system). */
DIMOS_API int dimos_nl_set_exceptions(dimos_ctx* ctx, dimos_nl* nl, const int32_t* pairs, const double* scale,
                                      int64_t n_exc, void* stream);

/* dimos_nl_export_edges -- the neighbour list as an edge list with distance vectors and periodic shifts, the form a
 * machine-learned interatomic potential consumes (PAPER.md:179-185 get_neighborlist, 251).  Like dimos_nl_export_pairs,
 * but only the pairs with minimum-image r < radius (0 < radius <= r_cut + skin) at the build positions, and per pair k
 *   pairs[k] = (a, b), a < b, original atom indices          dev, cap x 2 int32
 *   dvec[k]  = r_a - r_b - shift[k] * box (minimum image)    dev, cap x 3, float or double per the precision; may be NULL
 *   shift[k] = nearbyint((r_a - r_b) / box) per axis         dev, cap x 3 int32; may be NULL
 * in unspecified order (the three arrays share it).  n_pairs_host receives the number of edges; if it exceeds cap only
 * the first cap were written and the call returns DIMOS_EOVERFLOW.  Synchronises the stream. */
DIMOS_API int dimos_nl_export_edges(dimos_ctx* ctx, const dimos_nl* nl, double radius, int32_t* pairs, void* dvec,
                                    int32_t* shift, int64_t cap, int64_t* n_pairs_host, void* stream);

/* Number of unordered, non-excluded pairs of the list with minimum-image r < radius at the build
 * positions, 0 < radius <= r_cut + skin (radius = r_cut gives the in-cutoff pair count the
 * throughput metric "pair interactions/s" is quoted on).  Synchronises the stream. */
DIMOS_API int dimos_nl_count_within(dimos_ctx* ctx, const dimos_nl* nl, double radius, int64_t* n_pairs_host,
                                    void* stream);

/* Sizes of the list (host call, no device work). */
DIMOS_API int dimos_nl_stats(const dimos_nl* nl, dimos_nl_stats_t* out);

/* Number of kernels of this library launched through ctx since dimos_create (host counter). */
DIMOS_API int64_t dimos_launch_count(const dimos_ctx* ctx);

/* Per-kernel timing of the pair-force kernel (row A4) for bench.py's roofline: while enabled,
 * dimos_nonbonded records a CUDA event pair around that one kernel on the call's stream (at most
 * 4096 launches between reads).  dimos_profile_read synchronises on the recorded events, returns
 * the summed kernel time in milliseconds and the number of launches it covers, and resets. */
DIMOS_API int dimos_profile_enable(dimos_ctx* ctx, int on);
DIMOS_API int dimos_profile_read(dimos_ctx* ctx, double* pair_force_ms_host, int64_t* n_launches_host);

/* Peak-rate probe used by bench.py's roofline: runs an FFMA-only microkernel on the context's
 * device for about `ms_target` milliseconds and returns the measured FP32 rate in *tflops_host
 * (2 flops per FMA).  Synchronises. */
DIMOS_API int dimos_probe_fp32_peak(dimos_ctx* ctx, double ms_target, double* tflops_host, void* stream);

DIMOS_API const char* dimos_status_string(int status);
DIMOS_API const char* dimos_last_error(const dimos_ctx* ctx);
DIMOS_API const char* dimos_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DIMOS_H_ */
