// common.cuh -- internal declarations shared by the translation units of libdimos_b200.
// Product code: shares nothing with oracle/ (see DESIGN.md).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/dimos.h"

namespace dimos {

constexpr int UNIT = DIMOS_UNIT;  // atoms per i-cluster
constexpr int KD_MAX = 4096;      // max atoms per cell the in-cell sorter handles
constexpr int MAX_EXCL_PER_ATOM = 32;
constexpr int MAX_TYPES = 64;
constexpr int LIST_SLACK = 1024;  // entries readable past the last row (the force kernels prefetch two chunks ahead unguarded)
constexpr int SELF_CODE = 13;  // stencil code of offset (0,0,0): (dx+1)*9+(dy+1)*3+(dz+1)
// one list entry = one 32-bit word: slot of the j-atom (low 27 bits) | stencil code of its periodic image (high 5 bits);
// the 8-bit i-mask of an entry lives in a parallel byte array and is read for the masked chunks only
constexpr unsigned ENTRY_SLOT_BITS = 27;
constexpr unsigned ENTRY_SLOT_MASK = (1u << ENTRY_SLOT_BITS) - 1u;
// Offset (in entries, from the row's first entry) of chunk c of a row of `total` chunks: the first n_am = nA + nM chunks
// sit at the row's start, the remaining (mask-free, LJ-free) ones END at the row's capacity nu_cap = row_cap - m_res
// (the list builder fills the row from both ends).
__host__ __device__ inline int row_chunk_offset(int c, int total, int n_am, int nu_cap) { return c < n_am ? c * 32 : nu_cap - (total - c) * 32; }
__host__ __device__ inline unsigned entry_pack(int slot, int code) { return (unsigned)slot | ((unsigned)code << ENTRY_SLOT_BITS); }

// device error flag bits (NL::d_flags[0])
enum : int {
    FLAG_ROW_OVERFLOW = 1,     // a unit row needed more than row_cap entries
    FLAG_MASKED_OVERFLOW = 2,  // more masked entries than m_res in one unit
    FLAG_NONFINITE = 4,        // non-finite coordinate
    FLAG_CELL_OVERFLOW = 8,    // more than KD_MAX atoms in one cell
    FLAG_EXCL_OVERFLOW = 16,   // more than MAX_EXCL_PER_ATOM partners for one atom
    FLAG_EXCL_RANGE = 32,      // exclusion index out of range / not i<j
    FLAG_EXCL_DUP = 64         // the same exclusion pair listed twice
};

template <typename real> struct vec4;
template <> struct vec4<float> { using type = float4; };
template <> struct vec4<double> { using type = double4; };

struct DevBuf {
    void* p = nullptr;
    size_t bytes = 0;
};

struct Ctx {
    int device = 0;
    int precision = DIMOS_F32;
    bool has_alloc = false;
    dimos_allocator alloc{};
    std::string err;
    int64_t launches = 0;
    int sm_count = 148;
    int* h_pinned = nullptr;        // 64 ints pinned scratch for read-backs
    unsigned long long* d_rebuild_state = nullptr;  // TRIGGER_RING x {max bits, ticket}: one pair per trigger call in flight
    unsigned trigger_seq = 0;
    cudaEvent_t ev_flag = nullptr;  // dimos_step_host: marks the arrival of the trigger flag in pinned memory
    DevBuf scratch;  // small per-context device scratch (type histogram of dimos_dispersion_correction)
    std::vector<struct NL*> lists;
    struct PmePlan* pme = nullptr;  // cuFFT plans, mesh and accumulators of dimos_pme_recip (pme.cu), rebuilt when the mesh changes
    // optional per-kernel timing of the pair-force kernel (dimos_profile_enable / dimos_profile_read)
    bool profiling = false;
    std::vector<cudaEvent_t> prof_events;  // pairs (start, stop), recycled after each read
    size_t prof_used = 0;                  // events handed out since the last read
};
constexpr size_t PROF_MAX_EVENTS = 8192;
constexpr unsigned TRIGGER_RING = 64;
// reduction state of the next rebuild-trigger kernel: consecutive calls (possibly on different streams, several lists per
// context) never share a {max, ticket} pair unless more than TRIGGER_RING of them are in flight at once
inline unsigned long long* next_trigger_state(Ctx* ctx) { return ctx->d_rebuild_state + 2 * (ctx->trigger_seq++ % TRIGGER_RING); }

// geometry of the cell grid / list, passed by value to kernels
struct Grid {
    int n[3];          // cells per axis
    int pbc_mode;      // 0: image from cell offsets (all n >= 3), 1: per-pair minimum image
    double L[3];       // box
    double h[3];       // cell edge = L / n
    int64_t ncells;
};

struct NL {
    Ctx* ctx = nullptr;
    int64_t N = 0;
    double box[3] = {0, 0, 0};
    double r_cut = 0, skin = 0, r_nl = 0;
    Grid grid{};
    int64_t n_units = 0, n_slots = 0;
    int row_cap = 0;  // entries per unit row (multiple of 32), includes m_res
    int m_res = 128;  // max masked entries per row staged by the builder (multiple of 32); rows start m_res entries into their slab
    int n_grow = 0;
    int64_t n_entries = 0, n_entries_padded = 0;
    int64_t n_excl = 0;
    int max_cell_count = 0;

    // build-time device arrays
    DevBuf cell_count, cell_start, unit_start, scan_tmp;  // int[ncells+1] each
    DevBuf atom_cell, atom_rank, cell_atoms;              // int[N]
    DevBuf perm;       // int[n_slots]: original atom index, or ~src for padding slots
    DevBuf inv_perm;   // int[N]: slot of each original atom
    DevBuf ref;        // double[3*n_slots]: origin subtracted from the raw coordinate
    DevBuf xyz_build;  // real4[n_slots]: cell-relative coordinates at build time
    DevBuf bb_lo, bb_hi;  // real4[n_units] unit bounding boxes (cell-relative)
    DevBuf unit_cell;  // int[n_units]
    DevBuf excl_start, excl_adj;  // CSR over both directions: int[N+1], int[2*n_excl]
    DevBuf excl_pairs;            // int2[n_excl] copy (Ewald exclusion correction)
    DevBuf exc_pairs, exc_scale;  // 1-4 exceptions: int2[n_exc], double2[n_exc] = (Coulomb scale, LJ scale); survive rebuilds
    int64_t n_exc = 0;
    DevBuf entry;      // uint32[n_units*row_cap]: slot | code << 27
    DevBuf emask;      // uint8[n_units*row_cap]: i-mask of the entry (all-ones in the mask-free chunks)
    DevBuf row_info;   // int2[n_units]: {chunks in the row | partial-unit flag << 16, nA | nM << 16}: nA mask-free chunks of
                       // j-atoms assumed LJ-active, then nM chunks that read their masks, then (at the end of the row's
                       // capacity, see row_chunk_offset) the mask-free chunks of j-atoms assumed LJ-free
    DevBuf slot_hint;  // uint8[n_slots]: the LJ-activity flag the builder assumed for the slot's atom (1 without a hint)
    DevBuf atom_active;  // uint8[N]: LJ-activity of every atom at the last force call = the next build's hint
    bool hint_valid = false;
    DevBuf flags;      // int[16]: [0] error flags, [1] max cell count, [2..3] entry counters (u64), [4..5] padded, [6..7] needed
                       // capacities, [8] row order stale (an atom became LJ-active), [9] type index out of range, [10] exception check
    // per-step device arrays
    DevBuf xyzq;       // real4[n_slots]
    DevBuf stype;      // int[n_slots]
    DevBuf Facc;       // real4[n_slots] j-side force accumulators (atomics)
    DevBuf Fown;       // real4[n_slots] i-side forces (plain stores)
    DevBuf lj;         // real2[nt*nt] (c6,c12) + int[nt] row-active flags after it
    DevBuf partials;   // double[9 * n_partial_blocks]
    DevBuf accum;      // double[16] + unsigned ticket
    // host-call staging (dimos_nonbonded_host)
    DevBuf st_pos, st_charge, st_type, st_lj, st_F, st_EW, st_ref, st_flag;
    int st_static_ntypes = 0;  // ntypes of the charge / type / lj_table copies held in st_* (dimos_step_host), 0 = none
    DevBuf export_count;  // unsigned long long[1]
};

// ---- helpers implemented in api.cu ------------------------------------------------------------
int set_error(Ctx* ctx, int status, const std::string& msg);
int ensure(Ctx* ctx, DevBuf& b, size_t bytes, cudaStream_t s);
void release(Ctx* ctx, DevBuf& b);

#define DIMOS_CUDA_TRY(ctx, call)                                                                   \
    do {                                                                                            \
        cudaError_t e_ = (call);                                                                    \
        if (e_ != cudaSuccess)                                                                      \
            return ::dimos::set_error((ctx), DIMOS_ECUDA,                                           \
                                      std::string(#call) + ": " + cudaGetErrorString(e_));          \
    } while (0)

#define DIMOS_LAUNCH_CHECK(ctx, name)                                                               \
    do {                                                                                            \
        (ctx)->launches++;                                                                          \
        cudaError_t e_ = cudaGetLastError();                                                        \
        if (e_ != cudaSuccess)                                                                      \
            return ::dimos::set_error((ctx), DIMOS_ECUDA,                                           \
                                      std::string("launch ") + name + ": " + cudaGetErrorString(e_)); \
    } while (0)

// ---- entry points implemented per translation unit ---------------------------------------------
int nl_build_impl(Ctx* ctx, NL* nl, const void* pos, const int32_t* excl_pairs, int64_t n_excl,
                  void* pos_at_build, cudaStream_t s);
int nl_export_impl(Ctx* ctx, const NL* nl, int32_t* pairs, int64_t cap, int64_t* n_pairs_host, double radius, cudaStream_t s,
                   void* dvec = nullptr, int32_t* shift = nullptr);
int needs_rebuild_impl(Ctx* ctx, const void* pos, const void* ref, int64_t N, double skin, int32_t* flag_dev,
                       cudaStream_t s);
int nonbonded_impl(Ctx* ctx, NL* nl, const void* pos, const void* charge, const int32_t* type,
                   const double* lj_table, int32_t ntypes, const dimos_nb_params* prm, void* F, double* E,
                   double* virial, cudaStream_t s);
int probe_fp32_impl(Ctx* ctx, double ms_target, double* tflops, cudaStream_t s);
int check_exceptions_impl(Ctx* ctx, const NL* nl, const int32_t* pairs, int64_t n_exc, int* bad_dev, cudaStream_t s);
int pme_recip_impl(Ctx* ctx, const void* pos, const void* charge, int64_t n, const double* box, double alpha, const int32_t* mesh,
                   int32_t order, double ke, void* F, double* E, double* W, int accumulate, cudaStream_t s);
void pme_release(Ctx* ctx);
int vv_kick_drift_impl(Ctx* ctx, void* pos, void* vel, const void* F, const void* inv_mass, int64_t N, double dt,
                       const void* pos_at_build, double skin, int32_t* flag_dev, cudaStream_t s);
int bbox_impl(Ctx* ctx, const void* pos, int64_t N, unsigned* out_dev, cudaStream_t s);
int type_histogram_impl(Ctx* ctx, const int32_t* type, int64_t N, int nt, unsigned long long* counts_dev, int* bad_dev,
                        cudaStream_t s);
int vv_kick_impl(Ctx* ctx, void* vel, const void* F, const void* inv_mass, int64_t N, double dt, const int32_t* skip, cudaStream_t s);
int langevin_ou_impl(Ctx* ctx, void* vel, const void* inv_mass, const void* xi, int64_t N, double gamma, double dt, double T, cudaStream_t s);
int settle_impl(Ctx* ctx, const void* pos_old, void* pos, void* vel, const int32_t* water, int64_t n_w, double m_O,
                double m_H, double d_OH, double d_HH, double dt, cudaStream_t s);
int water_step_a_impl(Ctx* ctx, void* pos, void* vel, const void* F, const int32_t* water, int64_t n_w, double m_O, double m_H,
                      double d_OH, double d_HH, double dt, const void* ref, double skin, int32_t* flag_dev, cudaStream_t s);
int water_step_b_impl(Ctx* ctx, const void* pos, void* vel, const void* F, const int32_t* water, int64_t n_w, double m_O,
                      double m_H, double dt, double* ke_dev, const int32_t* skip, cudaStream_t s);
int kinetic_energy_impl(Ctx* ctx, const void* vel, const void* inv_mass, int64_t N, double* ke_dev, cudaStream_t s);
int berendsen_scale_impl(Ctx* ctx, void* vel, int64_t N, const double* ke_dev, double two_over_dof_kb, double T0,
                         double dt_over_tau, cudaStream_t s);
int settle_vel_impl(Ctx* ctx, const void* pos, void* vel, const int32_t* water, int64_t n_w, double m_O, double m_H,
                    cudaStream_t s);

// stencil code <-> offset
__host__ __device__ inline int stencil_code(int dx, int dy, int dz) { return (dx + 1) * 9 + (dy + 1) * 3 + (dz + 1); }

}  // namespace dimos
