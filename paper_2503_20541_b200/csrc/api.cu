// api.cu -- the extern "C" boundary of libdimos_b200 (include/dimos.h): argument validation,
// context / workspace management and dispatch to the kernels in nl_build.cu and nonbonded.cu.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "common.cuh"

namespace dimos {

int set_error(Ctx* ctx, int status, const std::string& msg)
{
    if (ctx) ctx->err = msg;
    return status;
}

int ensure(Ctx* ctx, DevBuf& b, size_t bytes, cudaStream_t s)
{
    if (bytes == 0) bytes = 16;
    if (b.p && b.bytes >= bytes) return DIMOS_OK;
    // grow with headroom so that small size changes between rebuilds do not reallocate
    size_t want = b.p ? bytes + bytes / 8 : bytes;
    want = (want + 255) & ~(size_t)255;
    if (b.p) release(ctx, b);
    void* p = nullptr;
    if (ctx->has_alloc) {
        p = ctx->alloc.alloc(want, (void*)s, ctx->alloc.user);
        if (!p) return set_error(ctx, DIMOS_ENOMEM, "allocator callback returned NULL for " + std::to_string(want) + " bytes");
    } else {
        cudaError_t e = cudaMalloc(&p, want);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return set_error(ctx, DIMOS_ENOMEM, std::string("cudaMalloc: ") + cudaGetErrorString(e));
        }
    }
    b.p = p;
    b.bytes = want;
    return DIMOS_OK;
}

void release(Ctx* ctx, DevBuf& b)
{
    if (!b.p) return;
    if (ctx->has_alloc) ctx->alloc.free_(b.p, ctx->alloc.user);
    else cudaFree(b.p);
    b.p = nullptr;
    b.bytes = 0;
}

static void free_list(Ctx* ctx, NL* nl)
{
    DevBuf* bufs[] = {&nl->cell_count, &nl->cell_start, &nl->unit_start, &nl->scan_tmp, &nl->atom_cell, &nl->atom_rank,
                      &nl->cell_atoms, &nl->perm, &nl->inv_perm, &nl->ref, &nl->xyz_build, &nl->bb_lo, &nl->bb_hi,
                      &nl->unit_cell, &nl->excl_start, &nl->excl_adj, &nl->excl_pairs, &nl->jslot, &nl->meta, &nl->row_info,
                      &nl->flags, &nl->xyzq, &nl->stype, &nl->Facc, &nl->Fown, &nl->lj, &nl->partials, &nl->accum,
                      &nl->st_pos, &nl->st_charge, &nl->st_type, &nl->st_lj, &nl->st_F, &nl->st_EW, &nl->export_count};
    for (DevBuf* b : bufs) release(ctx, *b);
    delete nl;
}

static size_t list_workspace_bytes(const NL* nl)
{
    const DevBuf* bufs[] = {&nl->cell_count, &nl->cell_start, &nl->unit_start, &nl->scan_tmp, &nl->atom_cell, &nl->atom_rank,
                            &nl->cell_atoms, &nl->perm, &nl->inv_perm, &nl->ref, &nl->xyz_build, &nl->bb_lo, &nl->bb_hi,
                            &nl->unit_cell, &nl->excl_start, &nl->excl_adj, &nl->excl_pairs, &nl->jslot, &nl->meta,
                            &nl->row_info, &nl->flags, &nl->xyzq, &nl->stype, &nl->Facc, &nl->Fown, &nl->lj, &nl->partials,
                            &nl->accum, &nl->st_pos, &nl->st_charge, &nl->st_type, &nl->st_lj, &nl->st_F, &nl->st_EW,
                            &nl->export_count};
    size_t t = 0;
    for (const DevBuf* b : bufs) t += b->bytes;
    return t;
}

static bool list_belongs(const Ctx* ctx, const NL* nl)
{
    return nl && std::find(ctx->lists.begin(), ctx->lists.end(), nl) != ctx->lists.end();
}

}  // namespace dimos

using namespace dimos;

extern "C" {

DIMOS_API int dimos_create(dimos_ctx** out, int device, int precision, const dimos_allocator* allocator)
{
    if (!out) return DIMOS_EINVAL;
    *out = nullptr;
    if (precision != DIMOS_F32 && precision != DIMOS_F64 && precision != DIMOS_MIXED) return DIMOS_EINVAL;
    if (allocator && (!allocator->alloc || !allocator->free_)) return DIMOS_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) { cudaGetLastError(); return DIMOS_ECUDA; }
    if (device < 0 || device >= ndev) return DIMOS_EINVAL;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return DIMOS_ECUDA; }
    Ctx* ctx = new (std::nothrow) Ctx();
    if (!ctx) return DIMOS_ENOMEM;
    ctx->device = device;
    ctx->precision = precision;
    if (allocator) { ctx->has_alloc = true; ctx->alloc = *allocator; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { delete ctx; return DIMOS_ECUDA; }
    ctx->sm_count = prop.multiProcessorCount;
    if (prop.major < 10) { delete ctx; return DIMOS_ECUDA; }  // built for sm_100a only
    if (cudaMallocHost((void**)&ctx->h_pinned, 64 * sizeof(int)) != cudaSuccess) { delete ctx; return DIMOS_ENOMEM; }
    if (cudaMalloc((void**)&ctx->d_rebuild_state, 2 * sizeof(unsigned long long)) != cudaSuccess) {
        cudaFreeHost(ctx->h_pinned); delete ctx; return DIMOS_ENOMEM;
    }
    cudaMemset(ctx->d_rebuild_state, 0, 2 * sizeof(unsigned long long));
    *out = reinterpret_cast<dimos_ctx*>(ctx);
    return DIMOS_OK;
}

DIMOS_API int dimos_destroy(dimos_ctx* c)
{
    if (!c) return DIMOS_EINVAL;
    Ctx* ctx = reinterpret_cast<Ctx*>(c);
    cudaSetDevice(ctx->device);
    for (NL* nl : ctx->lists) free_list(ctx, nl);
    ctx->lists.clear();
    if (ctx->h_pinned) cudaFreeHost(ctx->h_pinned);
    if (ctx->d_rebuild_state) cudaFree(ctx->d_rebuild_state);
    delete ctx;
    return DIMOS_OK;
}

DIMOS_API int dimos_nl_destroy(dimos_ctx* c, dimos_nl* l)
{
    if (!c || !l) return DIMOS_EINVAL;
    Ctx* ctx = reinterpret_cast<Ctx*>(c);
    NL* nl = reinterpret_cast<NL*>(l);
    auto it = std::find(ctx->lists.begin(), ctx->lists.end(), nl);
    if (it == ctx->lists.end()) return set_error(ctx, DIMOS_EINVAL, "list does not belong to this context");
    ctx->lists.erase(it);
    free_list(ctx, nl);
    return DIMOS_OK;
}

DIMOS_API int dimos_nl_build(dimos_ctx* c, const void* pos, int64_t N, const double* box, double r_cut, double skin,
                             const int32_t* excl_pairs, int64_t n_excl, void* pos_at_build, void* stream, dimos_nl** inout)
{
    if (!c) return DIMOS_EINVAL;
    Ctx* ctx = reinterpret_cast<Ctx*>(c);
    if (!pos || !box || !pos_at_build || !inout) return set_error(ctx, DIMOS_EINVAL, "NULL argument");
    if (N <= 0 || N > 0x7fffffffLL - 64) return set_error(ctx, DIMOS_EINVAL, "N out of range");
    if (n_excl < 0 || (n_excl > 0 && !excl_pairs)) return set_error(ctx, DIMOS_EINVAL, "bad exclusion list");
    if (!(r_cut > 0) || !(skin >= 0) || !isfinite(r_cut) || !isfinite(skin)) return set_error(ctx, DIMOS_EINVAL, "r_cut must be > 0 and skin >= 0");
    double Lmin = 1e300;
    for (int a = 0; a < 3; ++a) {
        if (!isfinite(box[a]) || !(box[a] > 0)) return set_error(ctx, DIMOS_EINVAL, "box edges must be finite and positive");
        Lmin = std::min(Lmin, box[a]);
    }
    if (r_cut > 0.5 * Lmin) return set_error(ctx, DIMOS_EBOX, "r_cut exceeds half the shortest box edge");
    if (cudaSetDevice(ctx->device) != cudaSuccess) return set_error(ctx, DIMOS_ECUDA, "cudaSetDevice failed");

    NL* nl = reinterpret_cast<NL*>(*inout);
    bool created = false;
    if (nl) {
        if (!list_belongs(ctx, nl)) return set_error(ctx, DIMOS_EINVAL, "list does not belong to this context");
    } else {
        nl = new (std::nothrow) NL();
        if (!nl) return set_error(ctx, DIMOS_ENOMEM, "host allocation failed");
        nl->ctx = ctx;
        created = true;
    }
    const double r_nl = r_cut + skin;
    const bool same_geom = !created && nl->N == N && nl->r_nl == r_nl && nl->box[0] == box[0] && nl->box[1] == box[1] &&
                           nl->box[2] == box[2];
    if (!same_geom) nl->row_cap = 0;  // re-estimate the row capacity
    nl->N = N;
    nl->r_cut = r_cut;
    nl->skin = skin;
    nl->r_nl = r_nl;
    Grid& g = nl->grid;
    g.pbc_mode = 0;
    g.ncells = 1;
    for (int a = 0; a < 3; ++a) {
        nl->box[a] = box[a];
        g.L[a] = box[a];
        double nf = floor(box[a] / r_nl);  // cells of edge >= r_nl (reading C-18)
        int n = nf < 1 ? 1 : (nf > 1024 ? 1024 : (int)nf);
        g.n[a] = n;
        g.h[a] = box[a] / n;
        if (n < 3) g.pbc_mode = 1;
        g.ncells *= n;
    }
    int rc = nl_build_impl(ctx, nl, pos, excl_pairs, n_excl, pos_at_build, (cudaStream_t)stream);
    if (rc != DIMOS_OK) {
        if (created) free_list(ctx, nl);
        else nl->N = 0;  // marks the list unusable
        return rc;
    }
    if (created) ctx->lists.push_back(nl);
    *inout = reinterpret_cast<dimos_nl*>(nl);
    return DIMOS_OK;
}

DIMOS_API int dimos_nl_needs_rebuild(dimos_ctx* c, const void* pos, const void* pos_at_build, int64_t N, double skin,
                                     int32_t* flag_dev, int32_t* flag_host, void* stream)
{
    if (!c) return DIMOS_EINVAL;
    Ctx* ctx = reinterpret_cast<Ctx*>(c);
    if (!pos || !pos_at_build || !flag_dev) return set_error(ctx, DIMOS_EINVAL, "NULL argument");
    if (N <= 0 || !(skin >= 0)) return set_error(ctx, DIMOS_EINVAL, "bad N or skin");
    if (cudaSetDevice(ctx->device) != cudaSuccess) return set_error(ctx, DIMOS_ECUDA, "cudaSetDevice failed");
    cudaStream_t s = (cudaStream_t)stream;
    int rc = needs_rebuild_impl(ctx, pos, pos_at_build, N, skin, flag_dev, s);
    if (rc) return rc;
    if (flag_host) {
        DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_pinned + 32, flag_dev, sizeof(int), cudaMemcpyDeviceToHost, s));
        DIMOS_CUDA_TRY(ctx, cudaStreamSynchronize(s));
        *flag_host = ctx->h_pinned[32];
    }
    return DIMOS_OK;
}

static int check_nb_args(Ctx* ctx, const NL* nl, int32_t ntypes, const double* box, const dimos_nb_params* p)
{
    if (!list_belongs(ctx, nl)) return set_error(ctx, DIMOS_EINVAL, "list does not belong to this context");
    if (nl->N <= 0) return set_error(ctx, DIMOS_ESTALE, "list is not built");
    if (ntypes < 1 || ntypes > MAX_TYPES) return set_error(ctx, DIMOS_EINVAL, "ntypes must be in 1..64");
    if (p->method != DIMOS_RF && p->method != DIMOS_EWALD_REAL) return set_error(ctx, DIMOS_EINVAL, "unknown method");
    if (box[0] != nl->box[0] || box[1] != nl->box[1] || box[2] != nl->box[2]) return set_error(ctx, DIMOS_ESTALE, "box differs from the build box");
    if (p->r_cut != nl->r_cut) return set_error(ctx, DIMOS_ESTALE, "r_cut differs from the build r_cut");
    if (!(p->coulomb_const >= 0) || !isfinite(p->coulomb_const)) return set_error(ctx, DIMOS_EINVAL, "bad coulomb_const");
    if (p->method == DIMOS_RF && !(2.0 * p->eps_rf + 1.0 != 0.0)) return set_error(ctx, DIMOS_EINVAL, "bad eps_rf");
    if (p->method == DIMOS_EWALD_REAL && !(p->alpha > 0)) return set_error(ctx, DIMOS_EINVAL, "alpha must be > 0");
    return DIMOS_OK;
}

DIMOS_API int dimos_nonbonded(dimos_ctx* c, const dimos_nl* l, const void* pos, const void* charge, const int32_t* type,
                              const double* lj_table, int32_t ntypes, const double* box, const dimos_nb_params* params,
                              void* F, double* E, double* virial, void* stream)
{
    if (!c) return DIMOS_EINVAL;
    Ctx* ctx = reinterpret_cast<Ctx*>(c);
    if (!l || !pos || !charge || !type || !lj_table || !box || !params || !F || !E) return set_error(ctx, DIMOS_EINVAL, "NULL argument");
    NL* nl = const_cast<NL*>(reinterpret_cast<const NL*>(l));  // per-step workspace lives in the list
    int rc = check_nb_args(ctx, nl, ntypes, box, params);
    if (rc) return rc;
    if (cudaSetDevice(ctx->device) != cudaSuccess) return set_error(ctx, DIMOS_ECUDA, "cudaSetDevice failed");
    return nonbonded_impl(ctx, nl, pos, charge, type, lj_table, ntypes, params, F, E, virial, (cudaStream_t)stream);
}

DIMOS_API int dimos_nonbonded_host(dimos_ctx* c, dimos_nl* l, const void* pos_host, const void* charge_host,
                                   const int32_t* type_host, const double* lj_table_host, int32_t ntypes, const double* box,
                                   const dimos_nb_params* params, void* F_host, double* E_host, double* virial_host, void* stream)
{
    if (!c) return DIMOS_EINVAL;
    Ctx* ctx = reinterpret_cast<Ctx*>(c);
    if (!l || !pos_host || !charge_host || !type_host || !lj_table_host || !box || !params || !F_host || !E_host)
        return set_error(ctx, DIMOS_EINVAL, "NULL argument");
    NL* nl = reinterpret_cast<NL*>(l);
    int rc = check_nb_args(ctx, nl, ntypes, box, params);
    if (rc) return rc;
    if (cudaSetDevice(ctx->device) != cudaSuccess) return set_error(ctx, DIMOS_ECUDA, "cudaSetDevice failed");
    cudaStream_t s = (cudaStream_t)stream;
    const size_t rs = ctx->precision == DIMOS_F64 ? sizeof(double) : sizeof(float);
    const size_t N = (size_t)nl->N;
    if ((rc = ensure(ctx, nl->st_pos, 3 * N * rs, s))) return rc;
    if ((rc = ensure(ctx, nl->st_charge, N * rs, s))) return rc;
    if ((rc = ensure(ctx, nl->st_type, N * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->st_lj, (size_t)ntypes * ntypes * 2 * sizeof(double), s))) return rc;
    if ((rc = ensure(ctx, nl->st_F, 3 * N * rs, s))) return rc;
    if ((rc = ensure(ctx, nl->st_EW, 16 * sizeof(double), s))) return rc;
    DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(nl->st_pos.p, pos_host, 3 * N * rs, cudaMemcpyHostToDevice, s));
    DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(nl->st_charge.p, charge_host, N * rs, cudaMemcpyHostToDevice, s));
    DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(nl->st_type.p, type_host, N * sizeof(int), cudaMemcpyHostToDevice, s));
    DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(nl->st_lj.p, lj_table_host, (size_t)ntypes * ntypes * 2 * sizeof(double), cudaMemcpyHostToDevice, s));
    double* EW = (double*)nl->st_EW.p;
    rc = nonbonded_impl(ctx, nl, nl->st_pos.p, nl->st_charge.p, (const int32_t*)nl->st_type.p, (const double*)nl->st_lj.p,
                        ntypes, params, nl->st_F.p, EW, EW + 4, s);
    if (rc) return rc;
    DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(F_host, nl->st_F.p, 3 * N * rs, cudaMemcpyDeviceToHost, s));
    DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(E_host, EW, 4 * sizeof(double), cudaMemcpyDeviceToHost, s));
    if (virial_host) DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(virial_host, EW + 4, 9 * sizeof(double), cudaMemcpyDeviceToHost, s));
    DIMOS_CUDA_TRY(ctx, cudaStreamSynchronize(s));
    return DIMOS_OK;
}

DIMOS_API int dimos_nl_export_pairs(dimos_ctx* c, const dimos_nl* l, int32_t* pairs, int64_t cap, int64_t* n_pairs_host, void* stream)
{
    if (!c) return DIMOS_EINVAL;
    Ctx* ctx = reinterpret_cast<Ctx*>(c);
    if (!l || !n_pairs_host || cap < 0 || (cap > 0 && !pairs)) return set_error(ctx, DIMOS_EINVAL, "bad argument");
    const NL* nl = reinterpret_cast<const NL*>(l);
    if (!list_belongs(ctx, nl) || nl->N <= 0) return set_error(ctx, DIMOS_EINVAL, "list not built with this context");
    if (cudaSetDevice(ctx->device) != cudaSuccess) return set_error(ctx, DIMOS_ECUDA, "cudaSetDevice failed");
    return nl_export_impl(ctx, nl, pairs, cap, n_pairs_host, (cudaStream_t)stream);
}

DIMOS_API int dimos_nl_stats(const dimos_nl* l, dimos_nl_stats_t* out)
{
    if (!l || !out) return DIMOS_EINVAL;
    const NL* nl = reinterpret_cast<const NL*>(l);
    memset(out, 0, sizeof(*out));
    out->n_atoms = nl->N;
    out->n_units = nl->n_units;
    out->n_slots = nl->n_slots;
    out->n_entries = nl->n_entries;
    out->n_entries_padded = nl->n_entries_padded;
    out->n_pair_slots = nl->n_entries_padded * UNIT;
    out->list_bytes = nl->n_entries_padded * 6 + nl->n_units * 8;
    out->workspace_bytes = (int64_t)list_workspace_bytes(nl);
    for (int a = 0; a < 3; ++a) out->n_cells[a] = nl->grid.n[a];
    out->pbc_mode = nl->grid.pbc_mode;
    out->row_capacity = nl->row_cap;
    out->n_rebuild_grow = nl->n_grow;
    return DIMOS_OK;
}

DIMOS_API int64_t dimos_launch_count(const dimos_ctx* c)
{
    return c ? reinterpret_cast<const Ctx*>(c)->launches : 0;
}

DIMOS_API int dimos_probe_fp32_peak(dimos_ctx* c, double ms_target, double* tflops_host, void* stream)
{
    if (!c || !tflops_host) return DIMOS_EINVAL;
    Ctx* ctx = reinterpret_cast<Ctx*>(c);
    if (cudaSetDevice(ctx->device) != cudaSuccess) return set_error(ctx, DIMOS_ECUDA, "cudaSetDevice failed");
    return probe_fp32_impl(ctx, ms_target, tflops_host, (cudaStream_t)stream);
}

DIMOS_API const char* dimos_status_string(int status)
{
    switch (status) {
        case DIMOS_OK: return "DIMOS_OK";
        case DIMOS_EINVAL: return "DIMOS_EINVAL: invalid argument";
        case DIMOS_EBOX: return "DIMOS_EBOX: r_cut larger than half the box";
        case DIMOS_ENOMEM: return "DIMOS_ENOMEM: allocation failed";
        case DIMOS_EOVERFLOW: return "DIMOS_EOVERFLOW: internal capacity exceeded";
        case DIMOS_ECUDA: return "DIMOS_ECUDA: CUDA error or no CUDA device";
        case DIMOS_ESTALE: return "DIMOS_ESTALE: list does not match the arguments";
        default: return "unknown status";
    }
}

DIMOS_API const char* dimos_last_error(const dimos_ctx* c)
{
    return c ? reinterpret_cast<const Ctx*>(c)->err.c_str() : "";
}

DIMOS_API const char* dimos_version(void) { return "dimos_b200 0.1 (sm_100a)"; }

}  // extern "C"
