// nonbonded.cu -- per-step kernels.
//
//   A3  needs_rebuild: warp-reduced max of |pos - pos_at_build|^2.
//   gather: current positions -> cell-relative sorted float4 (x,y,z,q), LJ type, zeroed j-side force
//           accumulators; block 0 also converts the (sigma, eps) table to (c6, c12).
//   A4  pair_force (the generic kernel: DIMOS_MIXED, fp32 boxes with fewer than three cells per axis, rows or LJ tables too
//       large for the others; fp32 boxes otherwise run pair_f32x2.cu, DIMOS_F64 runs pair_f64.cu): one warp per unit of 8 i-atoms held in registers; every lane owns one j-atom of
//       a 32-wide chunk of the unit's list, evaluates it against the 8 i-atoms (LJ Eq. 4 + reaction
//       field Eq. 8, or + Ewald direct space Eq. 10), accumulates F_i in registers over the whole
//       row and F_j over the 8 slots, then issues ONE vector reduction (red.global.add.v4.f32) per
//       j-atom.  F_i is reduced across the warp once per unit by recursive halving shuffles.
//       Energy and virial are per-lane partial sums, reduced per warp, per block and finally in
//       fp64 (A6).  The virial uses W = sum_i x_i (x) F_i^unit + sum_entries x_j' (x) F_j^entry in
//       unit-local coordinates, so it costs 6 FMA per entry instead of 6 per pair.
//   A5  excl_correction: Ewald erf correction over the static exclusion list.
//   A6  finalize: F[orig] = F_own + F_acc, fp64 reduction of block partials, E[4], W[9].
#include <math.h>
#include <stdlib.h>

#include <string>
#include <type_traits>

#include "pair_common.cuh"
#include "trigger.cuh"

namespace dimos {

// rsqrt: one MUFU.RSQ in fp32 (2^-22.9 max relative error); IEEE-quality in fp64
__device__ __forceinline__ float rsqrt_r(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ double rsqrt_r(double x) { return 1.0 / sqrt(x); }
__device__ __forceinline__ float fma_r(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fma_r(double a, double b, double c) { return fma(a, b, c); }
// accumulate a*b into an accumulator that may be wider than the operands (DIMOS_MIXED: fp64 from the first add)
__device__ __forceinline__ float fma_acc(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fma_acc(float a, float b, double c) { return c + (double)(a * b); }
__device__ __forceinline__ double fma_acc(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float rintr(float x) { return rintf(x); }
__device__ __forceinline__ double rintr(double x) { return rint(x); }
__device__ __forceinline__ float erfc_r(float x) { return erfcf(x); }
__device__ __forceinline__ double erfc_r(double x) { return erfc(x); }
__device__ __forceinline__ float erf_r(float x) { return erff(x); }
__device__ __forceinline__ double erf_r(double x) { return erf(x); }
__device__ __forceinline__ float exp_r(float x) { return expf(x); }
__device__ __forceinline__ double exp_r(double x) { return exp(x); }

__constant__ double ERFC_CHEB[28] = {
#include "erfc_cheb.inc"
};
constexpr double ERFC_CHEB_XMAX = 3.6;
// erfc(x) and exp(-x^2), x >= 0.  fp64 with `fast`: erfc(x) = g(x) exp(-x^2), g = erfc(x) exp(x^2) from its degree-27
// Chebyshev series on [0, 3.6] (Clenshaw recurrence, 6e-16 relative; the host sets `fast` only when alpha r_cut <= 3.6, and
// larger arguments belong to slots beyond the cutoff, whose result is discarded: they are clamped).  One exp instead of
// libm's erfc + exp: the fp64 Ewald pair kernel spent most of its time there.
__device__ __forceinline__ void erfc_exp_r(float x, bool, float& erfc_x, float& ex)
{
    erfc_x = erfcf(x);
    ex = expf(-x * x);
}
__device__ __forceinline__ void erfc_exp_r(double x, bool fast, double& erfc_x, double& ex)
{
    if (!fast) {
        erfc_x = erfc(x);
        ex = exp(-x * x);
        return;
    }
    const double xc = fmin(x, ERFC_CHEB_XMAX);
    ex = exp(-xc * xc);
    const double t2 = 2.0 * (2.0 * xc - ERFC_CHEB_XMAX) / ERFC_CHEB_XMAX;  // 2 t, t in [-1, 1]
    double b1 = 0.0, b2 = 0.0;
#pragma unroll
    for (int j = 27; j >= 1; --j) {
        const double b0 = fma(t2, b1, ERFC_CHEB[j] - b2);
        b2 = b1;
        b1 = b0;
    }
    erfc_x = (fma(0.5 * t2, b1, ERFC_CHEB[0] - b2)) * ex;
}

// ------------------------------------------------------------------------------------------------
// A3: rebuild trigger
// ------------------------------------------------------------------------------------------------
template <typename real>
__global__ void needs_rebuild_kernel(const real* __restrict__ pos, const real* __restrict__ ref, int64_t N, real thr2,
                                     unsigned long long* __restrict__ state, int* __restrict__ flag)
{
    real m = 0;
    const int64_t n3 = 3 * N;
    // each thread handles whole atoms; consecutive threads read consecutive atoms (12-byte stride, coalesced)
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
        real dx = pos[3 * i] - ref[3 * i];
        real dy = pos[3 * i + 1] - ref[3 * i + 1];
        real dz = pos[3 * i + 2] - ref[3 * i + 2];
        real d2 = dx * dx + dy * dy + dz * dz;
        m = d2 > m ? d2 : m;
        if (!(d2 == d2)) m = (real)INFINITY;  // NaN -> force a rebuild
    }
    (void)n3;
    trigger_reduce_and_flag<real>(m, thr2, state, flag);
}

int needs_rebuild_impl(Ctx* ctx, const void* pos, const void* ref, int64_t N, double skin, int32_t* flag_dev, cudaStream_t s)
{
    int blocks = (int)((N + 255) / 256);
    int maxb = ctx->sm_count * 8;
    if (blocks > maxb) blocks = maxb;
    if (blocks < 1) blocks = 1;
    if (ctx->precision == DIMOS_F64) {
        double h = 0.5 * skin;
        needs_rebuild_kernel<double><<<blocks, 256, 0, s>>>((const double*)pos, (const double*)ref, N, h * h, next_trigger_state(ctx), flag_dev);
    } else {
        float h = 0.5f * (float)skin;
        needs_rebuild_kernel<float><<<blocks, 256, 0, s>>>((const float*)pos, (const float*)ref, N, h * h, next_trigger_state(ctx), flag_dev);
    }
    DIMOS_LAUNCH_CHECK(ctx, "needs_rebuild");
    return DIMOS_OK;
}

// ------------------------------------------------------------------------------------------------
// gather: caller-order inputs -> sorted, cell-relative device arrays
// ------------------------------------------------------------------------------------------------
template <typename real>
__global__ void gather_kernel(const real* __restrict__ pos, const real* __restrict__ charge, const int* __restrict__ type,
                              const int* __restrict__ perm, const double* __restrict__ ref, int64_t n_slots,
                              typename vec4<real>::type* __restrict__ xyzq, int* __restrict__ stype,
                              typename vec4<real>::type* __restrict__ Facc, const double* __restrict__ lj_table, int nt,
                              real* __restrict__ lj_out, int* __restrict__ row_active, double* __restrict__ accum,
                              int* __restrict__ order_stale, const unsigned char* __restrict__ slot_hint,
                              unsigned char* __restrict__ atom_active, const int* __restrict__ skip)
{
    if (skip != nullptr && *skip != 0) return;  // dimos_nb_params.skip_flag: the list is stale, the caller rebuilds and calls again
    // per type: does it have any non-zero LJ partner?  (every block recomputes the tiny table: no inter-block order)
    __shared__ int act_sh[MAX_TYPES];
    for (int t = threadIdx.x; t < nt; t += blockDim.x) {
        int act = 0;
        for (int u = 0; u < nt; ++u)
            if (lj_table[2 * (t * nt + u) + 1] != 0.0 && lj_table[2 * (t * nt + u)] != 0.0) act = 1;
        act_sh[t] = act;
    }
    __syncthreads();
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n_slots) {
        int o = perm[s];
        const bool pad = o < 0;
        if (pad) o = ~o;
        const double x = (double)pos[3 * (int64_t)o] - ref[3 * s];
        const double y = (double)pos[3 * (int64_t)o + 1] - ref[3 * s + 1];
        const double z = (double)pos[3 * (int64_t)o + 2] - ref[3 * s + 2];
        xyzq[s] = mk4((real)x, (real)y, (real)z, pad ? (real)0 : charge[o]);
        int t = type[o];
        if (t < 0 || t >= nt) {  // reported by the next synchronising call on this list; evaluated as type 0 meanwhile
            atomicOr(order_stale + 1, 1);
            t = 0;
        }
        const int st = t | (act_sh[t] ? STYPE_ACTIVE : 0);  // bit 30: the atom has LJ partners
        // the builder ordered the rows by the LJ activity it ASSUMED (the flags of the last force call before the build,
        // all active without one): an atom assumed LJ-free that has LJ partners would be skipped, so the pair kernels are
        // told to evaluate LJ in every chunk until the next build; the flag seen now is the next build's hint
        if (!pad) {
            if (!slot_hint[s] && (st & STYPE_ACTIVE)) atomicOr(order_stale, 1);
            atom_active[o] = (st & STYPE_ACTIVE) ? 1 : 0;
        }
        stype[s] = st;
        Facc[s] = mk4((real)0, (real)0, (real)0, (real)0);
    }
    if (blockIdx.x == 0) {
        // (sigma, eps) -> c6 = 4 eps sigma^6, c12 = 4 eps sigma^12, 6 c6, 12 c12  (Eq. 4)
        for (int k = threadIdx.x; k < nt * nt; k += blockDim.x) {
            double sg = lj_table[2 * k], ep = lj_table[2 * k + 1];
            double s2 = sg * sg, s6 = s2 * s2 * s2;
            const double c6 = 4.0 * ep * s6, c12 = 4.0 * ep * s6 * s6;
            lj_out[4 * k] = (real)c6;
            lj_out[4 * k + 1] = (real)c12;
            lj_out[4 * k + 2] = (real)(6.0 * c6);    // pre-scaled for the force: 24 eps [2 (s/r)^12 - (s/r)^6]
            lj_out[4 * k + 3] = (real)(12.0 * c12);
        }
        for (int t = threadIdx.x; t < nt; t += blockDim.x) row_active[t] = act_sh[t];
        if (threadIdx.x < 16) accum[threadIdx.x] = 0.0;
    }
}

// ------------------------------------------------------------------------------------------------
// A4: pair-force kernel
// ------------------------------------------------------------------------------------------------
// One pair slot (i-atom i of the unit  x  the lane's j-atom).  LJ: this i-atom has LJ partners
// (warp-uniform).  MASKED: honour the entry's i-mask bit.  All arithmetic is written as explicit
// FMAs so that one slot is ~24 (no LJ) / ~32 (LJ) issued instructions.
#define DIMOS_SLOT(i, LJ, MASKED)                                                                    \
    do {                                                                                             \
        const real dx = xi[i] - xj, dy = yi[i] - yj, dz = zi[i] - zj;                                \
        real ddx = dx, ddy = dy, ddz = dz;                                                           \
        if (PBC == 1) {                                                                              \
            ddx -= P.L[0] * rintr(ddx * P.invL[0]);                                                  \
            ddy -= P.L[1] * rintr(ddy * P.invL[1]);                                                  \
            ddz -= P.L[2] * rintr(ddz * P.invL[2]);                                                  \
        }                                                                                            \
        const real r2 = fma_r(ddz, ddz, fma_r(ddy, ddy, ddx * ddx));                                 \
        bool in = r2 < P.rc2;                                                                        \
        if (MASKED) in = in && ((mask >> i) & 1u);                                                   \
        real rinv = rsqrt_r(r2);                                                                     \
        if (LJ || MASKED || METHOD != DIMOS_RF) rinv = in ? rinv : (real)0;                          \
        const real qq = in ? qi[i] * qj : (real)0;                                                   \
        const real rinv2 = rinv * rinv;                                                              \
        real fr2;                                                                                    \
        if (METHOD == DIMOS_RF) {                                                                    \
            const real t = fma_r(P.krf, r2, rinv);              /* 1/r + k_rf r^2 */                 \
            e_c = fma_acc(qq, t - P.crf, e_c);                  /* Eq. 8 */                          \
            fr2 = qq * fma_r(P.m2krf, r2, rinv);                /* r^2 k_e qq (1/r^3 - 2 k_rf) */    \
        } else {                                                                                     \
            const real r = r2 * rinv;                                                                \
            const real ar = P.alpha * r;                                                             \
            real erfc_ar, ex;                                                                        \
            erfc_exp_r(ar, P.erfc_fast != 0, erfc_ar, ex);                                           \
            const real qr = qq * rinv;                                                               \
            e_c = fma_acc(qr, erfc_ar, e_c);                    /* Eq. 10, n = 0 */                  \
            fr2 = fma_r(qq * P.two_a_sqrtpi, ex, qr * erfc_ar);                                      \
        }                                                                                            \
        if (LJ) {                                                                                    \
            const real4 cc = ljt[ti[i] + tj];                   /* c6, c12, 6 c6, 12 c12 */          \
            const real rinv6 = rinv2 * rinv2 * rinv2;                                                \
            real elj = fma_r(cc.y, rinv6, -cc.x) * rinv6;       /* Eq. 4 */                          \
            real flj = fma_r(cc.w, rinv6, -cc.z) * rinv6;       /* r (-dU/dr) */                     \
            if (P.sw_on) {                                      /* Eq. 6: U -> S(x) U */             \
                const real r_ = r2 * rinv;                                                           \
                const real x_ = (r_ - P.rs) * P.inv_sw;                                              \
                if (x_ > (real)0) {                                                                  \
                    const real x2_ = x_ * x_, xm_ = x_ - (real)1;                                    \
                    const real S_ = fma_r(fma_r(fma_r((real)-6, x_, (real)15), x_, (real)-10), x2_ * x_, (real)1); \
                    const real dS_ = (real)-30 * x2_ * xm_ * xm_ * P.inv_sw;                         \
                    flj = S_ * flj - dS_ * elj * r_;                                                 \
                    elj = S_ * elj;                                                                  \
                }                                                                                    \
            }                                                                                        \
            e_lj = e_lj + (acc_t)elj;                                                                \
            fr2 += flj;                                                                              \
        }                                                                                            \
        const real fs = fr2 * rinv2;                                                                 \
        fix[i] = fma_r(fs, ddx, fix[i]); fiy[i] = fma_r(fs, ddy, fiy[i]); fiz[i] = fma_r(fs, ddz, fiz[i]); \
        fjx = fma_r(-fs, ddx, fjx); fjy = fma_r(-fs, ddy, fjy); fjz = fma_r(-fs, ddz, fjz);          \
        if (PBC == 1) { /* the image can differ per pair: direct per-pair virial */                  \
            const real fx = fs * ddx, fy = fs * ddy, fz = fs * ddz;                                  \
            w[0] += (acc_t)(ddx * fx); w[1] += (acc_t)(ddx * fy); w[2] += (acc_t)(ddx * fz);         \
            w[3] += (acc_t)(ddy * fy); w[4] += (acc_t)(ddy * fz); w[5] += (acc_t)(ddz * fz);         \
        }                                                                                            \
        if (E64 && in) { /* small fp32 box: the pair ENERGY in fp64 from the same fp32 inputs */     \
            double ex_ = (double)xi[i] - (double)xj, ey_ = (double)yi[i] - (double)yj, ez_ = (double)zi[i] - (double)zj; \
            ex_ -= P.d_L[0] * rint(ex_ / P.d_L[0]);                                                  \
            ey_ -= P.d_L[1] * rint(ey_ / P.d_L[1]);                                                  \
            ez_ -= P.d_L[2] * rint(ez_ / P.d_L[2]);                                                  \
            const double r2d_ = ex_ * ex_ + ey_ * ey_ + ez_ * ez_, rd_ = sqrt(r2d_);                 \
            const double qqd_ = (double)qraw[i] * (double)qj * P.d_ke;                               \
            if (METHOD == DIMOS_RF) e_c64 += qqd_ * (1.0 / rd_ + P.d_krf * r2d_ - P.d_crf);          \
            else e_c64 += qqd_ * erfc(P.d_alpha * rd_) / rd_;                                        \
            if (LJ) {                                                                                \
                const real4 cd_ = ljt[ti[i] + tj];                                                   \
                const double ri6_ = 1.0 / (r2d_ * r2d_ * r2d_);                                      \
                double el_ = ((double)cd_.y * ri6_ - (double)cd_.x) * ri6_;                          \
                if (P.sw_on) {                                                                       \
                    const double xs_ = (rd_ - P.d_rs) * P.d_inv_sw;                                  \
                    if (xs_ > 0.0) el_ *= 1.0 + xs_ * xs_ * xs_ * (-10.0 + xs_ * (15.0 - 6.0 * xs_)); \
                }                                                                                    \
                e_lj64 += el_;                                                                       \
            }                                                                                        \
        }                                                                                            \
    } while (0)

template <typename real, typename acc_t, int METHOD, int PBC>
__global__ __launch_bounds__(PF_WARPS * 32, sizeof(real) == 4 ? 2 : 1) void pair_force_kernel(ForceParams<real> P)
{
    using real4 = typename vec4<real>::type;
    __shared__ real4 off_s[27];
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    real4* ljt = reinterpret_cast<real4*>(dyn_smem);  // [nt*nt] (c6, c12, 6 c6, 12 c12)

    if (P.skip != nullptr && *P.skip != 0) return;  // dimos_nb_params.skip_flag (the whole grid sees the same word)
    for (int k = threadIdx.x; k < P.nt * P.nt; k += blockDim.x) ljt[k] = P.lj4[k];
    if (threadIdx.x < 27) {
        const int c = threadIdx.x;
        off_s[c] = mk4((real)(c / 9 - 1) * P.h[0], (real)((c / 3) % 3 - 1) * P.h[1], (real)(c % 3 - 1) * P.h[2], (real)0);
    }
    __syncthreads();  // the only CTA-wide barrier: warps are independent from here on

    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int wib = threadIdx.x >> 5;
    const int comp = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);  // reduce8_scatter's element of this lane
    double acc_d = 0.0;  // running fp64 total of component `comp` over all units of this warp
    // Boxes with fewer than three cells per axis (per-pair minimum image) are small: their energy is a sum that cancels
    // to ~1e-4 of the sum of magnitudes, below what fp32 pair terms resolve, so in fp32 mode the pair
    // ENERGY of such boxes is evaluated in fp64 from the same fp32 inputs; forces and virial stay fp32.
    constexpr bool E64 = PBC == 1 && sizeof(real) == 4 && sizeof(acc_t) == 4;
    const bool lj_all = *P.order_stale != 0;  // an atom became LJ-active after the rows were ordered: LJ in every chunk

    // dynamic unit scheduling: every warp draws unit indices from one global counter, so no warp
    // waits for another (rows differ in length) and the tail is at most one unit long
    long long U = 0, U_next = 0;
    if (lane == 0) U = (long long)atomicAdd(P.unit_counter, 1ull);
    U = __shfl_sync(FULL, U, 0);

    while (U < P.n_units) {
        if (lane == 0) U_next = (long long)atomicAdd(P.unit_counter, 1ull);  // in flight while this unit is processed

        // ---- the unit's 8 i-atoms in registers (uniform across the warp) ----
        real xi[UNIT], yi[UNIT], zi[UNIT], qi[UNIT], qraw[UNIT];
        int ti[UNIT];
        real fix[UNIT], fiy[UNIT], fiz[UNIT];
#pragma unroll
        for (int i = 0; i < UNIT; ++i) {
            const real4 v = P.xyzq[U * UNIT + i];
            xi[i] = v.x; yi[i] = v.y; zi[i] = v.z;
            qi[i] = v.w * P.ke;  // k_e folded into the i-side charge
            qraw[i] = v.w;
            const int t = P.stype[U * UNIT + i] & STYPE_MASK;
            ti[i] = P.row_active[t] ? t * P.nt : -1;
            fix[i] = fiy[i] = fiz[i] = 0;
        }
        const int2 ri = P.row_info[U];
        const int total = ri.x & 0xFFFF;  // chunks in the row
        const int n_a = ri.y & 0xFFFF;    // leading mask-free chunks ...
        const unsigned n_m = (unsigned)ri.y >> 16;  // ... then this many chunks that read their masks, then mask-free again
        acc_t e_lj = 0, e_c = 0;
        double e_lj64 = 0.0, e_c64 = 0.0;  // E64 only
        acc_t w[6] = {0, 0, 0, 0, 0, 0};

        // software pipeline: (jslot, meta) two chunks ahead, (xyzq, stype) one chunk ahead
        const int64_t e0 = U * (int64_t)P.row_cap + P.m_res + lane;
        const int n_am = n_a + (int)n_m, nu_cap = P.row_cap - P.m_res;
        unsigned jn = 0, jn2 = 0;  // packed entries
        int tjn = 0;
        unsigned mn = 0, mn2 = 0;  // i-masks
        real4 pjn = mk4((real)0, (real)0, (real)0, (real)0);
        if (total > 0) { const int64_t e = e0 + row_chunk_offset(0, total, n_am, nu_cap); jn = P.entry[e]; mn = P.emask[e]; }
        if (total > 1) { const int64_t e = e0 + row_chunk_offset(1, total, n_am, nu_cap); jn2 = P.entry[e]; mn2 = P.emask[e]; }
        if (total > 0) { pjn = P.xyzq[jn & ENTRY_SLOT_MASK]; tjn = P.stype[jn & ENTRY_SLOT_MASK] & STYPE_MASK; }

        for (int c = 0; c < total; ++c) {
            const int j = (int)(jn & ENTRY_SLOT_MASK);
            const unsigned code = jn >> ENTRY_SLOT_BITS;
            const unsigned m = mn;
            const real4 pj = pjn;
            const int tj = tjn;
            jn = jn2; mn = mn2;
            if (c + 1 < total) { pjn = P.xyzq[jn & ENTRY_SLOT_MASK]; tjn = P.stype[jn & ENTRY_SLOT_MASK] & STYPE_MASK; }
            if (c + 2 < total) { const int64_t e = e0 + row_chunk_offset(c + 2, total, n_am, nu_cap); jn2 = P.entry[e]; mn2 = P.emask[e]; }

            const real4 off = off_s[code];
            const real xj = pj.x + off.x, yj = pj.y + off.y, zj = pj.z + off.z;
            const real qj = pj.w;
            const bool plain = !((unsigned)(c - n_a) < n_m);  // warp-uniform: no mask needed
            const unsigned mask = plain ? 0xFFu : m;
            real fjx = 0, fjy = 0, fjz = 0;

            // the builder put the j-atoms assumed to have LJ partners in front of and inside the masked region
            const bool lj_chunk = lj_all || c < n_a + (int)n_m;
            if (plain) {
#pragma unroll
                for (int i = 0; i < UNIT; ++i) {
                    if (ti[i] >= 0 && lj_chunk) DIMOS_SLOT(i, true, false);
                    else DIMOS_SLOT(i, false, false);
                }
            } else {
#pragma unroll
                for (int i = 0; i < UNIT; ++i) {
                    if (ti[i] >= 0) DIMOS_SLOT(i, true, true);
                    else DIMOS_SLOT(i, false, true);
                }
            }
            if (PBC == 0) {  // x_j' (x) F_j^entry, unit-local coordinates
                w[0] = fma_acc(xj, fjx, w[0]); w[1] = fma_acc(xj, fjy, w[1]); w[2] = fma_acc(xj, fjz, w[2]);
                w[3] = fma_acc(yj, fjy, w[3]); w[4] = fma_acc(yj, fjz, w[4]); w[5] = fma_acc(zj, fjz, w[5]);
            }
            if (mask) red_add_xyz(&P.Facc[j], fjx, fjy, fjz);
        }

        // ---- F_i: reduce over the warp once per unit; lanes 0,4,..,28 end up holding one i-atom each ----
        const real rx = reduce8_scatter(fix, lane);
        const real ry = reduce8_scatter(fiy, lane);
        const real rz = reduce8_scatter(fiz, lane);
        if ((lane & 3) == 0) {
            P.Fown[U * UNIT + comp] = mk4(rx, ry, rz, (real)0);
            if (PBC == 0) {  // x_i (x) F_i^unit
                const real4 v = P.xyzq[U * UNIT + comp];
                w[0] += (acc_t)(v.x * rx); w[1] += (acc_t)(v.x * ry); w[2] += (acc_t)(v.x * rz);
                w[3] += (acc_t)(v.y * ry); w[4] += (acc_t)(v.y * rz); w[5] += (acc_t)(v.z * rz);
            }
        }
        // ---- energy / virial of this unit: lane partials -> fp64 warp totals, kept per warp ----
        double red[8] = {E64 ? e_lj64 : (double)e_lj, E64 ? e_c64 : (double)e_c, (double)w[0], (double)w[1], (double)w[2], (double)w[3], (double)w[4], (double)w[5]};
        acc_d += reduce8_scatter(red, lane);

        U = __shfl_sync(FULL, U_next, 0);
    }

    // one fp64 partial row per warp; the final reduction is finalize_kernel's (A6)
    const int64_t prow = ((int64_t)blockIdx.x * PF_WARPS + wib) * N_PART;
    if ((lane & 3) == 0) P.partials[prow + comp] = acc_d;
    if (lane == 1) P.partials[prow + 8] = 0.0;
}
#undef DIMOS_SLOT

// ------------------------------------------------------------------------------------------------
// A5: Ewald exclusion correction  -k_e q_i q_j erf(alpha r)/r over all excluded pairs (reading C-15)
// ------------------------------------------------------------------------------------------------
template <typename real>
__global__ void excl_correction_kernel(const int2* __restrict__ pairs, int64_t n_excl, const int* __restrict__ inv_perm,
                                       const typename vec4<real>::type* __restrict__ xyzq, const double* __restrict__ ref,
                                       typename vec4<real>::type* __restrict__ Facc, double* __restrict__ partials,
                                       real ke, real alpha, real two_a_sqrtpi, double Lx, double Ly, double Lz,
                                       const int* __restrict__ skip)
{
    if (skip != nullptr && *skip != 0) return;  // dimos_nb_params.skip_flag: the list is stale, the caller rebuilds and calls again
    using real4 = typename vec4<real>::type;
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double e = 0, w[6] = {0, 0, 0, 0, 0, 0};
    if (k < n_excl) {
        const int2 p = pairs[k];
        const int si = inv_perm[p.x], sj = inv_perm[p.y];
        const real4 a = xyzq[si], b = xyzq[sj];
        // raw-coordinate difference formed in fp64 from cell-relative parts, then nearest image (C-3)
        double ddx = ((double)a.x - (double)b.x) + (ref[3 * (int64_t)si] - ref[3 * (int64_t)sj]);
        double ddy = ((double)a.y - (double)b.y) + (ref[3 * (int64_t)si + 1] - ref[3 * (int64_t)sj + 1]);
        double ddz = ((double)a.z - (double)b.z) + (ref[3 * (int64_t)si + 2] - ref[3 * (int64_t)sj + 2]);
        ddx -= Lx * rint(ddx / Lx);
        ddy -= Ly * rint(ddy / Ly);
        ddz -= Lz * rint(ddz / Lz);
        const real dx = (real)ddx, dy = (real)ddy, dz = (real)ddz;
        const real r2 = dx * dx + dy * dy + dz * dz;
        const real rinv = (real)1 / sqrt(r2);
        const real r = r2 * rinv;
        const real qq = ke * a.w * b.w;
        const real erf_ar = erf_r(alpha * r);
        const real ex = exp_r(-(alpha * r) * (alpha * r));
        const real ee = -qq * erf_ar * rinv;
        const real fs = qq * (two_a_sqrtpi * ex - erf_ar * rinv) * rinv * rinv;
        const real fx = fs * dx, fy = fs * dy, fz = fs * dz;
        red_add_xyz(&Facc[si], fx, fy, fz);
        red_add_xyz(&Facc[sj], -fx, -fy, -fz);
        e = (double)ee;
        w[0] = (double)(dx * fx); w[1] = (double)(dx * fy); w[2] = (double)(dx * fz);
        w[3] = (double)(dy * fy); w[4] = (double)(dy * fz); w[5] = (double)(dz * fz);
    }
    // block reduction of 7 values
    __shared__ double sh[8][7];
    double v[7] = {e, w[0], w[1], w[2], w[3], w[4], w[5]};
#pragma unroll
    for (int q = 0; q < 7; ++q)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], o);
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5;
    if (lane == 0)
        for (int q = 0; q < 7; ++q) sh[wi][q] = v[q];
    __syncthreads();
    if (threadIdx.x < N_PART) {
        double sum = 0;
        int q = -1;
        if (threadIdx.x == 8) q = 0;                       // E_excl
        else if (threadIdx.x >= 2) q = threadIdx.x - 1;    // W components
        if (q >= 0)
            for (int ww = 0; ww < (int)(blockDim.x >> 5); ++ww) sum += sh[ww][q];
        partials[(int64_t)blockIdx.x * N_PART + threadIdx.x] = sum;
    }
}

// ------------------------------------------------------------------------------------------------
// 1-4 exceptions (reading C-21): s_lj U_LJ (Eq. 4) + s_c k_e q_i q_j / r (Eq. 7) over a static pair list
// ------------------------------------------------------------------------------------------------
template <typename real>
__global__ void exceptions_kernel(const int2* __restrict__ pairs, const double2* __restrict__ scale, int64_t n_exc,
                                  const int* __restrict__ inv_perm, const typename vec4<real>::type* __restrict__ xyzq,
                                  const int* __restrict__ stype, const double* __restrict__ ref,
                                  const double* __restrict__ lj_table, int nt,
                                  typename vec4<real>::type* __restrict__ Facc, double* __restrict__ partials, real ke,
                                  double Lx, double Ly, double Lz, const int* __restrict__ skip)
{
    if (skip != nullptr && *skip != 0) return;  // dimos_nb_params.skip_flag: the list is stale, the caller rebuilds and calls again
    using real4 = typename vec4<real>::type;
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double v[8] = {0, 0, 0, 0, 0, 0, 0, 0};  // E_lj, E_coul, Wxx, Wxy, Wxz, Wyy, Wyz, Wzz
    if (k < n_exc) {
        const int2 p = pairs[k];
        const double2 sc = scale[k];
        const int si = inv_perm[p.x], sj = inv_perm[p.y];
        const real4 a = xyzq[si], b = xyzq[sj];
        // raw-coordinate difference formed in fp64 from cell-relative parts, then nearest image (C-3)
        double ddx = ((double)a.x - (double)b.x) + (ref[3 * (int64_t)si] - ref[3 * (int64_t)sj]);
        double ddy = ((double)a.y - (double)b.y) + (ref[3 * (int64_t)si + 1] - ref[3 * (int64_t)sj + 1]);
        double ddz = ((double)a.z - (double)b.z) + (ref[3 * (int64_t)si + 2] - ref[3 * (int64_t)sj + 2]);
        ddx -= Lx * rint(ddx / Lx);
        ddy -= Ly * rint(ddy / Ly);
        ddz -= Lz * rint(ddz / Lz);
        const real dx = (real)ddx, dy = (real)ddy, dz = (real)ddz;
        const real r2 = dx * dx + dy * dy + dz * dz;
        const real rinv = (real)1 / sqrt(r2);
        const real rinv2 = rinv * rinv;
        const int ti = stype[si] & STYPE_MASK, tj = stype[sj] & STYPE_MASK;
        const double sg = lj_table[2 * (ti * nt + tj)], ep = lj_table[2 * (ti * nt + tj) + 1];
        const double s2 = sg * sg, s6 = s2 * s2 * s2;
        const real c6 = (real)(4.0 * ep * s6), c12 = (real)(4.0 * ep * s6 * s6);
        const real rinv6 = rinv2 * rinv2 * rinv2;
        const real e_lj = (real)sc.y * (c12 * rinv6 - c6) * rinv6;
        const real e_c = (real)sc.x * ke * a.w * b.w * rinv;
        const real fs = ((real)sc.y * ((real)12 * c12 * rinv6 - (real)6 * c6) * rinv6 + e_c) * rinv2;
        const real fx = fs * dx, fy = fs * dy, fz = fs * dz;
        red_add_xyz(&Facc[si], fx, fy, fz);
        red_add_xyz(&Facc[sj], -fx, -fy, -fz);
        v[0] = (double)e_lj; v[1] = (double)e_c;
        v[2] = (double)(dx * fx); v[3] = (double)(dx * fy); v[4] = (double)(dx * fz);
        v[5] = (double)(dy * fy); v[6] = (double)(dy * fz); v[7] = (double)(dz * fz);
    }
    __shared__ double sh[8][8];
#pragma unroll
    for (int q = 0; q < 8; ++q)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], o);
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5;
    if (lane == 0)
        for (int q = 0; q < 8; ++q) sh[wi][q] = v[q];
    __syncthreads();
    if (threadIdx.x < N_PART) {  // columns: E_lj, E_coul, W (6), E_excl
        double sum = 0;
        if (threadIdx.x < 8)
            for (int ww = 0; ww < (int)(blockDim.x >> 5); ++ww) sum += sh[ww][threadIdx.x];
        partials[(int64_t)blockIdx.x * N_PART + threadIdx.x] = sum;
    }
}

// setup-time check of a 1-4 exception list: indices in range, i < j, and every pair also in the exclusion list (C-21)
__global__ void check_exceptions_kernel(const int2* __restrict__ pairs, int64_t n_exc, int64_t N, const int* __restrict__ excl_start,
                                        const int* __restrict__ excl_adj, int* __restrict__ bad)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_exc) return;
    const int2 p = pairs[k];
    if (p.x < 0 || p.y < 0 || p.x >= N || p.y >= N || p.x >= p.y) { atomicOr(bad, 1); return; }
    bool found = false;
    for (int e = excl_start[p.x]; e < excl_start[p.x + 1]; ++e) found = found || excl_adj[e] == p.y;
    if (!found) atomicOr(bad, 2);
}

int check_exceptions_impl(Ctx* ctx, const NL* nl, const int32_t* pairs, int64_t n_exc, int* bad_dev, cudaStream_t s)
{
    check_exceptions_kernel<<<(unsigned)((n_exc + 255) / 256), 256, 0, s>>>((const int2*)pairs, n_exc, nl->N, (const int*)nl->excl_start.p,
                                                                            (const int*)nl->excl_adj.p, bad_dev);
    DIMOS_LAUNCH_CHECK(ctx, "check_exceptions");
    return DIMOS_OK;
}

// ------------------------------------------------------------------------------------------------
// A6: finalize
// ------------------------------------------------------------------------------------------------
template <typename real>
__global__ void finalize_kernel(const int* __restrict__ perm, int64_t n_slots,
                                const typename vec4<real>::type* __restrict__ Fown,
                                const typename vec4<real>::type* __restrict__ Facc, real* __restrict__ F,
                                const double* __restrict__ partials, int64_t n_part_rows, double* __restrict__ accum,
                                double* __restrict__ E, double* __restrict__ W, const int* __restrict__ skip)
{
    if (skip != nullptr && *skip != 0) return;  // dimos_nb_params.skip_flag: the list is stale, the caller rebuilds and calls again
    using real4 = typename vec4<real>::type;
    for (int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; s < n_slots; s += (int64_t)gridDim.x * blockDim.x) {
        const int o = perm[s];
        if (o >= 0) {
            const real4 a = Fown[s], b = Facc[s];
            F[3 * (int64_t)o] = a.x + b.x;
            F[3 * (int64_t)o + 1] = a.y + b.y;
            F[3 * (int64_t)o + 2] = a.z + b.z;
        }
    }
    // fp64 reduction of the block partials: thread t of every block sums a strided share of column t%9
    __shared__ double sh[256];
    __shared__ bool last;
    {
        const int col = threadIdx.x % N_PART;
        const int lanes_per_col = blockDim.x / N_PART;  // 28 for 256 threads
        const int sub = threadIdx.x / N_PART;
        double sum = 0;
        if (sub < lanes_per_col)
            for (int64_t r = (int64_t)blockIdx.x * lanes_per_col + sub; r < n_part_rows; r += (int64_t)gridDim.x * lanes_per_col)
                sum += partials[r * N_PART + col];
        sh[threadIdx.x] = sub < lanes_per_col ? sum : 0.0;
        __syncthreads();
        if (threadIdx.x < N_PART) {
            double t = 0;
            for (int k = 0; k < lanes_per_col; ++k) t += sh[k * N_PART + threadIdx.x];
            atomicAdd(&accum[threadIdx.x], t);
        }
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned long long* ticket = reinterpret_cast<unsigned long long*>(accum + 15);
            unsigned long long t = atomicAdd(ticket, 1ull);
            last = (t == (unsigned long long)gridDim.x - 1);
        }
        __syncthreads();
        if (last && threadIdx.x == 0) {
            __threadfence();
            volatile double* a = accum;
            const double elj = a[0], ec = a[1], eex = a[8];
            E[1] = elj; E[2] = ec; E[3] = eex; E[0] = elj + ec + eex;
            if (W) {
                W[0] = a[2]; W[1] = a[3]; W[2] = a[4];
                W[3] = a[3]; W[4] = a[5]; W[5] = a[6];
                W[6] = a[4]; W[7] = a[6]; W[8] = a[7];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// FP32 peak probe (roofline denominator for bench.py)
// ------------------------------------------------------------------------------------------------
__global__ void fma_probe_kernel(float* out, int iters, float a, float b)
{
    float r[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) r[k] = threadIdx.x * 0.001f + k;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 16; ++k) r[k] = fmaf(r[k], a, b);
    }
    float s = 0;
#pragma unroll
    for (int k = 0; k < 16; ++k) s += r[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

int probe_fp32_impl(Ctx* ctx, double ms_target, double* tflops, cudaStream_t s)
{
    const int blocks = ctx->sm_count * 8, thr = 256;
    float* out = nullptr;
    DIMOS_CUDA_TRY(ctx, cudaMalloc(&out, (size_t)blocks * thr * sizeof(float)));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    int iters = 2000;
    double best = 0;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0, s);
        fma_probe_kernel<<<blocks, thr, 0, s>>>(out, iters, 1.0001f, 0.5f);
        ctx->launches++;
        cudaEventRecord(e1, s);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaFree(out); return set_error(ctx, DIMOS_ECUDA, cudaGetErrorString(e)); }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        double tf = 2.0 * 16.0 * iters * (double)blocks * thr / (ms * 1e-3) * 1e-12;
        if (rep > 0 && tf > best) best = tf;
        if (rep == 0 && ms > 0) {  // scale the loop to the requested duration
            double want = ms_target > 0 ? ms_target : 2.0;
            double f = want / ms;
            iters = (int)(iters * (f < 0.1 ? 0.1 : (f > 50 ? 50 : f)));
            if (iters < 100) iters = 100;
        }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    *tflops = best;
    return DIMOS_OK;
}

// ------------------------------------------------------------------------------------------------
// host orchestration of one force call
// ------------------------------------------------------------------------------------------------
// packed-FP32 kernel (pair_f32x2.cu): fp32 accumulation, image shift from the stencil code;
// DIMOS_PAIR_KERNEL=generic disables it (A/B timing)
static bool use_f32x2(const Ctx* ctx, const NL* nl, int method)
{
    static const bool enabled = [] { const char* e = getenv("DIMOS_PAIR_KERNEL"); return !(e && std::string(e) == "generic"); }();
    return enabled && ctx->precision == DIMOS_F32 && nl->grid.pbc_mode == 0 && (method == DIMOS_RF || method == DIMOS_EWALD_REAL);
}

template <typename real, typename acc_t>
static int launch_pair_force(Ctx* ctx, const NL* nl, const ForceParams<real>& P, int method, unsigned nb, size_t dyn, cudaStream_t s)
{
    const int pbc = nl->grid.pbc_mode;
    cudaEvent_t ev_stop = nullptr;
    if (ctx->profiling && ctx->prof_used + 2 <= PROF_MAX_EVENTS) {  // per-kernel timing for bench.py's roofline
        while (ctx->prof_events.size() < ctx->prof_used + 2) {
            cudaEvent_t e;
            if (cudaEventCreate(&e) != cudaSuccess) return set_error(ctx, DIMOS_ECUDA, "cudaEventCreate failed");
            ctx->prof_events.push_back(e);
        }
        cudaEventRecord(ctx->prof_events[ctx->prof_used], s);
        ev_stop = ctx->prof_events[ctx->prof_used + 1];
        ctx->prof_used += 2;
    }
#define DIMOS_PF(M, B)                                                                                            \
    do {                                                                                                          \
        /* 48 KB without the opt-in, static (offset table, < 1 KB) + dynamic */                                   \
        if (dyn > 46 * 1024) cudaFuncSetAttribute(pair_force_kernel<real, acc_t, M, B>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn); \
        pair_force_kernel<real, acc_t, M, B><<<nb, PF_WARPS * 32, dyn, s>>>(P);                                   \
    } while (0)
    bool done = false;
    if constexpr (std::is_same<real, float>::value && std::is_same<acc_t, float>::value) {
        if (use_f32x2(ctx, nl, method)) done = launch_pair_force_f32x2(P, method, nb, dyn, s);
    }
    if constexpr (std::is_same<real, double>::value) {
        static const bool generic64 = [] { const char* e = getenv("DIMOS_PAIR_KERNEL"); return e && std::string(e) == "generic"; }();
        if (!generic64) done = launch_pair_force_f64(P, method, pbc, nb, s);
    }
    if (done) {}
    else if (method == DIMOS_RF) { if (pbc == 0) DIMOS_PF(DIMOS_RF, 0); else DIMOS_PF(DIMOS_RF, 1); }
    else { if (pbc == 0) DIMOS_PF(DIMOS_EWALD_REAL, 0); else DIMOS_PF(DIMOS_EWALD_REAL, 1); }
#undef DIMOS_PF
    if (ev_stop) cudaEventRecord(ev_stop, s);
    DIMOS_LAUNCH_CHECK(ctx, "pair_force");
    return DIMOS_OK;
}

template <typename real>
static int nonbonded_typed(Ctx* ctx, NL* nl, const real* pos, const real* charge, const int32_t* type,
                           const double* lj_table, int32_t nt, const dimos_nb_params* prm, real* F, double* E,
                           double* W, cudaStream_t s)
{
    using real4 = typename vec4<real>::type;
    int rc;
    const int64_t nsl = nl->n_slots, nun = nl->n_units;
    // persistent-style grid: at most 2 resident CTAs per SM (fp32; 1 for fp64), warps draw units dynamically
    const bool fx = sizeof(real) == 4 && use_f32x2(ctx, nl, prm->method);
    const int wpb = fx ? FX_WARPS : PF_WARPS;  // warps per CTA
    const unsigned nb_full = (unsigned)((nun + wpb - 1) / wpb);
    const unsigned nb_res = (unsigned)ctx->sm_count * (fx ? (unsigned)FX_CTAS_PER_SM : (sizeof(real) == 8 ? (unsigned)F64_MIN_CTAS : 2u));
    const unsigned nb_force = nb_full < nb_res ? nb_full : nb_res;
    const size_t n_force_rows = (size_t)nb_force * wpb;  // one fp64 partial row per warp
    const bool ewald = prm->method == DIMOS_EWALD_REAL;
    const unsigned nb_excl = ewald && nl->n_excl > 0 ? (unsigned)((nl->n_excl + 255) / 256) : 0;
    if ((rc = ensure(ctx, nl->xyzq, nsl * sizeof(real4), s))) return rc;
    if ((rc = ensure(ctx, nl->stype, nsl * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->atom_active, (size_t)nl->N, s))) return rc;
    if ((rc = ensure(ctx, nl->Facc, nsl * sizeof(real4), s))) return rc;
    if ((rc = ensure(ctx, nl->Fown, nsl * sizeof(real4), s))) return rc;
    if ((rc = ensure(ctx, nl->lj, (size_t)MAX_TYPES * MAX_TYPES * 4 * sizeof(double) + MAX_TYPES * sizeof(int), s))) return rc;
    const unsigned nb_exc = nl->n_exc > 0 ? (unsigned)((nl->n_exc + 255) / 256) : 0;
    if ((rc = ensure(ctx, nl->partials, (n_force_rows + (size_t)((nl->n_excl + 255) / 256) + nb_exc + 1) * N_PART * sizeof(double), s))) return rc;
    if ((rc = ensure(ctx, nl->accum, 16 * sizeof(double), s))) return rc;
    real* lj_dev = (real*)nl->lj.p;
    int* row_active = (int*)((char*)nl->lj.p + (size_t)MAX_TYPES * MAX_TYPES * 4 * sizeof(double));

    const int* skip = reinterpret_cast<const int*>(prm->skip_flag);
    const int T = 256;
    gather_kernel<real><<<(unsigned)((nsl + T - 1) / T), T, 0, s>>>(pos, charge, type, (const int*)nl->perm.p, (const double*)nl->ref.p,
                                                                    nsl, (real4*)nl->xyzq.p, (int*)nl->stype.p, (real4*)nl->Facc.p,
                                                                    lj_table, nt, lj_dev, row_active, (double*)nl->accum.p,
                                                                    (int*)nl->flags.p + 8, (const unsigned char*)nl->slot_hint.p,
                                                                    (unsigned char*)nl->atom_active.p, skip);
    DIMOS_LAUNCH_CHECK(ctx, "gather");
    // atom_active now holds this call's LJ-activity flags: the next build files its entries by them (a call that may be
    // skipped on the device proves nothing; the unconditional call after the rebuild does)
    if (skip == nullptr) nl->hint_valid = true;

    ForceParams<real> P;
    P.n_units = nun; P.n_slots = nsl; P.row_cap = nl->row_cap; P.m_res = nl->m_res; P.nt = nt;
    P.xyzq = (const real4*)nl->xyzq.p; P.stype = (const int*)nl->stype.p;
    P.entry = (const unsigned*)nl->entry.p; P.emask = (const unsigned char*)nl->emask.p; P.row_info = (const int2*)nl->row_info.p;
    P.lj4 = (const real4*)lj_dev; P.row_active = row_active; P.order_stale = (const int*)nl->flags.p + 8;
    P.skip = skip;
    P.unit_counter = reinterpret_cast<unsigned long long*>((double*)nl->accum.p + 14);
    P.Facc = (real4*)nl->Facc.p; P.Fown = (real4*)nl->Fown.p; P.partials = (double*)nl->partials.p;
    const double rc_ = prm->r_cut;
    P.rc2 = (real)rc_ * (real)rc_;
    P.ke = (real)prm->coulomb_const;
    P.krf = (real)((prm->eps_rf - 1.0) / ((2.0 * prm->eps_rf + 1.0) * rc_ * rc_ * rc_));  // Eq. 8 constants, reading C-1
    P.m2krf = (real)-2 * P.krf;
    P.crf = (real)(3.0 * prm->eps_rf / ((2.0 * prm->eps_rf + 1.0) * rc_));
    P.sw_on = (prm->r_switch > 0.0 && prm->r_switch < rc_) ? 1 : 0;  // Eq. 6; otherwise plain truncation (reading C-8)
    P.rs = (real)prm->r_switch;
    P.inv_sw = P.sw_on ? (real)(1.0 / (rc_ - prm->r_switch)) : (real)0;
    P.d_ke = prm->coulomb_const;
    P.d_krf = (prm->eps_rf - 1.0) / ((2.0 * prm->eps_rf + 1.0) * rc_ * rc_ * rc_);
    P.d_crf = 3.0 * prm->eps_rf / ((2.0 * prm->eps_rf + 1.0) * rc_);
    P.d_alpha = prm->alpha;
    P.d_rs = prm->r_switch;
    P.d_inv_sw = P.sw_on ? 1.0 / (rc_ - prm->r_switch) : 0.0;
    for (int a = 0; a < 3; ++a) P.d_L[a] = nl->grid.L[a];
    P.alpha = (real)prm->alpha;
    P.erfc_fast = (prm->alpha * rc_ <= ERFC_CHEB_XMAX) ? 1 : 0;
    P.two_a_sqrtpi = (real)(2.0 * prm->alpha / sqrt(M_PI));
    for (int a = 0; a < 3; ++a) { P.L[a] = (real)nl->grid.L[a]; P.invL[a] = (real)(1.0 / nl->grid.L[a]); P.h[a] = (real)nl->grid.h[a]; }
    const size_t dyn = (size_t)nt * nt * sizeof(real4);
    if (ctx->precision == DIMOS_MIXED) { if ((rc = launch_pair_force<real, double>(ctx, nl, P, prm->method, nb_force, dyn, s))) return rc; }
    else { if ((rc = launch_pair_force<real, real>(ctx, nl, P, prm->method, nb_force, dyn, s))) return rc; }

    if (nb_excl) {
        excl_correction_kernel<real><<<nb_excl, 256, 0, s>>>((const int2*)nl->excl_pairs.p, nl->n_excl, (const int*)nl->inv_perm.p,
                                                              (const real4*)nl->xyzq.p, (const double*)nl->ref.p, (real4*)nl->Facc.p,
                                                              (double*)nl->partials.p + n_force_rows * N_PART, P.ke, P.alpha,
                                                              P.two_a_sqrtpi, nl->grid.L[0], nl->grid.L[1], nl->grid.L[2], skip);
        DIMOS_LAUNCH_CHECK(ctx, "excl_correction");
    }
    if (nb_exc) {
        exceptions_kernel<real><<<nb_exc, 256, 0, s>>>((const int2*)nl->exc_pairs.p, (const double2*)nl->exc_scale.p, nl->n_exc,
                                                        (const int*)nl->inv_perm.p, (const real4*)nl->xyzq.p, (const int*)nl->stype.p,
                                                        (const double*)nl->ref.p, lj_table, nt, (real4*)nl->Facc.p,
                                                        (double*)nl->partials.p + (n_force_rows + nb_excl) * N_PART, P.ke,
                                                        nl->grid.L[0], nl->grid.L[1], nl->grid.L[2], skip);
        DIMOS_LAUNCH_CHECK(ctx, "exceptions");
    }
    int fb = (int)((nsl + T - 1) / T);
    const int maxfb = ctx->sm_count * 8;
    if (fb > maxfb) fb = maxfb;
    if (fb < 1) fb = 1;
    finalize_kernel<real><<<fb, T, 0, s>>>((const int*)nl->perm.p, nsl, (const real4*)nl->Fown.p, (const real4*)nl->Facc.p, F,
                                           (const double*)nl->partials.p, (int64_t)n_force_rows + nb_excl + nb_exc, (double*)nl->accum.p, E, W, skip);
    DIMOS_LAUNCH_CHECK(ctx, "finalize");
    return DIMOS_OK;
}

int nonbonded_impl(Ctx* ctx, NL* nl, const void* pos, const void* charge, const int32_t* type, const double* lj_table,
                   int32_t ntypes, const dimos_nb_params* prm, void* F, double* E, double* virial, cudaStream_t s)
{
    if (ctx->precision == DIMOS_F64)
        return nonbonded_typed<double>(ctx, nl, (const double*)pos, (const double*)charge, type, lj_table, ntypes, prm,
                                       (double*)F, E, virial, s);
    return nonbonded_typed<float>(ctx, nl, (const float*)pos, (const float*)charge, type, lj_table, ntypes, prm, (float*)F, E,
                                  virial, s);
}

}  // namespace dimos
