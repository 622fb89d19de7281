// pair_f32x2.cu -- A4 pair-force kernel, packed-FP32 version.
//
// Same work decomposition as the generic kernel in nonbonded.cu (one warp per unit of 8 i-atoms held in
// registers, one lane per j-atom of a 32-entry chunk, F_i in registers over the whole row, one vector RED per
// j-atom), but the arithmetic of two i-atoms is issued as ONE packed instruction (fma/add/mul.rn.f32x2 ->
// FFMA2 / FADD2 / FMUL2 on sm_100a).  FFMA2 has the FLOP rate of FFMA at half the issue slots (measured,
// profiles/r1_b_pair_force_ncu.md), so MUFU.RSQ, the cutoff FSETP/FSEL, loads and loop bookkeeping ride in the
// freed slots and the kernel is bound by the FMA pipe instead of by instruction issue.
//
// Covers: fp32 positions, fp32 accumulation (DIMOS_F32), image shift from the stencil code (pbc_mode 0), reaction
// field (Eq. 8) and Ewald real space (Eq. 10).  Everything else (fp64, mixed, per-pair minimum image) stays on the
// generic kernel.
//
// LJ is evaluated only in chunks in which at least one j-atom has LJ partners (warp vote) and, there, only for
// i-atom pairs with an LJ-active member; rows are reordered LJ-active-j-first after a build (reorder_rows_kernel
// below), which is an optimisation only: correctness never depends on the order.
#include <math.h>

#include "pair_common.cuh"

namespace dimos {

namespace {

constexpr int NPAIR = UNIT / 2;

__device__ __forceinline__ float rsqrt_f(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ float2 f2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ float2 bc(float a) { return make_float2(a, a); }

struct UnitRegs {
    float2 x[NPAIR], y[NPAIR], z[NPAIR], q[NPAIR];     // i-atoms (q pre-multiplied by k_e)
    float2 fx[NPAIR], fy[NPAIR], fz[NPAIR];            // F_i accumulators over the row
    float2 e_c, e_lj;                                  // per-lane energy partials
};

struct Consts {
    float rc2, krf, m2krf, mcrf;   // reaction field
    float alpha, two_a_sqrtpi;     // Ewald real space
    float rs, inv_sw;              // LJ switch, Eq. 6: r_s and 1/(r_c - r_s)
};

__device__ __forceinline__ float rcp_f(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float ex2_f(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// erfc(x) and exp(-x^2) for two values, x >= 0: erfc(x) = t (a1 + t (a2 + t (a3 + t (a4 + t a5)))) exp(-x^2),
// t = 1 / (1 + p x)  (Abramowitz & Stegun 7.1.26, |error| <= 1.5e-7 absolute), with MUFU.RCP / MUFU.EX2 for the
// reciprocal and the exponential and packed FMAs for the rest.
__device__ __forceinline__ void erfc_exp2(float2 x, float2& erfc_x, float2& exp_mx2)
{
    const float2 den = __ffma2_rn(bc(0.3275911f), x, bc(1.0f));
    const float2 t = f2(rcp_f(den.x), rcp_f(den.y));
    const float2 y = __fmul2_rn(__fmul2_rn(x, x), bc(-1.4426950408889634f));  // -x^2 log2(e)
    exp_mx2 = f2(ex2_f(y.x), ex2_f(y.y));
    float2 pl = __ffma2_rn(bc(1.061405429f), t, bc(-1.453152027f));
    pl = __ffma2_rn(pl, t, bc(1.421413741f));
    pl = __ffma2_rn(pl, t, bc(-0.284496736f));
    pl = __ffma2_rn(pl, t, bc(0.254829592f));
    erfc_x = __fmul2_rn(__fmul2_rn(pl, t), exp_mx2);
}

// One chunk: the lane's j-atom against the 8 i-atoms, two i-atoms per packed instruction.
//   MASKED: honour the entry's i-mask (exclusions, intra-unit half, padding); LJ: evaluate Eq. 4 for the
//   i-pairs flagged in lj_pairs.  Returns F_j = -sum_i fs_i * d_i.
template <int METHOD, bool SW, bool MASKED, bool LJ>
__device__ __forceinline__ void chunk_body(UnitRegs& u, const Consts& k, const float4* __restrict__ ljt, const int* __restrict__ ti, float nxj,
                                           float nyj, float nzj, float qj, int tj, unsigned mask, unsigned lj_pairs,
                                           float& sx, float& sy, float& sz)
{
    const float2 nx2 = bc(nxj), ny2 = bc(nyj), nz2 = bc(nzj), qj2 = bc(qj);
    const float2 krf2 = bc(k.krf), m2krf2 = bc(k.m2krf), mcrf2 = bc(k.mcrf);
    float2 ax = f2(0.f, 0.f), ay = f2(0.f, 0.f), az = f2(0.f, 0.f);
#pragma unroll
    for (int p = 0; p < NPAIR; ++p) {
        const float2 dx = __fadd2_rn(u.x[p], nx2);
        const float2 dy = __fadd2_rn(u.y[p], ny2);
        const float2 dz = __fadd2_rn(u.z[p], nz2);
        float2 r2 = __fmul2_rn(dx, dx);
        r2 = __ffma2_rn(dy, dy, r2);
        r2 = __ffma2_rn(dz, dz, r2);
        bool in_a = r2.x < k.rc2, in_b = r2.y < k.rc2;
        if (MASKED) {
            in_a = in_a && ((mask >> (2 * p)) & 1u);
            in_b = in_b && ((mask >> (2 * p + 1)) & 1u);
        }
        float2 rinv = f2(rsqrt_f(r2.x), rsqrt_f(r2.y));
        if (MASKED) {  // padding entries point at the unit itself (r = 0)
            rinv.x = in_a ? rinv.x : 0.f;
            rinv.y = in_b ? rinv.y : 0.f;
        }
        float2 qq = __fmul2_rn(u.q[p], qj2);
        qq.x = in_a ? qq.x : 0.f;
        qq.y = in_b ? qq.y : 0.f;
        const float2 rinvsq = __fmul2_rn(rinv, rinv);
        float2 fs;
        if (METHOD == DIMOS_RF) {
            // reaction field, Eq. 8 (reading C-1): e = qq (1/r + k_rf r^2 - c_rf);  f/r = qq (1/r^3 - 2 k_rf)
            float2 t = __ffma2_rn(krf2, r2, rinv);
            t = __fadd2_rn(t, mcrf2);
            u.e_c = __ffma2_rn(qq, t, u.e_c);
            const float2 g = __ffma2_rn(rinvsq, rinv, m2krf2);
            fs = __fmul2_rn(qq, g);
        } else {
            // Ewald real space, Eq. 10 with n = 0 (readings C-14): e = qq erfc(a r)/r;
            // f/r = qq [erfc(a r)/r + (2a/sqrt(pi)) exp(-a^2 r^2)] / r^2
            const float2 ar = __fmul2_rn(__fmul2_rn(r2, rinv), bc(k.alpha));
            float2 erfc_ar, ex;
            erfc_exp2(ar, erfc_ar, ex);
            const float2 qr = __fmul2_rn(qq, rinv);
            u.e_c = __ffma2_rn(qr, erfc_ar, u.e_c);
            const float2 g = __ffma2_rn(__fmul2_rn(qq, bc(k.two_a_sqrtpi)), ex, __fmul2_rn(qr, erfc_ar));
            fs = __fmul2_rn(g, rinvsq);
        }
        if (LJ) {
            if (lj_pairs & (1u << p)) {  // warp-uniform
                const float4 ca = ljt[ti[2 * p] + (tj & STYPE_MASK)], cb = ljt[ti[2 * p + 1] + (tj & STYPE_MASK)];  // c6, c12, 6 c6, 12 c12
                float2 rinv6 = __fmul2_rn(__fmul2_rn(rinvsq, rinvsq), rinvsq);
                rinv6.x = in_a ? rinv6.x : 0.f;
                rinv6.y = in_b ? rinv6.y : 0.f;
                const float2 e6 = __ffma2_rn(f2(ca.y, cb.y), rinv6, f2(-ca.x, -cb.x));   // c12 r^-6 - c6
                const float2 p6 = __ffma2_rn(f2(ca.w, cb.w), rinv6, f2(-ca.z, -cb.z));   // 12 c12 r^-6 - 6 c6
                if (!SW) {
                    u.e_lj = __ffma2_rn(e6, rinv6, u.e_lj);                               // Eq. 4
                    fs = __ffma2_rn(__fmul2_rn(p6, rinv6), rinvsq, fs);
                } else {
                    // Eq. 6: U_LJ -> S(x) U_LJ, x = (r - r_s)/(r_c - r_s) clamped at 0 (S(0) = 1, S'(0) = 0);
                    // r F = S (r F_LJ) - r S'(x)/(r_c - r_s) U_LJ
                    float2 elj = __fmul2_rn(e6, rinv6);
                    float2 flj = __fmul2_rn(p6, rinv6);
                    const float2 r = __fmul2_rn(r2, rinv);
                    float2 x = __fmul2_rn(__fadd2_rn(r, bc(-k.rs)), bc(k.inv_sw));
                    x = f2(fmaxf(x.x, 0.f), fmaxf(x.y, 0.f));
                    const float2 x2 = __fmul2_rn(x, x);
                    float2 S = __ffma2_rn(bc(-6.f), x, bc(15.f));
                    S = __ffma2_rn(S, x, bc(-10.f));
                    S = __ffma2_rn(S, __fmul2_rn(x2, x), bc(1.f));
                    const float2 xd = __fmul2_rn(x, __fadd2_rn(x, bc(-1.f)));             // x (x - 1)
                    const float2 dS = __fmul2_rn(__fmul2_rn(xd, xd), bc(-30.f * k.inv_sw)); // S'(x)/(r_c - r_s)
                    flj = __ffma2_rn(S, flj, __fmul2_rn(__fmul2_rn(dS, elj), f2(-r.x, -r.y)));
                    elj = __fmul2_rn(S, elj);
                    u.e_lj = __fadd2_rn(u.e_lj, elj);
                    fs = __ffma2_rn(flj, rinvsq, fs);
                }
            }
        }
        u.fx[p] = __ffma2_rn(fs, dx, u.fx[p]);
        u.fy[p] = __ffma2_rn(fs, dy, u.fy[p]);
        u.fz[p] = __ffma2_rn(fs, dz, u.fz[p]);
        const float2 nfs = f2(-fs.x, -fs.y);  // operand negation, no instruction
        ax = __ffma2_rn(nfs, dx, ax);
        ay = __ffma2_rn(nfs, dy, ay);
        az = __ffma2_rn(nfs, dz, az);
    }
    sx = ax.x + ax.y;
    sy = ay.x + ay.y;
    sz = az.x + az.y;
}


// One chunk of the software pipeline.  (j0, m0) are the list entries of chunk c and (PJ, TJ) its gathered j-atoms;
// (j1, m1) / (j2, m2) are the entries of chunks c+1 / c+2, loaded two and three steps before their coordinates are
// gathered.  The step loads the entries of chunk c+3, gathers chunk c+1 into the other coordinate buffer,
// evaluates chunk c and rotates the entry registers.  Reads past the row's last chunk stay inside the list
// allocation (LIST_SLACK) and their indices are clamped, so the pipeline needs no guards.
#define DIMOS_CHUNK_STEP(PJ, TJ, PJn, TJn, EOFF, C)                                                              \
    do {                                                                                                         \
        const int jc = j0;          /* rotate FIRST (old values), then load straight into the freed registers */ \
        const unsigned mk = m0;                                                                                  \
        j0 = j1; m0 = m1; j1 = j2; m1 = m2;                                                                      \
        j2 = jp[(EOFF) + 96];                                                                                    \
        m2 = mp[(EOFF) + 96];                                                                                    \
        {                                                                                                        \
            const unsigned jj = min((unsigned)j0, slot_max);                                                     \
            PJn = P.xyzq[jj];                                                                                    \
            TJn = P.stype[jj];                                                                                   \
        }                                                                                                        \
        const float4 off = off_s[mk >> 8];                                                                       \
        const float nxj = off.x - PJ.x, nyj = off.y - PJ.y, nzj = off.z - PJ.z; /* -(x_j + image shift) */       \
        float sx, sy, sz;                                                                                        \
        if ((unsigned)((C) - c_plain) < n_plain) { /* warp-uniform: full chunk of a full unit, all masks 0xFF */ \
            if (lj_pairs != 0u && __any_sync(FULL, (TJ & STYPE_ACTIVE) != 0))                                    \
                chunk_body<METHOD, SW, false, true>(u, k, ljt, ti_w, nxj, nyj, nzj, PJ.w, TJ, 0xFFu, lj_pairs, sx, sy, sz);  \
            else                                                                                                 \
                chunk_body<METHOD, SW, false, false>(u, k, ljt, ti_w, nxj, nyj, nzj, PJ.w, TJ, 0xFFu, 0u, sx, sy, sz);       \
        } else {                                                                                                 \
            chunk_body<METHOD, SW, true, true>(u, k, ljt, ti_w, nxj, nyj, nzj, PJ.w, TJ, mk & 0xFFu, lj_pairs, sx, sy, sz);  \
        }                                                                                                        \
        /* virial: x_j' (x) F_j in unit-local coordinates, x_j' = -nxj */                                        \
        w[0] = fmaf(-nxj, sx, w[0]); w[1] = fmaf(-nxj, sy, w[1]); w[2] = fmaf(-nxj, sz, w[2]);                   \
        w[3] = fmaf(-nyj, sy, w[3]); w[4] = fmaf(-nyj, sz, w[4]); w[5] = fmaf(-nzj, sz, w[5]);                   \
        red_add_xyz(P.Facc + jc, sx, sy, sz);                                                                    \
    } while (0)

template <int METHOD, bool SW>
__global__ __launch_bounds__(FX_WARPS * 32, FX_CTAS_PER_SM) void pair_force_f32x2_kernel(ForceParams<float> P)
{
    __shared__ float4 off_s[27];
    __shared__ int ti_s[FX_WARPS][UNIT];  // type * nt of the warp's current i-atoms
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    float4* ljt = reinterpret_cast<float4*>(dyn_smem);  // [nt*nt] (c6, c12, 6 c6, 12 c12)

    for (int t = threadIdx.x; t < P.nt * P.nt; t += blockDim.x) ljt[t] = P.lj4[t];
    if (threadIdx.x < 27) {  // NEGATED image offsets: the kernel works with -x_j
        const int c = threadIdx.x;
        off_s[c] = make_float4(-(float)(c / 9 - 1) * P.h[0], -(float)((c / 3) % 3 - 1) * P.h[1], -(float)(c % 3 - 1) * P.h[2], 0.f);
    }
    __syncthreads();  // the only CTA-wide barrier: warps are independent from here on

    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int wib = threadIdx.x >> 5;
    int* ti_w = ti_s[wib];
    const int comp = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);  // reduce8_scatter's element of this lane
    const unsigned slot_max = (unsigned)(P.n_slots - 1);
    double acc_d = 0.0;  // running fp64 total of component `comp` over all units of this warp
    Consts k;
    k.rc2 = P.rc2; k.krf = P.krf; k.m2krf = P.m2krf; k.mcrf = -P.crf;
    k.alpha = P.alpha; k.two_a_sqrtpi = P.two_a_sqrtpi;
    k.rs = P.rs; k.inv_sw = P.inv_sw;

    long long U = 0, U_next = 0;
    if (lane == 0) U = (long long)atomicAdd(P.unit_counter, 1ull);
    U = __shfl_sync(FULL, U, 0);

    while (U < P.n_units) {
        if (lane == 0) U_next = (long long)atomicAdd(P.unit_counter, 1ull);  // in flight while this unit is processed

        const int2 ri = P.row_info[U];
        const int total = ri.x & 0xFFFF;        // chunks in the row
        const int c_plain = 0;                  // the mask-free chunks come first ...
        const unsigned n_plain = (unsigned)ri.y;  // ... this many of them

        // pipeline prologue: indices of chunks 0 and 1, coordinates of chunk 0
        const int64_t e0 = U * (int64_t)P.row_cap + P.m_res + lane;
        const int* jp = P.jslot + e0;
        const unsigned short* mp = P.meta + e0;
        int j0 = jp[0], j1 = jp[32], j2 = jp[64];
        unsigned m0 = mp[0], m1 = mp[32], m2 = mp[64];
        float4 pA, pB;
        int tA, tB;
        {
            const unsigned jj = min((unsigned)j0, slot_max);
            pA = P.xyzq[jj];
            tA = P.stype[jj];
        }

        // ---- the unit's 8 i-atoms: lanes 0..7 load one each; shuffles broadcast them straight into register pairs ----
        UnitRegs u;
        float4 mine = make_float4(0.f, 0.f, 0.f, 0.f);
        int my_t = 0;
        if (lane < UNIT) { mine = P.xyzq[U * UNIT + lane]; my_t = P.stype[U * UNIT + lane]; }
        __syncwarp();
        if (lane < UNIT) ti_w[lane] = (my_t & STYPE_MASK) * P.nt;
        __syncwarp();
        const unsigned act_bits = __ballot_sync(FULL, (my_t & STYPE_ACTIVE) != 0) & 0xFFu;
        const unsigned act_or = act_bits | (act_bits >> 1);  // bit 2p: pair p has an LJ-active atom
        const unsigned lj_pairs = (act_or & 1u) | ((act_or >> 1) & 2u) | ((act_or >> 2) & 4u) | ((act_or >> 3) & 8u);
        mine.w *= P.ke;  // k_e folded into the i-side charge
#pragma unroll
        for (int p = 0; p < NPAIR; ++p) {
            u.x[p] = f2(__shfl_sync(FULL, mine.x, 2 * p), __shfl_sync(FULL, mine.x, 2 * p + 1));
            u.y[p] = f2(__shfl_sync(FULL, mine.y, 2 * p), __shfl_sync(FULL, mine.y, 2 * p + 1));
            u.z[p] = f2(__shfl_sync(FULL, mine.z, 2 * p), __shfl_sync(FULL, mine.z, 2 * p + 1));
            u.q[p] = f2(__shfl_sync(FULL, mine.w, 2 * p), __shfl_sync(FULL, mine.w, 2 * p + 1));
            u.fx[p] = u.fy[p] = u.fz[p] = f2(0.f, 0.f);
        }
        u.e_c = f2(0.f, 0.f);
        u.e_lj = f2(0.f, 0.f);
        float w[6] = {0, 0, 0, 0, 0, 0};

        // ---- the row, two chunks per iteration (ping-pong buffers A/B: no register rotation) ----
        for (int c = 0; c < total; c += 2) {
            DIMOS_CHUNK_STEP(pA, tA, pB, tB, 0, c);
            if (c + 1 < total) DIMOS_CHUNK_STEP(pB, tB, pA, tA, 32, c + 1);
            jp += 64;
            mp += 64;
        }

        // ---- F_i: reduce over the warp once per unit; lanes 0,4,..,28 end up holding one i-atom each ----
        float fix[UNIT], fiy[UNIT], fiz[UNIT];
#pragma unroll
        for (int p = 0; p < NPAIR; ++p) {
            fix[2 * p] = u.fx[p].x; fix[2 * p + 1] = u.fx[p].y;
            fiy[2 * p] = u.fy[p].x; fiy[2 * p + 1] = u.fy[p].y;
            fiz[2 * p] = u.fz[p].x; fiz[2 * p + 1] = u.fz[p].y;
        }
        const float rx = reduce8_scatter(fix, lane);
        const float ry = reduce8_scatter(fiy, lane);
        const float rz = reduce8_scatter(fiz, lane);
        if ((lane & 3) == 0) {
            P.Fown[U * UNIT + comp] = make_float4(rx, ry, rz, 0.f);
            const float4 v = P.xyzq[U * UNIT + comp];  // x_i (x) F_i^unit
            w[0] += v.x * rx; w[1] += v.x * ry; w[2] += v.x * rz;
            w[3] += v.y * ry; w[4] += v.y * rz; w[5] += v.z * rz;
        }
        double red[8] = {(double)u.e_lj.x + (double)u.e_lj.y, (double)u.e_c.x + (double)u.e_c.y,
                         (double)w[0], (double)w[1], (double)w[2], (double)w[3], (double)w[4], (double)w[5]};
        acc_d += reduce8_scatter(red, lane);

        U = __shfl_sync(FULL, U_next, 0);
    }

    const int64_t prow = ((int64_t)blockIdx.x * FX_WARPS + wib) * N_PART;
    if ((lane & 3) == 0) P.partials[prow + comp] = acc_d;
    if (lane == 1) P.partials[prow + 8] = 0.0;
}
#undef DIMOS_CHUNK_STEP

// Stable partition of every full unit's mask-free entries: j-atoms with LJ partners first.  After it, only the
// leading ~1/3 of a water row's chunks take the LJ path of the pair kernel (which still decides per chunk by a
// warp vote, so a stale order costs time, never correctness).
constexpr int RO_WARPS = 4;
__global__ __launch_bounds__(RO_WARPS * 32) void reorder_rows_kernel(int* __restrict__ jslot, unsigned short* __restrict__ meta,
                                                                     const int2* __restrict__ row_info,
                                                                     const int* __restrict__ stype, int64_t n_units,
                                                                     int row_cap, int m_res)
{
    extern __shared__ __align__(16) unsigned char ro_smem[];
    const int cap = row_cap - m_res;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int64_t U = (int64_t)blockIdx.x * RO_WARPS + wib;
    if (U >= n_units) return;
    int* sj = reinterpret_cast<int*>(ro_smem) + (size_t)wib * cap;
    unsigned short* sm = reinterpret_cast<unsigned short*>(reinterpret_cast<int*>(ro_smem) + (size_t)RO_WARPS * cap) + (size_t)wib * cap;
    const int2 ri = row_info[U];
    const int nu = ri.y * 32 < cap ? ri.y * 32 : cap;  // entries of the mask-free chunks (0 for a partial unit)
    if (nu == 0) return;
    const int64_t base = U * (int64_t)row_cap + m_res;
    const unsigned FULL = 0xffffffffu, lt = (1u << lane) - 1u;
    int n_act = 0;
    for (int k0 = 0; k0 < nu; k0 += 32) {
        const int k = k0 + lane;
        bool act = false;
        if (k < nu) {
            const int j = jslot[base + k];
            sj[k] = j;
            act = (stype[j] & STYPE_ACTIVE) != 0;
            sm[k] = (unsigned short)(meta[base + k] | (act ? 0x8000u : 0u));  // bit 15 is free: remember the flag
        }
        n_act += __popc(__ballot_sync(FULL, act));
    }
    __syncwarp();
    int pa = 0, pi = n_act;
    for (int k0 = 0; k0 < nu; k0 += 32) {
        const int k = k0 + lane;
        bool act = false, ina = false;
        int j = 0;
        unsigned short m = 0;
        if (k < nu) {
            j = sj[k];
            m = sm[k];
            act = (m & 0x8000u) != 0;
            ina = !act;
        }
        const unsigned ba = __ballot_sync(FULL, act), bi = __ballot_sync(FULL, ina);
        if (k < nu) {
            const int pos = act ? pa + __popc(ba & lt) : pi + __popc(bi & lt);
            jslot[base + pos] = j;
            meta[base + pos] = (unsigned short)(m & 0x7FFFu);
        }
        pa += __popc(ba);
        pi += __popc(bi);
    }
}

}  // namespace

void launch_reorder_rows(int* jslot, unsigned short* meta, const int2* row_info, const int* stype, int64_t n_units,
                         int row_cap, int m_res, cudaStream_t s)
{
    const size_t smem = (size_t)RO_WARPS * (row_cap - m_res) * 6;
    if (smem > 48 * 1024) cudaFuncSetAttribute(reorder_rows_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const unsigned nb = (unsigned)((n_units + RO_WARPS - 1) / RO_WARPS);
    reorder_rows_kernel<<<nb, RO_WARPS * 32, smem, s>>>(jslot, meta, row_info, stype, n_units, row_cap, m_res);
}

template <int METHOD, bool SW>
static void launch_one(const ForceParams<float>& P, unsigned nb, size_t dyn, cudaStream_t s)
{
    if (dyn > 48 * 1024)
        cudaFuncSetAttribute(pair_force_f32x2_kernel<METHOD, SW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn);
    pair_force_f32x2_kernel<METHOD, SW><<<nb, FX_WARPS * 32, dyn, s>>>(P);
}

bool launch_pair_force_f32x2(const ForceParams<float>& P, int method, unsigned nb, size_t dyn, cudaStream_t s)
{
    if (method == DIMOS_RF) {
        if (P.sw_on) launch_one<DIMOS_RF, true>(P, nb, dyn, s);
        else launch_one<DIMOS_RF, false>(P, nb, dyn, s);
    } else if (method == DIMOS_EWALD_REAL) {
        if (P.sw_on) launch_one<DIMOS_EWALD_REAL, true>(P, nb, dyn, s);
        else launch_one<DIMOS_EWALD_REAL, false>(P, nb, dyn, s);
    } else {
        return false;
    }
    return true;
}

}  // namespace dimos
