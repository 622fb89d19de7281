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
// field (Eq. 8) and Ewald real space (Eq. 10).  fp64 runs csrc/pair_f64.cu; mixed precision and per-pair minimum image
// stay on the generic kernel of nonbonded.cu.
//
// Data movement: a unit's row of list entries is staged in the warp's shared-memory buffer by a TMA bulk copy issued one
// unit ahead; the gathered j-atoms pass through per-lane shared-memory slots filled by cp.async two chunks ahead.
// LJ is evaluated only in the row's first two phases (the builder filed the j-atoms by the LJ activity of the last force
// call, see nl_build.cu) and, there, only for i-atom pairs with an LJ-active member; that order is an optimisation:
// gather_kernel checks the assumption against the real types and the kernel falls back to LJ everywhere.
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

__device__ __forceinline__ float4 lds_f4(unsigned addr)
{
    float4 v;
    asm("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

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
__device__ __forceinline__ void chunk_body(UnitRegs& u, const Consts& k, unsigned ljrow, const unsigned (&ti16)[UNIT], float nxj,
                                           float nyj, float nzj, float qj, unsigned mask, unsigned lj_pairs,
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
                // (c6, c12, 6 c6, 12 c12) of the two i-atoms with the lane's j-atom: ljrow = shared address of the table
                // column of the j-type, ti16 = byte offset of the i-type's row (warp-uniform)
                const float4 ca = lds_f4(ljrow + ti16[2 * p]), cb = lds_f4(ljrow + ti16[2 * p + 1]);
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


// ---- shared-memory / TMA helpers (explicit shared-space addresses) ----
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// list rows are read once per force call: evict-first in L2 so that the gathered j-atom coordinates (14.7 MB, re-read
// ~60 times) stay resident; the bulk copy bypasses L1 altogether
__device__ __forceinline__ unsigned long long policy_evict_first()
{
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void bulk_row_to_smem(unsigned dst, const void* src, unsigned bytes, unsigned bar, unsigned long long pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar), "l"(pol)
                 : "memory");
}
// gathers of the next chunk's j-atom: volatile asm so that neither the compiler's scheduler nor its register-pressure
// heuristics sink them below the arithmetic they are meant to overlap with
__device__ __forceinline__ float4 ldg_f4(const float4* p)
{
    float4 v;
    asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ int ldg_s32(const int* p)
{
    int v;
    asm volatile("ld.global.nc.s32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
// j-atom gather straight into shared memory (16 bytes per lane, cp.async): it holds no registers while in flight, so the
// register allocator cannot turn its destination into scratch for the chunk's arithmetic and push the load behind it
__device__ __forceinline__ void gather_to_smem(unsigned dst, const float4* p)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;\ncp.async.commit_group;" ::"r"(dst), "l"(p) : "memory");
}
__device__ __forceinline__ void gather_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void gather_wait_but_one() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }
__device__ __forceinline__ float4 lds_f4v(unsigned addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ unsigned lds_u32(unsigned addr)
{
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
// image offset of an entry from the CTA's shared table
__device__ __forceinline__ float4 lds_offset(unsigned base, unsigned w)
{
    float4 v;
    const unsigned addr = base + ((w >> (ENTRY_SLOT_BITS - 4)) & 0x1F0u);
    asm("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

// One chunk of the software pipeline.  The unit's row of packed entries (slot | code << 27) sits in the warp's
// shared-memory buffer (one TMA bulk copy per row, issued one unit ahead).  EC is the entry of chunk c and (PJ, TJ) its
// gathered j-atom; EN is the entry of chunk c+1.  The step gathers chunk c+1 into the other coordinate buffer,
// replaces EC by the entry of chunk c+2 (two entry registers, two coordinate buffers: nothing is copied at the loop
// back-edge), and evaluates chunk c.  Reads past the row's last chunk stay inside the buffer's slack and their slot
// is clamped, so the pipeline needs no guards.
//   A row is three phases (written that way by build_list), each with its own loop: KIND 0 = mask-free chunks whose j-atoms have LJ
//   partners, KIND 1 = chunks that read their i-masks (always with LJ), KIND 2 = mask-free chunks without LJ.  Only
//   phases 0 and 1 gather the j-atom types (for the chunk after them, too: harmless at the phase boundary).
#define DIMOS_CHUNK_STEP(KIND, GX, TJ, EC, SOFF)                                                                 \
    do {                                                                                                         \
        const float4 off = lds_offset(off_base, EC);                                                             \
        const float4 PJ = lds_f4v(GX);  /* landed: every step ends with gather_wait_but_one() */                 \
        const unsigned jc = EC & ENTRY_SLOT_MASK;                                                                \
        const unsigned ljrow = (KIND) != 2 ? ljt_base + ((unsigned)(TJ & STYPE_MASK) << 4) : 0u;                  \
        /* refill this parity's set for chunk c + 2: entry from the row buffer, j-atom into the slot's twin */   \
        EC = lds_u32(sa + (SOFF) + 256u);                                                                        \
        GX ^= 1024u;                                                                                             \
        {                                                                                                        \
            const unsigned jj = min(EC & ENTRY_SLOT_MASK, slot_max);                                             \
            gather_to_smem(GX, P.xyzq + jj);                                                                     \
            if ((KIND) != 2) TJ = ldg_s32(P.stype + jj);                                                         \
        }                                                                                                        \
        unsigned mk = 0xFFu;                                                                                     \
        if ((KIND) == 1) { mk = c_m < n_m_true ? mk_n : 0xFFu; mk_n = mp[32]; }                                  \
        const float nxj = off.x - PJ.x, nyj = off.y - PJ.y, nzj = off.z - PJ.z; /* -(x_j + image shift) */       \
        float sx, sy, sz;                                                                                        \
        chunk_body<METHOD, SW, (KIND) == 1, (KIND) != 2>(u, k, ljrow, ti16, nxj, nyj, nzj, PJ.w, mk, lj_pairs, sx, sy, sz);      \
        /* virial: x_j' (x) F_j in unit-local coordinates, x_j' = -nxj */                                        \
        w[0] = fmaf(-nxj, sx, w[0]); w[1] = fmaf(-nxj, sy, w[1]); w[2] = fmaf(-nxj, sz, w[2]);                   \
        w[3] = fmaf(-nyj, sy, w[3]); w[4] = fmaf(-nyj, sz, w[4]); w[5] = fmaf(-nzj, sz, w[5]);                   \
        red_add_xyz(P.Facc + jc, sx, sy, sz);                                                                    \
        gather_wait_but_one();  /* the next chunk's j-atom has landed; the one after it may still be in flight */ \
    } while (0)

// One unit's row into a shared-memory buffer: the chunks at the row's start (LJ-active and masked) and the chunks that
// end at the row's capacity (see row_chunk_offset) become one contiguous sequence; one or two bulk copies, one mbarrier.
__device__ __forceinline__ void copy_row(const ForceParams<float>& P, long long U, int2 ri, unsigned dst, unsigned bar, unsigned long long pol)
{
    const int total = ri.x & 0xFFFF;
    const int n_am = (ri.y & 0xFFFF) + (int)((unsigned)ri.y >> 16);
    const unsigned bytes1 = (unsigned)n_am * 128u, bytes2 = (unsigned)(total - n_am) * 128u;
    const unsigned* row = P.entry + U * (int64_t)P.row_cap + P.m_res;
    mbar_expect_tx(bar, bytes1 + bytes2);
    if (bytes1) bulk_row_to_smem(dst, row, bytes1, bar, pol);
    if (bytes2) bulk_row_to_smem(dst + bytes1, row + (P.row_cap - P.m_res) - (total - n_am) * 32, bytes2, bar, pol);
}

// after an odd number of chunks the even / odd register sets change roles
#define DIMOS_SWAP_SETS()                                               \
    do {                                                                \
        const unsigned g_ = gA; gA = gB; gB = g_;                       \
        const unsigned e_ = ea; ea = eb; eb = e_;                       \
        const int t_ = tA; tA = tB; tB = t_;                            \
    } while (0)

template <int METHOD, bool SW>
__global__ __launch_bounds__(FX_WARPS * 32, FX_CTAS_PER_SM) void pair_force_f32x2_kernel(ForceParams<float> P)
{
    __shared__ float4 off_s[32];
    __shared__ __align__(8) unsigned long long bars[FX_WARPS][2];
    __shared__ __align__(2048) float4 gat_s[FX_WARPS][4][32];  // four gathered-j-atom slots per lane: even chunks use 0 / 2, odd 1 / 3
    extern __shared__ __align__(128) unsigned char dyn_smem[];
    // dynamic shared memory: FX_WARPS x 2 row buffers of P.row_words words (128-byte aligned), then the LJ table
    float4* ljt = reinterpret_cast<float4*>(dyn_smem + (size_t)FX_WARPS * 2 * P.row_words * 4);  // [nt*nt] (c6, c12, 6 c6, 12 c12)

    if (P.skip != nullptr && *P.skip != 0) return;  // dimos_nb_params.skip_flag (the whole grid sees the same word)
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int wib = threadIdx.x >> 5;
    for (int t = threadIdx.x; t < P.nt * P.nt; t += blockDim.x) ljt[t] = P.lj4[t];
    if (threadIdx.x < 32) {  // NEGATED image offsets: the kernel works with -x_j
        const int c = threadIdx.x < 27 ? threadIdx.x : SELF_CODE;
        off_s[threadIdx.x] = make_float4(-(float)(c / 9 - 1) * P.h[0], -(float)((c / 3) % 3 - 1) * P.h[1], -(float)(c % 3 - 1) * P.h[2], 0.f);
    }
    const unsigned bar0 = smem_u32(&bars[wib][0]);
    if (lane == 0) {
        mbar_init(bar0, 1);
        mbar_init(bar0 + 8, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();  // the only CTA-wide barrier: warps are independent from here on

    const unsigned ljt_base = smem_u32(ljt);
    const int comp = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);  // reduce8_scatter's element of this lane
    const unsigned slot_max = (unsigned)(P.n_slots - 1);
    const unsigned long long pol_stream = policy_evict_first();
    const unsigned off_base = smem_u32(off_s);
    const unsigned row_bytes = (unsigned)P.row_words * 4u;
    const unsigned buf0 = smem_u32(dyn_smem) + (unsigned)wib * 2u * row_bytes;  // this warp's two row buffers
    const bool lj_all = *P.order_stale != 0;  // the LJ activity of some atom changed since the rows were ordered
    double acc_d = 0.0;  // running fp64 total of component `comp` over all units of this warp
    Consts k;
    k.rc2 = P.rc2; k.krf = P.krf; k.m2krf = P.m2krf; k.mcrf = -P.crf;
    k.alpha = P.alpha; k.two_a_sqrtpi = P.two_a_sqrtpi;
    k.rs = P.rs; k.inv_sw = P.inv_sw;

    // dynamic unit scheduling: every warp draws unit indices from one global counter (rows differ in length); the next
    // unit is claimed at the start of the current one, its row_info read after the first phase and its row copied
    // after the second, so that none of the three waits on the one before
    long long U = 0;
    if (lane == 0) U = (long long)atomicAdd(P.unit_counter, 1ull);
    U = __shfl_sync(FULL, U, 0);
    if (U >= P.n_units) {
        const int64_t prow0 = ((int64_t)blockIdx.x * FX_WARPS + wib) * N_PART;
        if (lane < N_PART) P.partials[prow0 + lane] = 0.0;
        return;
    }
    int2 ri = P.row_info[U];
    unsigned kbuf = 0;  // units processed by this warp: buffer = kbuf & 1
    unsigned phase = 0;  // bit b: parity of the next completion of buffer b's mbarrier (flips only when a row was copied into b:
                         // a unit without entries copies nothing and waits for nothing)
    if (lane == 0 && (ri.x & 0xFFFF) != 0) copy_row(P, U, ri, buf0, bar0, pol_stream);
    // pipeline state handed from one unit to the next: first two entries, first j-atom, the unit's own atoms
    unsigned ea = 0, eb = 0;
    unsigned gA = smem_u32(&gat_s[wib][0][lane]), gB = smem_u32(&gat_s[wib][1][lane]);  // slot of the current even / odd chunk's j-atom (^ 1024: its twin)
    int tA = 0, tB = 0;
    float4 mine = make_float4(0.f, 0.f, 0.f, 0.f);
    int my_t = 0;
    if ((ri.x & 0xFFFF) != 0) {
        mbar_wait(bar0, 0);
        phase ^= 1u;
        ea = lds_u32(buf0 + lane * 4u);
        eb = lds_u32(buf0 + lane * 4u + 128u);
        const unsigned ja = min(ea & ENTRY_SLOT_MASK, slot_max), jb = min(eb & ENTRY_SLOT_MASK, slot_max);
        gather_to_smem(gA, P.xyzq + ja);
        gather_to_smem(gB, P.xyzq + jb);
        tA = P.stype[ja];
        tB = P.stype[jb];
    }
    if (lane < UNIT) { mine = P.xyzq[U * UNIT + lane]; my_t = P.stype[U * UNIT + lane]; }

    while (true) {
        long long Un = 0;
        if (lane == 0) Un = (long long)atomicAdd(P.unit_counter, 1ull);  // in flight during the first phase
        const int total = ri.x & 0xFFFF;                  // chunks in the row
        const int n_a = ri.y & 0xFFFF;                  // mask-free chunks whose j-atoms were assumed LJ-active
        const int n_m_true = (int)((unsigned)ri.y >> 16);  // chunks after them that read their i-masks
        // lj_all (an atom assumed LJ-free turned out to have LJ partners): the trailing mask-free chunks go through the
        // masked-with-LJ loop as well, with all-ones masks
        const int n_m = lj_all ? total - n_a : n_m_true;
        const int n_b = total - n_a - n_m;                 // trailing mask-free chunks without LJ
        int c_m = 0;                                       // index inside the masked loop
        const unsigned b = kbuf & 1u;

        const unsigned char* mp = P.emask + U * (int64_t)P.row_cap + P.m_res + lane + n_a * 32;
        unsigned mk_n = mp[0];  // i-mask of the first masked chunk
        unsigned sa = buf0 + b * row_bytes + lane * 4u;  // shared address of this lane's entry of the current chunk

        // ---- the unit's 8 i-atoms: lanes 0..7 hold one each; shuffles broadcast them straight into register pairs ----
        UnitRegs u;
        unsigned ti16[UNIT];  // byte offset of every i-atom's row in the shared LJ table (warp-uniform)
#pragma unroll
        for (int i = 0; i < UNIT; ++i) ti16[i] = __shfl_sync(FULL, (unsigned)((my_t & STYPE_MASK) * P.nt) << 4, i);
        const unsigned act_bits = __ballot_sync(FULL, (my_t & STYPE_ACTIVE) != 0) & 0xFFu;
        const unsigned act_or = act_bits | (act_bits >> 1);  // bit 2p: pair p has an LJ-active atom
        const unsigned lj_pairs = (act_or & 1u) | ((act_or >> 1) & 2u) | ((act_or >> 2) & 4u) | ((act_or >> 3) & 8u);
        const float4 own = mine;  // kept for the virial term x_i (x) F_i
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
        gather_wait_all();  // the first two chunks' j-atoms, requested at the hand-off

        // ---- the row: three phases, two chunks per iteration (ping-pong entry registers and coordinate buffers; a
        //      phase with an odd number of chunks ends with one swap) ----
        for (int c = 0; c < n_a; c += 2) {
            DIMOS_CHUNK_STEP(0, gA, tA, ea, 0u);
            if (c + 1 < n_a) { DIMOS_CHUNK_STEP(0, gB, tB, eb, 128u); sa += 256u; }
            else { DIMOS_SWAP_SETS(); sa += 128u; }
        }
        Un = __shfl_sync(FULL, Un, 0);
        const bool more = Un < P.n_units;
        int2 ri_n = make_int2(0, 0);
        if (more) ri_n = P.row_info[Un];
        for (c_m = 0; c_m < n_m; ++c_m) {
            DIMOS_CHUNK_STEP(1, gA, tA, ea, 0u);
            DIMOS_SWAP_SETS();
            sa += 128u;
            mp += 32;
        }
        // the next unit's row: bulk copy into the other buffer (last read by the previous unit, which is finished)
        const int total_n = ri_n.x & 0xFFFF;
        __syncwarp();
        if (lane == 0 && total_n != 0) copy_row(P, Un, ri_n, buf0 + (b ^ 1u) * row_bytes, bar0 + 8u * (b ^ 1u), pol_stream);
        for (int c = 0; c < n_b; c += 2) {
            DIMOS_CHUNK_STEP(2, gA, tA, ea, 0u);
            if (c + 1 < n_b) { DIMOS_CHUNK_STEP(2, gB, tB, eb, 128u); }
            sa += 256u;
        }

        // ---- hand-off: the next unit's first two entries, its first j-atom and its own atoms are requested BEFORE this
        //      unit's reductions, so their latency is covered by the shuffles below ----
        float4 mine_n = make_float4(0.f, 0.f, 0.f, 0.f);
        int my_t_n = 0;
        if (more) {
            if (total_n != 0) {
                mbar_wait(bar0 + 8u * (b ^ 1u), (phase >> (b ^ 1u)) & 1u);
                phase ^= 1u << (b ^ 1u);
                const unsigned sn = buf0 + (b ^ 1u) * row_bytes + lane * 4u;
                ea = lds_u32(sn);
                eb = lds_u32(sn + 128u);
                const unsigned ja = min(ea & ENTRY_SLOT_MASK, slot_max), jb = min(eb & ENTRY_SLOT_MASK, slot_max);
                gather_wait_all();  // nothing of this row may still be landing in the slots
                gather_to_smem(gA, P.xyzq + ja);
                gather_to_smem(gB, P.xyzq + jb);
                tA = P.stype[ja];
                tB = P.stype[jb];
            }
            if (lane < UNIT) { mine_n = P.xyzq[Un * UNIT + lane]; my_t_n = P.stype[Un * UNIT + lane]; }
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
        const float vx = __shfl_sync(FULL, own.x, comp), vy = __shfl_sync(FULL, own.y, comp), vz = __shfl_sync(FULL, own.z, comp);
        if ((lane & 3) == 0) {
            P.Fown[U * UNIT + comp] = make_float4(rx, ry, rz, 0.f);
            w[0] += vx * rx; w[1] += vx * ry; w[2] += vx * rz;  // x_i (x) F_i^unit
            w[3] += vy * ry; w[4] += vy * rz; w[5] += vz * rz;
        }
        // energy / virial of this unit: per-lane fp32 partials -> fp32 warp sums -> fp64 running totals (reading C-11)
        float red[8] = {u.e_lj.x + u.e_lj.y, u.e_c.x + u.e_c.y, w[0], w[1], w[2], w[3], w[4], w[5]};
        acc_d += (double)reduce8_scatter(red, lane);

        if (!more) break;
        U = Un;
        ri = ri_n;
        mine = mine_n;
        my_t = my_t_n;
        ++kbuf;
    }

    const int64_t prow = ((int64_t)blockIdx.x * FX_WARPS + wib) * N_PART;
    if ((lane & 3) == 0) P.partials[prow + comp] = acc_d;
    if (lane == 1) P.partials[prow + 8] = 0.0;
}
#undef DIMOS_CHUNK_STEP
#undef DIMOS_SWAP_SETS

}  // namespace

template <int METHOD, bool SW>
static bool launch_one(const ForceParams<float>& P, unsigned nb, size_t dyn, cudaStream_t s)
{
    // Without the opt-in a CTA may use 48 KB of shared memory, STATIC + dynamic: the kernel's static part (gather slots,
    // offset table, barriers) is ~17 KB, so short rows (dyn of 25 .. 48 KB) need the attribute as well
    if (dyn > 24 * 1024 &&
        cudaFuncSetAttribute(pair_force_f32x2_kernel<METHOD, SW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    pair_force_f32x2_kernel<METHOD, SW><<<nb, FX_WARPS * 32, dyn, s>>>(P);
    return true;
}

// Returns false when the case is not covered (the caller then runs the generic kernel): an unknown method, or rows too
// long for the two shared-memory row buffers per warp.
bool launch_pair_force_f32x2(const ForceParams<float>& P_in, int method, unsigned nb, size_t lj_bytes, cudaStream_t s)
{
    ForceParams<float> P = P_in;
    P.row_words = ((P.row_cap - P.m_res) + 64 + 31) & ~31;  // two chunks of slack: the pipeline reads two chunks ahead
    const size_t dyn = (size_t)FX_WARPS * 2 * P.row_words * 4 + lj_bytes;
    if (dyn > 110 * 1024) return false;  // two CTAs per SM must fit
    if (method == DIMOS_RF) return P.sw_on ? launch_one<DIMOS_RF, true>(P, nb, dyn, s) : launch_one<DIMOS_RF, false>(P, nb, dyn, s);
    if (method == DIMOS_EWALD_REAL)
        return P.sw_on ? launch_one<DIMOS_EWALD_REAL, true>(P, nb, dyn, s) : launch_one<DIMOS_EWALD_REAL, false>(P, nb, dyn, s);
    return false;
}

}  // namespace dimos
