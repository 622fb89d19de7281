// pair_f64.cu -- A4 pair-force kernel for DIMOS_F64 contexts (BASELINE
// configs[0] and configs[4] in fp64).
//
// Same decomposition as the other pair kernels (one warp per unit of 8 i-atoms, one lane per j-atom of a 32-entry chunk,
// one vector of REDs per j-atom), but written for double precision, where one pair inside the cutoff costs a few hundred
// instructions (IEEE 1/sqrt, exp, the erfc series) and only 44 % of the listed pair slots are inside the cutoff:
//   pass 1  every lane tests its j-atom against the 8 i-atoms (distance only) and the warp writes the in-cutoff pairs of
//           the chunk, j-major, into a dense queue in shared memory;
//   pass 2  the queue is worked off 32 pairs at a time, one pair per lane, so that the expensive arithmetic runs on full
//           warps (~4 batches per chunk instead of 8 half-empty passes over the i-atoms).  F_i goes to a per-lane column
//           of a padded shared-memory array (summed once per unit), F_j through a segmented warp sum over the consecutive
//           lanes that hold the same j-atom.
// The i-atoms live in shared memory and the code is rolled: the unrolled generic kernel (nonbonded.cu) is 13,000
// instructions in fp64 and spends 95 % of its cycles waiting for instruction fetch (profiles/r2_f64_pair_force_ncu.md).
#include <math.h>

#include "pair_common.cuh"

namespace dimos {

namespace {

constexpr int F64_WARPS = 8;
constexpr int F64_PAD = 32;  // per-(i, component) row of 32 lane partials: a lane's column is its own bank whatever i it works on

__constant__ double CHEB[28] = {
#include "erfc_cheb.inc"
};
constexpr double CHEB_XMAX = 3.6;

// erfc(x) and exp(-x^2) for x >= 0 (see nonbonded.cu erfc_exp_r for the derivation of the series path)
__device__ __forceinline__ void erfc_exp(double x, bool fast, double& erfc_x, double& ex)
{
    if (!fast) {
        erfc_x = erfc(x);
        ex = exp(-x * x);
        return;
    }
    const double xc = fmin(x, CHEB_XMAX);
    ex = exp(-xc * xc);
    const double t2 = 2.0 * (2.0 * xc - CHEB_XMAX) / CHEB_XMAX;
    double b1 = 0.0, b2 = 0.0;
#pragma unroll
    for (int j = 27; j >= 1; --j) {
        const double b0 = fma(t2, b1, CHEB[j] - b2);
        b2 = b1;
        b1 = b0;
    }
    erfc_x = fma(0.5 * t2, b1, CHEB[0] - b2) * ex;
}

template <int METHOD, int PBC>
__global__ __launch_bounds__(F64_WARPS * 32, F64_MIN_CTAS) void pair_force_f64_kernel(ForceParams<double> P)
{
    __shared__ double4 off_s[27];
    __shared__ double4 iat_s[F64_WARPS][UNIT];  // the warp's current i-atoms: x, y, z, k_e q
    __shared__ int ti_s[F64_WARPS][UNIT];       // their LJ table row offset (type * nt), or -1 without LJ partners
    __shared__ double4 jat_s[F64_WARPS][32];    // the chunk's j-atoms (image-shifted x, y, z, q), one per lane
    __shared__ double fj_s[F64_WARPS][32 * 3];  // F_j of the chunk's j-atoms, summed over the batches
    __shared__ int tj_s[F64_WARPS][32];         // their types
    __shared__ double ftot_s[F64_WARPS][UNIT * 3];  // F_i of the unit, summed over the lanes' columns
    __shared__ unsigned char que_s[F64_WARPS][32 * UNIT];  // the chunk's in-cutoff pairs: j-lane << 3 | i
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    double4* ljt = reinterpret_cast<double4*>(dyn_smem);                          // [nt*nt] (c6, c12, 6 c6, 12 c12)
    double* facc = reinterpret_cast<double*>(ljt + P.nt * P.nt);                  // [F64_WARPS][UNIT*3][F64_PAD]

    if (P.skip != nullptr && *P.skip != 0) return;  // dimos_nb_params.skip_flag (the whole grid sees the same word)
    for (int t = threadIdx.x; t < P.nt * P.nt; t += blockDim.x) ljt[t] = P.lj4[t];
    if (threadIdx.x < 27) {
        const int c = threadIdx.x;
        off_s[c] = make_double4((double)(c / 9 - 1) * P.h[0], (double)((c / 3) % 3 - 1) * P.h[1], (double)(c % 3 - 1) * P.h[2], 0.0);
    }
    __syncthreads();  // the only CTA-wide barrier

    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int wib = threadIdx.x >> 5;
    double4* iat = iat_s[wib];
    int* tis = ti_s[wib];
    double4* jat = jat_s[wib];
    double* fjs = fj_s[wib];
    int* tjs = tj_s[wib];
    double* ftot = ftot_s[wib];
    unsigned char* que = que_s[wib];
    for (int k = lane; k < 32 * 3; k += 32) fjs[k] = 0.0;
    double* fw = facc + (size_t)wib * UNIT * 3 * F64_PAD;
    const bool lj_all = *P.order_stale != 0;
    const bool fast = P.erfc_fast != 0;
    double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};  // per-lane running sums over all units: E_lj, E_coul, Wxx, Wxy, Wxz, Wyy, Wyz, Wzz

    long long U = 0, U_next = 0;
    if (lane == 0) U = (long long)atomicAdd(P.unit_counter, 1ull);
    U = __shfl_sync(FULL, U, 0);

    while (U < P.n_units) {
        if (lane == 0) U_next = (long long)atomicAdd(P.unit_counter, 1ull);
        __syncwarp();
        if (lane < UNIT) {
            double4 v = P.xyzq[U * UNIT + lane];
            v.w *= P.ke;
            iat[lane] = v;
            const int t = P.stype[U * UNIT + lane] & STYPE_MASK;
            tis[lane] = P.row_active[t] ? t * P.nt : -1;
        }
        for (int k = lane; k < UNIT * 3 * F64_PAD; k += 32) fw[k] = 0.0;
        __syncwarp();

        const int2 ri = P.row_info[U];
        const int total = ri.x & 0xFFFF;
        const int n_a = ri.y & 0xFFFF;
        const unsigned n_m = (unsigned)ri.y >> 16;
        const int64_t e0 = U * (int64_t)P.row_cap + P.m_res + lane;
        const int n_am = n_a + (int)n_m, nu_cap = P.row_cap - P.m_res;
        unsigned jn = 0, mn = 0;
        if (total > 0) { const int64_t e = e0 + row_chunk_offset(0, total, n_am, nu_cap); jn = P.entry[e]; mn = P.emask[e]; }
        double4 pjn = make_double4(0, 0, 0, 0);
        int tjn = 0;
        if (total > 0) { pjn = P.xyzq[jn & ENTRY_SLOT_MASK]; tjn = P.stype[jn & ENTRY_SLOT_MASK] & STYPE_MASK; }

        for (int c = 0; c < total; ++c) {
            const int j = (int)(jn & ENTRY_SLOT_MASK);
            const unsigned code = jn >> ENTRY_SLOT_BITS;
            const bool plain = !((unsigned)(c - n_a) < n_m);
            const unsigned mask = plain ? 0xFFu : mn;
            const double4 pj = pjn;
            const int tj = tjn;
            if (c + 1 < total) {  // next chunk: entry, mask, then the gathered atom (its latency is covered by this chunk's math)
                const int64_t e = e0 + row_chunk_offset(c + 1, total, n_am, nu_cap);
                jn = P.entry[e];
                mn = P.emask[e];
                pjn = P.xyzq[jn & ENTRY_SLOT_MASK];
                tjn = P.stype[jn & ENTRY_SLOT_MASK] & STYPE_MASK;
            }
            const double4 off = off_s[code];
            const double xj = pj.x + off.x, yj = pj.y + off.y, zj = pj.z + off.z, qj = pj.w;
            const bool lj_chunk = lj_all || c < n_a + (int)n_m;
            // ---- pass 1 (cheap): which of the 8 i-atoms does this lane's j-atom have inside the cutoff ----
            unsigned bits = 0;
#pragma unroll
            for (int i = 0; i < UNIT; ++i) {
                const double4 a = iat[i];
                double dx = a.x - xj, dy = a.y - yj, dz = a.z - zj;
                if (PBC == 1) {
                    dx -= P.L[0] * rint(dx * P.invL[0]);
                    dy -= P.L[1] * rint(dy * P.invL[1]);
                    dz -= P.L[2] * rint(dz * P.invL[2]);
                }
                const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                bits |= (r2 < P.rc2 ? 1u : 0u) << i;
            }
            bits &= mask;
            // ---- the in-cutoff pairs of the chunk as a dense queue, j-major: entry = j-lane << 3 | i ----
            jat[lane] = make_double4(xj, yj, zj, qj);
            tjs[lane] = tj;
            const int cnt = __popc(bits);
            int o = cnt;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int y = __shfl_up_sync(FULL, o, d);
                if (lane >= d) o += y;
            }
            const int T = __shfl_sync(FULL, o, 31);
            o -= cnt;
            for (unsigned b = bits; b; b &= b - 1u) que[o++] = (unsigned char)((lane << 3) | (__ffs(b) - 1));
            __syncwarp();
            // ---- pass 2 (the expensive arithmetic): one pair per lane, 32 pairs per batch ----
            for (int q0 = 0; q0 < T; q0 += 32) {
                const int q = q0 + lane;
                const bool valid = q < T;
                const unsigned e = valid ? (unsigned)que[q] : 0u;
                const int i = (int)(e & 7u), jl = valid ? (int)(e >> 3) : 32 + lane;  // invalid lanes: a segment of their own
                const double4 a = iat[i];
                const double4 b = jat[jl & 31];
                double dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z;
                if (PBC == 1) {
                    dx -= P.L[0] * rint(dx * P.invL[0]);
                    dy -= P.L[1] * rint(dy * P.invL[1]);
                    dz -= P.L[2] * rint(dz * P.invL[2]);
                }
                double fs = 0.0;
                if (valid) {
                    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));  // the same expression as in pass 1: inside the cutoff
                    const double rinv = rsqrt(r2);  // 1 ulp (CUDA math library), far inside the 1e-10 bar
                    const double rinv2 = rinv * rinv;
                    const double qq = a.w * b.w;
                    double fr2;
                    if (METHOD == DIMOS_RF) {  // Eq. 8, reading C-1
                        acc[1] += qq * (fma(P.krf, r2, rinv) - P.crf);
                        fr2 = qq * fma(P.m2krf, r2, rinv);
                    } else {  // Eq. 10 with n = 0, reading C-14
                        const double r = r2 * rinv;
                        double erfc_ar, ex;
                        erfc_exp(P.alpha * r, fast, erfc_ar, ex);
                        const double qr = qq * rinv;
                        acc[1] += qr * erfc_ar;
                        fr2 = fma(qq * P.two_a_sqrtpi, ex, qr * erfc_ar);
                    }
                    const int ti = tis[i];
                    if (ti >= 0 && lj_chunk) {  // Eq. 4 (+ Eq. 6)
                        const double4 cc = ljt[ti + tjs[jl]];
                        const double rinv6 = rinv2 * rinv2 * rinv2;
                        double elj = fma(cc.y, rinv6, -cc.x) * rinv6;
                        double flj = fma(cc.w, rinv6, -cc.z) * rinv6;
                        if (P.sw_on) {
                            const double r_ = r2 * rinv;
                            const double x_ = (r_ - P.rs) * P.inv_sw;
                            if (x_ > 0.0) {
                                const double x2_ = x_ * x_, xm_ = x_ - 1.0;
                                const double S_ = fma(fma(fma(-6.0, x_, 15.0), x_, -10.0), x2_ * x_, 1.0);
                                const double dS_ = -30.0 * x2_ * xm_ * xm_ * P.inv_sw;
                                flj = S_ * flj - dS_ * elj * r_;
                                elj = S_ * elj;
                            }
                        }
                        acc[0] += elj;
                        fr2 += flj;
                    }
                    fs = fr2 * rinv2;
                }
                const double fx = fs * dx, fy = fs * dy, fz = fs * dz;
                if (valid) {  // F_i: this lane's own column of the i-atom's three rows
                    fw[(3 * i) * F64_PAD + lane] += fx;
                    fw[(3 * i + 1) * F64_PAD + lane] += fy;
                    fw[(3 * i + 2) * F64_PAD + lane] += fz;
                }
                if (PBC == 1) {  // the image can differ per pair: direct per-pair virial
                    acc[2] += dx * fx; acc[3] += dx * fy; acc[4] += dx * fz;
                    acc[5] += dy * fy; acc[6] += dy * fz; acc[7] += dz * fz;
                }
                // F_j: the pairs of one j-atom are consecutive lanes (at most 8): segmented sum, the segment's first lane adds
                // it to the j-atom's accumulator (one segment per j-atom and batch: plain read-modify-write)
                double sx = -fx, sy = -fy, sz = -fz;
#pragma unroll
                for (int d = 1; d < UNIT; d <<= 1) {
                    const int jo = __shfl_down_sync(FULL, jl, d);
                    const double tx = __shfl_down_sync(FULL, sx, d), ty = __shfl_down_sync(FULL, sy, d), tz = __shfl_down_sync(FULL, sz, d);
                    if (lane + d < 32 && jo == jl) { sx += tx; sy += ty; sz += tz; }
                }
                const int jprev = __shfl_up_sync(FULL, jl, 1);
                if (valid && (lane == 0 || jprev != jl)) {
                    fjs[3 * jl] += sx;
                    fjs[3 * jl + 1] += sy;
                    fjs[3 * jl + 2] += sz;
                }
                __syncwarp();  // a j-atom's segment can continue in the next batch
            }
            const double fjx = fjs[3 * lane], fjy = fjs[3 * lane + 1], fjz = fjs[3 * lane + 2];
            fjs[3 * lane] = 0.0; fjs[3 * lane + 1] = 0.0; fjs[3 * lane + 2] = 0.0;
            if (PBC == 0) {  // x_j' (x) F_j^entry in unit-local coordinates
                acc[2] = fma(xj, fjx, acc[2]); acc[3] = fma(xj, fjy, acc[3]); acc[4] = fma(xj, fjz, acc[4]);
                acc[5] = fma(yj, fjy, acc[5]); acc[6] = fma(yj, fjz, acc[6]); acc[7] = fma(zj, fjz, acc[7]);
            }
            if (mask) red_add_xyz(&P.Facc[j], fjx, fjy, fjz);
            __syncwarp();  // every lane is done with jat / tjs / que before the next chunk overwrites them
        }
        __syncwarp();
        // F_i of the unit: lane l < 24 sums row l (i = l / 3, component l % 3) of the padded array
        if (lane < UNIT * 3) {
            double s = 0.0;
            for (int k = 0; k < 32; ++k) s += fw[lane * F64_PAD + ((k + lane) & 31)];  // rotated: the rows' banks differ
            ftot[lane] = s;
        }
        __syncwarp();
        if (lane < UNIT) {
            const double rx = ftot[3 * lane], ry = ftot[3 * lane + 1], rz = ftot[3 * lane + 2];
            P.Fown[U * UNIT + lane] = make_double4(rx, ry, rz, 0.0);
            if (PBC == 0) {  // x_i (x) F_i^unit
                const double4 v = iat[lane];
                acc[2] += v.x * rx; acc[3] += v.x * ry; acc[4] += v.x * rz;
                acc[5] += v.y * ry; acc[6] += v.y * rz; acc[7] += v.z * rz;
            }
        }
        U = __shfl_sync(FULL, U_next, 0);
    }
    // one fp64 partial row per warp
    const double r = reduce8_scatter(acc, lane);
    const int comp = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
    const int64_t prow = ((int64_t)blockIdx.x * F64_WARPS + wib) * N_PART;
    if ((lane & 3) == 0) P.partials[prow + comp] = r;
    if (lane == 1) P.partials[prow + 8] = 0.0;
}

template <int METHOD, int PBC>
bool launch_one(const ForceParams<double>& P, unsigned nb, size_t dyn, cudaStream_t s)
{
    if (dyn > 16 * 1024 &&  // 48 KB without the opt-in, static (~23 KB) + dynamic
        cudaFuncSetAttribute(pair_force_f64_kernel<METHOD, PBC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    pair_force_f64_kernel<METHOD, PBC><<<nb, F64_WARPS * 32, dyn, s>>>(P);
    return true;
}

}  // namespace

// Returns false when the LJ table does not fit beside the accumulators (the caller then runs the generic kernel).
bool launch_pair_force_f64(const ForceParams<double>& P, int method, int pbc, unsigned nb, cudaStream_t s)
{
    static_assert(F64_WARPS == PF_WARPS, "the caller sizes the partial-sum rows with PF_WARPS");
    const size_t dyn = (size_t)P.nt * P.nt * sizeof(double4) + (size_t)F64_WARPS * UNIT * 3 * F64_PAD * sizeof(double);
    if (dyn > 100 * 1024) return false;
    if (method == DIMOS_RF) return pbc == 0 ? launch_one<DIMOS_RF, 0>(P, nb, dyn, s) : launch_one<DIMOS_RF, 1>(P, nb, dyn, s);
    if (method == DIMOS_EWALD_REAL) return pbc == 0 ? launch_one<DIMOS_EWALD_REAL, 0>(P, nb, dyn, s) : launch_one<DIMOS_EWALD_REAL, 1>(P, nb, dyn, s);
    return false;
}

}  // namespace dimos
