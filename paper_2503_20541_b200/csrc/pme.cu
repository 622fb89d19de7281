// pme.cu -- reciprocal-space electrostatics by smooth particle-mesh Ewald (Eq. 11,
// PAPER.md:227 Eq. 12, "we implement smooth PME ... B-splines based on the recursive definition").
//
//   pme_spread   one warp per 32 atoms: every lane computes the scaled fractional coordinate (fp64 from the raw position, so
//                the spline argument is exact to the rounding of `real`) and the 3 x n cardinal B-spline weights of its
//                atom by the recursion; the warp then adds q * w1 w2 w3 to the n^3 mesh points of one atom after the other,
//                points dealt to the lanes with z (contiguous in memory) fastest
//   cuFFT        real-to-complex 3-D transform of the charge mesh (library call; SURVEY.md §8(f) 3 names it)
//   pme_solve    per wave vector: B(m) C(m), energy 1/2 B C |F(Q)|^2, virial, F(Q) *= B C  (half spectrum, weights 1 / 2)
//   cuFFT        complex-to-real transform: the convolution theta_rec * Q
//   pme_gather   same decomposition: F_i = -q_i sum_k grad(theta_i)(k) (theta_rec * Q)(k)
//   pme_self     Eq. 12: -k_e alpha / sqrt(pi) sum q^2
//
// The mesh is indexed [k1][k2][k3] with k3 fastest.  Energies and virial are reduced in fp64.
#include <cufft.h>
#include <math.h>

#include <vector>

#include "common.cuh"

namespace dimos {

struct PmePlan {
    int K[3] = {0, 0, 0};
    int order = 0;
    bool dbl = false;
    cufftHandle fwd = 0, inv = 0;
    bool have_plans = false;
    DevBuf grid;     // real[K1*K2*K3]
    DevBuf spec;     // complex[K1*K2*(K3/2+1)]
    DevBuf moduli;   // double[K1+K2+K3]: |b(m)|^2 per axis
    DevBuf tables;   // double[2*(K1+K2+K3)]: per axis {m_k, |b|^2 exp(-pi^2 m_k^2/alpha^2)} for the alpha and box below
    double tab_alpha = 0, tab_L[3] = {0, 0, 0};
    DevBuf work;     // cuFFT work area (shared by both plans)
    DevBuf acc;      // double[8]: E_recip, Wxx, Wxy, Wxz, Wyy, Wyz, Wzz, sum q^2
};

namespace {

constexpr int PME_MAX_ORDER = 6;

// cardinal B-spline weights M_n(w + j), j = 0..n-1, and their derivatives, by the recursion of Essmann et al. Eq. 4.1/4.2
template <typename real, int N>
__device__ __forceinline__ void bspline_weights(real w, real (&th)[PME_MAX_ORDER], real (&dth)[PME_MAX_ORDER])
{
    // order 2 on the two support points: M_2(w) = w, M_2(w + 1) = 1 - w; build up to order N - 1, differentiate, then order N
    real a[PME_MAX_ORDER];
#pragma unroll
    for (int j = 0; j < PME_MAX_ORDER; ++j) a[j] = (real)0;
    a[0] = w;
    a[1] = (real)1 - w;
#pragma unroll
    for (int k = 3; k <= N; ++k) {
        if (k == N) {  // dM_N(u) = M_{N-1}(u) - M_{N-1}(u - 1) at u = w + j
#pragma unroll
            for (int j = 0; j < N; ++j) dth[j] = a[j] - (j > 0 ? a[j - 1] : (real)0);
        }
        const real inv = (real)1 / (real)(k - 1);
        // M_k(w + j) = (w + j)/(k-1) M_{k-1}(w + j) + (k - w - j)/(k-1) M_{k-1}(w + j - 1)
#pragma unroll
        for (int j = k - 1; j >= 0; --j) {
            const real u = w + (real)j;
            const real prev = j > 0 ? a[j - 1] : (real)0;
            a[j] = inv * (u * a[j] + ((real)k - u) * prev);
        }
    }
    if (N == 2) {
        dth[0] = (real)1;
        dth[1] = (real)-1;
    }
#pragma unroll
    for (int j = 0; j < N; ++j) th[j] = a[j];
}

template <typename real>
__device__ __forceinline__ void scaled_fraction(const real* __restrict__ pos, int64_t i, int a, double L, int K, int& fl, real& w)
{
    double x = (double)pos[3 * i + a];
    if (!isfinite(x)) x = 0.0;
    double f = x / L;
    f -= floor(f);
    const double u = f * K;
    int k = (int)u;
    if (k >= K) k = K - 1;
    fl = k;
    w = (real)(u - (double)k);
}

// Spread and gather: one warp per 32 consecutive atoms.  First every lane computes the spline weights of ITS atom (3 axes,
// the recursion runs for 32 atoms at once) and leaves them in the warp's shared-memory table; then the warp walks over its
// atoms one after the other with the N^3 mesh points of the atom dealt to the lanes, z (contiguous in memory) fastest, so
// that the N points of a mesh row sit in adjacent lanes: one warp-wide RED / load touches ~32/N rows instead of 32.
constexpr int PME_WARPS = 4;

template <typename real, int N, bool DERIV>
struct PmeWarpTable {
    real th[32][3][N];                   // [atom of the warp][axis][j]: a lane's stores have the odd stride 3 N
    real dth[DERIV ? 32 : 1][3][N];
};

template <typename real, int N, bool DERIV>
__device__ __forceinline__ void pme_warp_weights(const real* __restrict__ pos, int64_t i, bool have, double Lx, double Ly, double Lz,
                                                 int K1, int K2, int K3, PmeWarpTable<real, N, DERIV>& tab, int lane, int& f1, int& f2,
                                                 int& f3)
{
    f1 = f2 = f3 = 0;
    if (have) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const double L = a == 0 ? Lx : (a == 1 ? Ly : Lz);
            const int K = a == 0 ? K1 : (a == 1 ? K2 : K3);
            int fl;
            real w;
            scaled_fraction(pos, i, a, L, K, fl, w);
            real t[PME_MAX_ORDER], d[PME_MAX_ORDER];
            bspline_weights<real, N>(w, t, d);
#pragma unroll
            for (int j = 0; j < N; ++j) {
                tab.th[lane][a][j] = t[j];
                if (DERIV) tab.dth[lane][a][j] = d[j];
            }
            if (a == 0) f1 = fl; else if (a == 1) f2 = fl; else f3 = fl;
        }
    }
    __syncwarp();
}

template <typename real, int N>
__global__ __launch_bounds__(PME_WARPS * 32) void pme_spread_kernel(const real* __restrict__ pos, const real* __restrict__ charge,
                                                                     int64_t n_atoms, double Lx, double Ly, double Lz, int K1, int K2,
                                                                     int K3, real* __restrict__ grid)
{
    __shared__ PmeWarpTable<real, N, false> tabs[PME_WARPS];
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int64_t a0 = (((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5) * 32;
    if (a0 >= n_atoms) return;  // whole warps leave; there is no block-wide barrier
    const int cnt = (int)((n_atoms - a0) < 32 ? (n_atoms - a0) : 32);
    PmeWarpTable<real, N, false>& tab = tabs[wib];
    int f1m, f2m, f3m;
    pme_warp_weights<real, N, false>(pos, a0 + lane, lane < cnt, Lx, Ly, Lz, K1, K2, K3, tab, lane, f1m, f2m, f3m);
    const real qm = lane < cnt ? charge[a0 + lane] : (real)0;
    // this lane's mesh points inside an atom's N^3 block do not depend on the atom: decompose the point indices once
    constexpr int NP = N * N * N, NIT = (NP + 31) / 32;
    int j1[NIT], j2[NIT], j3[NIT];
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
        const int p = it * 32 + lane, j12 = p / N;
        j3[it] = p - j12 * N;
        j1[it] = j12 / N;
        j2[it] = j12 - j1[it] * N;
    }
    for (int a = 0; a < cnt; ++a) {
        const int f1 = __shfl_sync(FULL, f1m, a), f2 = __shfl_sync(FULL, f2m, a), f3 = __shfl_sync(FULL, f3m, a);
        const real q = __shfl_sync(FULL, qm, a);
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            if (it * 32 + lane < NP) {
                int k1 = f1 - j1[it]; if (k1 < 0) k1 += K1;
                int k2 = f2 - j2[it]; if (k2 < 0) k2 += K2;
                int k3 = f3 - j3[it]; if (k3 < 0) k3 += K3;
                const real v = q * tab.th[a][0][j1[it]] * tab.th[a][1][j2[it]] * tab.th[a][2][j3[it]];
                atomicAdd(grid + ((int64_t)k1 * K2 + k2) * K3 + k3, v);
            }
        }
    }
}

template <typename real> struct cplx;
template <> struct cplx<float> { using type = float2; };
template <> struct cplx<double> { using type = double2; };

// Per-axis tables of the influence function, one thread per mesh index: tab[0][k] = m_k = k'/L (k' = k or k - K),
// tab[1][k] = |b(k)|^2 exp(-pi^2 m_k^2 / alpha^2).  exp(-pi^2 m^2 / alpha^2) is separable in the three axes, so the
// per-wave-vector kernel below needs no exponential.
__global__ void pme_axis_tables_kernel(const double* __restrict__ mod, int K, double L, double alpha, double* __restrict__ tab)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= K) return;
    const double m = (double)(k <= K / 2 ? k : k - K) / L;
    tab[k] = m;
    tab[K + k] = mod[k] * exp(-M_PI * M_PI * m * m / (alpha * alpha));
}

// acc[0] += E, acc[1..6] += W (xx, xy, xz, yy, yz, zz)
template <typename real>
__global__ __launch_bounds__(256) void pme_solve_kernel(typename cplx<real>::type* __restrict__ spec, int K1, int K2, int K3, double alpha,
                                                        double ke_over_piV, const double* __restrict__ t1, const double* __restrict__ t2,
                                                        const double* __restrict__ t3, double* __restrict__ acc)
{
    const int K3h = K3 / 2 + 1;
    const int64_t rows = (int64_t)K1 * K2;  // one (k1, k2) row of K3h wave vectors per warp iteration
    double v[7] = {0, 0, 0, 0, 0, 0, 0};
    const double pi2_a2 = M_PI * M_PI / (alpha * alpha);
    const int lane = threadIdx.x & 31;
    const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t r = warp; r < rows; r += n_warps) {
        const int k2 = (int)(r % K2), k1 = (int)(r / K2);
        const double mx = t1[k1], my = t2[k2];
        const bool nyq_x = 2 * k1 == K1, nyq_y = 2 * k2 == K2;
        const double f12 = ke_over_piV * t1[K1 + k1] * t2[K2 + k2], m12 = mx * mx + my * my;
        // four wave vectors per lane at a time: their loads are issued together (one row is K3h <= 4 x 32 for meshes up to
        // 254, i.e. one batch), the arithmetic and the stores follow
        constexpr int UB = 4;
        for (int kb = 0; kb < K3h; kb += 32 * UB) {
            typename cplx<real>::type c[UB];
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int k3 = kb + u * 32 + lane;
                if (k3 < K3h) c[u] = spec[r * K3h + k3];
            }
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int k3 = kb + u * 32 + lane;
                if (k3 >= K3h) continue;
                const int64_t t = r * K3h + k3;
                if (k1 == 0 && k2 == 0 && k3 == 0) {
                    spec[t].x = (real)0;
                    spec[t].y = (real)0;
                    continue;
                }
                const double mz = t3[k3];  // k3 <= K3/2 in the half spectrum
                const double m2 = m12 + mz * mz;
                const double inv_m2 = 1.0 / m2;
                const double bc = f12 * t3[K3 + k3] * inv_m2;
                const double re = (double)c[u].x, im = (double)c[u].y;
                // the half spectrum holds every wave vector with 0 < k3 < K3/2 once for itself and once for its conjugate
                const double wgt = (k3 == 0 || 2 * k3 == K3) ? 1.0 : 2.0;
                const double e = 0.5 * wgt * bc * (re * re + im * im);
                const double fac = 2.0 * (inv_m2 + pi2_a2);
                // The conjugate sits at mesh index (K1 - k1, K2 - k2, K3 - k3); its wave vector is -m, except that an index
                // K/2 of an even mesh maps to +K/2 for both (m' = m for m <= K/2, Essmann's convention, which the oracle
                // follows): the off-diagonal virial terms of the pair then cancel instead of doubling
                const double sx = (wgt == 2.0 && nyq_x) ? 0.0 : 1.0, sy = (wgt == 2.0 && nyq_y) ? 0.0 : 1.0;
                const double sxy = (wgt == 2.0 && (nyq_x != nyq_y)) ? 0.0 : 1.0;
                v[0] += e;
                v[1] += e * (1.0 - fac * mx * mx);
                v[2] += sxy * e * (-fac * mx * my);
                v[3] += sx * e * (-fac * mx * mz);
                v[4] += e * (1.0 - fac * my * my);
                v[5] += sy * e * (-fac * my * mz);
                v[6] += e * (1.0 - fac * mz * mz);
                typename cplx<real>::type o;
                o.x = (real)(bc * re);
                o.y = (real)(bc * im);
                spec[t] = o;
            }
        }
    }
    __shared__ double sh[8][7];
#pragma unroll
    for (int q = 0; q < 7; ++q)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], o);
    const int wi = threadIdx.x >> 5;
    if (lane == 0)
        for (int q = 0; q < 7; ++q) sh[wi][q] = v[q];
    __syncthreads();
    if (threadIdx.x < 7) {
        double s = 0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += sh[w][threadIdx.x];
        atomicAdd(&acc[threadIdx.x], s);
    }
}

template <typename real, int N>
__global__ __launch_bounds__(PME_WARPS * 32) void pme_gather_kernel(const real* __restrict__ pos, const real* __restrict__ charge,
                                                                     int64_t n_atoms, double Lx, double Ly, double Lz, int K1, int K2,
                                                                     int K3, const real* __restrict__ grid, real* __restrict__ F,
                                                                     int accumulate)
{
    __shared__ PmeWarpTable<real, N, true> tabs[PME_WARPS];
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int64_t a0 = (((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5) * 32;
    if (a0 >= n_atoms) return;
    const int cnt = (int)((n_atoms - a0) < 32 ? (n_atoms - a0) : 32);
    PmeWarpTable<real, N, true>& tab = tabs[wib];
    int f1m, f2m, f3m;
    pme_warp_weights<real, N, true>(pos, a0 + lane, lane < cnt, Lx, Ly, Lz, K1, K2, K3, tab, lane, f1m, f2m, f3m);
    constexpr int NP = N * N * N, NIT = (NP + 31) / 32;
    int j1[NIT], j2[NIT], j3[NIT];
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
        const int p = it * 32 + lane, j12 = p / N;
        j3[it] = p - j12 * N;
        j1[it] = j12 / N;
        j2[it] = j12 - j1[it] * N;
    }
    real Fx = (real)0, Fy = (real)0, Fz = (real)0;  // lane a ends up with the sums of atom a
    for (int a = 0; a < cnt; ++a) {
        const int f1 = __shfl_sync(FULL, f1m, a), f2 = __shfl_sync(FULL, f2m, a), f3 = __shfl_sync(FULL, f3m, a);
        real fx = (real)0, fy = (real)0, fz = (real)0;
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            if (it * 32 + lane < NP) {
                int k1 = f1 - j1[it]; if (k1 < 0) k1 += K1;
                int k2 = f2 - j2[it]; if (k2 < 0) k2 += K2;
                int k3 = f3 - j3[it]; if (k3 < 0) k3 += K3;
                const real ph = grid[((int64_t)k1 * K2 + k2) * K3 + k3];
                const real s1 = tab.th[a][0][j1[it]], s2 = tab.th[a][1][j2[it]], s3 = tab.th[a][2][j3[it]];
                fx += tab.dth[a][0][j1[it]] * s2 * s3 * ph;
                fy += s1 * tab.dth[a][1][j2[it]] * s3 * ph;
                fz += s1 * s2 * tab.dth[a][2][j3[it]] * ph;
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            fx += __shfl_xor_sync(FULL, fx, o);
            fy += __shfl_xor_sync(FULL, fy, o);
            fz += __shfl_xor_sync(FULL, fz, o);
        }
        if (lane == a) { Fx = fx; Fy = fy; Fz = fz; }
    }
    if (lane < cnt) {
        const int64_t i = a0 + lane;
        const real q = charge[i];
        const real gx = -q * (real)((double)K1 / Lx) * Fx, gy = -q * (real)((double)K2 / Ly) * Fy, gz = -q * (real)((double)K3 / Lz) * Fz;
        if (accumulate) { F[3 * i] += gx; F[3 * i + 1] += gy; F[3 * i + 2] += gz; }
        else { F[3 * i] = gx; F[3 * i + 1] = gy; F[3 * i + 2] = gz; }
    }
}

template <typename real>
__global__ __launch_bounds__(256) void pme_charge_sq_kernel(const real* __restrict__ charge, int64_t n, double* __restrict__ acc)
{
    double s = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const double q = (double)charge[i];
        s += q * q;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    __shared__ double sh[8];
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += sh[w];
        atomicAdd(&acc[7], t);
    }
}

// E[0] = reciprocal energy, E[1] = self energy (Eq. 12); virial 3x3 from the six accumulated components
__global__ void pme_finish_kernel(const double* __restrict__ acc, double self_factor, double* __restrict__ E, double* __restrict__ W)
{
    if (threadIdx.x == 0) {
        E[0] = acc[0];
        E[1] = self_factor * acc[7];
        if (W) {
            W[0] = acc[1]; W[1] = acc[2]; W[2] = acc[3];
            W[3] = acc[2]; W[4] = acc[4]; W[5] = acc[5];
            W[6] = acc[3]; W[7] = acc[5]; W[8] = acc[6];
        }
    }
}

__global__ void pme_zero_kernel(double* acc)
{
    if (threadIdx.x < 8) acc[threadIdx.x] = 0.0;
}

// |b(m)|^2 per axis on the host (fp64), Essmann Eq. 4.4; zero denominators (odd order, 2 m = K) take the neighbours'
// average as OpenMM does (reading C-25)
double host_bspline(int n, double u)
{
    if (n == 2) return (u >= 0.0 && u <= 2.0) ? 1.0 - fabs(u - 1.0) : 0.0;
    return u / (n - 1) * host_bspline(n - 1, u) + (n - u) / (n - 1) * host_bspline(n - 1, u - 1.0);
}
void host_moduli(int n, int K, double* out)
{
    std::vector<double> den(K);
    for (int m = 0; m < K; ++m) {
        double sc = 0, ss = 0;
        for (int k = 0; k < n - 1; ++k) {
            const double w = host_bspline(n, k + 1.0), arg = 2.0 * M_PI * m * k / K;
            sc += w * cos(arg);
            ss += w * sin(arg);
        }
        den[m] = sc * sc + ss * ss;
    }
    for (int m = 0; m < K; ++m) {
        double d = den[m];
        if (d < 1e-7) d = 0.5 * (den[(m + K - 1) % K] + den[(m + 1) % K]);
        out[m] = 1.0 / d;
    }
}

template <typename real, int N>
int launch_spread_gather(Ctx* ctx, bool gather, const real* pos, const real* charge, int64_t n, const double* L, const int* K, real* grid,
                         real* F, int accumulate, cudaStream_t s)
{
    const unsigned nb = (unsigned)((n + 32 * PME_WARPS - 1) / (32 * PME_WARPS));  // one warp per 32 atoms
    if (!gather) {
        pme_spread_kernel<real, N><<<nb, PME_WARPS * 32, 0, s>>>(pos, charge, n, L[0], L[1], L[2], K[0], K[1], K[2], grid);
        DIMOS_LAUNCH_CHECK(ctx, "pme_spread");
    } else {
        pme_gather_kernel<real, N><<<nb, PME_WARPS * 32, 0, s>>>(pos, charge, n, L[0], L[1], L[2], K[0], K[1], K[2], grid, F, accumulate);
        DIMOS_LAUNCH_CHECK(ctx, "pme_gather");
    }
    return DIMOS_OK;
}

template <typename real>
int spread_gather(Ctx* ctx, int order, bool gather, const real* pos, const real* charge, int64_t n, const double* L, const int* K, real* grid,
                  real* F, int accumulate, cudaStream_t s)
{
    switch (order) {
        case 3: return launch_spread_gather<real, 3>(ctx, gather, pos, charge, n, L, K, grid, F, accumulate, s);
        case 4: return launch_spread_gather<real, 4>(ctx, gather, pos, charge, n, L, K, grid, F, accumulate, s);
        case 5: return launch_spread_gather<real, 5>(ctx, gather, pos, charge, n, L, K, grid, F, accumulate, s);
        case 6: return launch_spread_gather<real, 6>(ctx, gather, pos, charge, n, L, K, grid, F, accumulate, s);
    }
    return set_error(ctx, DIMOS_EINVAL, "PME spline order must be 3..6");
}

}  // namespace

void pme_release(Ctx* ctx)
{
    PmePlan* p = ctx->pme;
    if (!p) return;
    if (p->have_plans) { cufftDestroy(p->fwd); cufftDestroy(p->inv); }
    release(ctx, p->grid);
    release(ctx, p->spec);
    release(ctx, p->moduli);
    release(ctx, p->tables);
    release(ctx, p->work);
    release(ctx, p->acc);
    delete p;
    ctx->pme = nullptr;
}

static int pme_prepare_impl(Ctx* ctx, const int* K, int order, bool dbl, cudaStream_t s)
{
    PmePlan* p = ctx->pme;
    if (p && (p->K[0] != K[0] || p->K[1] != K[1] || p->K[2] != K[2] || p->order != order || p->dbl != dbl)) {
        pme_release(ctx);
        p = nullptr;
    }
    if (p) {
        cufftSetStream(p->fwd, s);
        cufftSetStream(p->inv, s);
        return DIMOS_OK;
    }
    p = new (std::nothrow) PmePlan();
    if (!p) return set_error(ctx, DIMOS_ENOMEM, "out of host memory");
    ctx->pme = p;
    for (int a = 0; a < 3; ++a) p->K[a] = K[a];
    p->order = order;
    p->dbl = dbl;
    const size_t rs = dbl ? 8 : 4;
    const size_t n_real = (size_t)K[0] * K[1] * K[2], n_spec = (size_t)K[0] * K[1] * (K[2] / 2 + 1);
    int rc;
    if ((rc = ensure(ctx, p->grid, n_real * rs, s))) return rc;
    if ((rc = ensure(ctx, p->spec, n_spec * 2 * rs, s))) return rc;
    if ((rc = ensure(ctx, p->moduli, (size_t)(K[0] + K[1] + K[2]) * sizeof(double), s))) return rc;
    if ((rc = ensure(ctx, p->acc, 8 * sizeof(double), s))) return rc;
    if ((rc = ensure(ctx, p->tables, (size_t)2 * (K[0] + K[1] + K[2]) * sizeof(double), s))) return rc;
    std::vector<double> mod(K[0] + K[1] + K[2]);
    host_moduli(order, K[0], mod.data());
    host_moduli(order, K[1], mod.data() + K[0]);
    host_moduli(order, K[2], mod.data() + K[0] + K[1]);
    DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(p->moduli.p, mod.data(), mod.size() * sizeof(double), cudaMemcpyHostToDevice, s));
    DIMOS_CUDA_TRY(ctx, cudaStreamSynchronize(s));  // `mod` is a host temporary
    // cuFFT plans sharing one caller-allocated work area
    size_t ws_f = 0, ws_i = 0;
    if (cufftCreate(&p->fwd) != CUFFT_SUCCESS || cufftCreate(&p->inv) != CUFFT_SUCCESS) return set_error(ctx, DIMOS_ECUDA, "cufftCreate failed");
    p->have_plans = true;
    cufftSetAutoAllocation(p->fwd, 0);
    cufftSetAutoAllocation(p->inv, 0);
    if (cufftMakePlan3d(p->fwd, K[0], K[1], K[2], dbl ? CUFFT_D2Z : CUFFT_R2C, &ws_f) != CUFFT_SUCCESS ||
        cufftMakePlan3d(p->inv, K[0], K[1], K[2], dbl ? CUFFT_Z2D : CUFFT_C2R, &ws_i) != CUFFT_SUCCESS) {
        pme_release(ctx);  // no half-made plan may survive for the next call with the same mesh
        return set_error(ctx, DIMOS_ECUDA, "cufftMakePlan3d failed (mesh size not supported)");
    }
    if ((rc = ensure(ctx, p->work, std::max(ws_f, ws_i), s))) { pme_release(ctx); return rc; }
    cufftSetWorkArea(p->fwd, p->work.p);
    cufftSetWorkArea(p->inv, p->work.p);
    cufftSetStream(p->fwd, s);
    cufftSetStream(p->inv, s);
    return DIMOS_OK;
}

// a plan that could not be completed (allocation, cuFFT) is torn down, so that the next call starts from scratch
static int pme_prepare(Ctx* ctx, const int* K, int order, bool dbl, cudaStream_t s)
{
    const int rc = pme_prepare_impl(ctx, K, order, dbl, s);
    if (rc != DIMOS_OK) pme_release(ctx);
    return rc;
}

template <typename real>
static int pme_recip_typed(Ctx* ctx, const real* pos, const real* charge, int64_t n, const double* L, double alpha, const int* K, int order,
                           double ke, real* F, double* E, double* W, int accumulate, cudaStream_t s)
{
    int rc;
    if ((rc = pme_prepare(ctx, K, order, sizeof(real) == 8, s))) return rc;
    PmePlan* p = ctx->pme;
    real* grid = (real*)p->grid.p;
    double* acc = (double*)p->acc.p;
    const size_t n_real = (size_t)K[0] * K[1] * K[2];
    DIMOS_CUDA_TRY(ctx, cudaMemsetAsync(grid, 0, n_real * sizeof(real), s));
    pme_zero_kernel<<<1, 32, 0, s>>>(acc);
    DIMOS_LAUNCH_CHECK(ctx, "pme_zero");
    if ((rc = spread_gather<real>(ctx, order, false, pos, charge, n, L, K, grid, nullptr, 0, s))) return rc;
    cufftResult fr;
    if (sizeof(real) == 8) fr = cufftExecD2Z(p->fwd, (cufftDoubleReal*)grid, (cufftDoubleComplex*)p->spec.p);
    else fr = cufftExecR2C(p->fwd, (cufftReal*)grid, (cufftComplex*)p->spec.p);
    if (fr != CUFFT_SUCCESS) return set_error(ctx, DIMOS_ECUDA, "cuFFT forward transform failed");
    ctx->launches++;
    const double V = L[0] * L[1] * L[2];
    const int64_t n_spec = (int64_t)K[0] * K[1] * (K[2] / 2 + 1);
    int nb = (int)((n_spec + 255) / 256);
    if (nb > ctx->sm_count * 8) nb = ctx->sm_count * 8;
    const double* mod = (const double*)p->moduli.p;
    double* tab = (double*)p->tables.p;
    if (p->tab_alpha != alpha || p->tab_L[0] != L[0] || p->tab_L[1] != L[1] || p->tab_L[2] != L[2]) {  // once per (alpha, box)
        int off_m = 0, off_t = 0;
        for (int a = 0; a < 3; ++a) {
            pme_axis_tables_kernel<<<(K[a] + 255) / 256, 256, 0, s>>>(mod + off_m, K[a], L[a], alpha, tab + off_t);
            DIMOS_LAUNCH_CHECK(ctx, "pme_axis_tables");
            off_m += K[a];
            off_t += 2 * K[a];
        }
        p->tab_alpha = alpha;
        for (int a = 0; a < 3; ++a) p->tab_L[a] = L[a];
    }
    nb = ctx->sm_count * 8;
    pme_solve_kernel<real><<<nb, 256, 0, s>>>((typename cplx<real>::type*)p->spec.p, K[0], K[1], K[2], alpha, ke / (M_PI * V), tab,
                                              tab + 2 * K[0], tab + 2 * K[0] + 2 * K[1], acc);
    DIMOS_LAUNCH_CHECK(ctx, "pme_solve");
    if (sizeof(real) == 8) fr = cufftExecZ2D(p->inv, (cufftDoubleComplex*)p->spec.p, (cufftDoubleReal*)grid);
    else fr = cufftExecC2R(p->inv, (cufftComplex*)p->spec.p, (cufftReal*)grid);
    if (fr != CUFFT_SUCCESS) return set_error(ctx, DIMOS_ECUDA, "cuFFT inverse transform failed");
    ctx->launches++;
    if (F && (rc = spread_gather<real>(ctx, order, true, pos, charge, n, L, K, grid, F, accumulate, s))) return rc;
    int nbq = (int)((n + 255) / 256);
    if (nbq > ctx->sm_count * 4) nbq = ctx->sm_count * 4;
    pme_charge_sq_kernel<real><<<nbq, 256, 0, s>>>(charge, n, acc);
    DIMOS_LAUNCH_CHECK(ctx, "pme_charge_sq");
    pme_finish_kernel<<<1, 32, 0, s>>>(acc, -ke * alpha / sqrt(M_PI), E, W);
    DIMOS_LAUNCH_CHECK(ctx, "pme_finish");
    return DIMOS_OK;
}

int pme_recip_impl(Ctx* ctx, const void* pos, const void* charge, int64_t n, const double* box, double alpha, const int32_t* mesh,
                   int32_t order, double ke, void* F, double* E, double* W, int accumulate, cudaStream_t s)
{
    const int K[3] = {mesh[0], mesh[1], mesh[2]};
    if (ctx->precision == DIMOS_F64)
        return pme_recip_typed<double>(ctx, (const double*)pos, (const double*)charge, n, box, alpha, K, order, ke, (double*)F, E, W, accumulate, s);
    return pme_recip_typed<float>(ctx, (const float*)pos, (const float*)charge, n, box, alpha, K, order, ke, (float*)F, E, W, accumulate, s);
}

}  // namespace dimos
