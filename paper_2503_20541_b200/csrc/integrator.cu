// integrator.cu -- velocity-Verlet update (steps 1, 2 and 5), with the
// skin-displacement rebuild trigger (row A3) fused into the position update: the drift kernel already
// holds every new position in registers, so max |x - x_at_build|^2 costs one more 12-byte read per atom and saves
// the separate needs_rebuild pass.  Constraints (steps 3, 6) and thermostats (step 7) are not built.
//
// Units: nm, ps, amu, kJ mol^-1 nm^-1: a = F / m is in nm ps^-2 without a conversion factor.
#include <math.h>

#include "common.cuh"
#include "trigger.cuh"

namespace dimos {

// steps 1 + 2:  v += (dt/2) F / m;  x += dt v;  [flag = max_i |x_i - x_build,i| > skin/2]
template <typename real, bool TRIGGER>
__global__ void vv_kick_drift_kernel(real* __restrict__ pos, real* __restrict__ vel, const real* __restrict__ F,
                                     const real* __restrict__ inv_mass, int64_t N, real dt, const real* __restrict__ ref,
                                     real thr2, unsigned long long* __restrict__ state, int* __restrict__ flag)
{
    real m = 0;
    const real hdt = (real)0.5 * dt;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
        const real im = inv_mass[i];
        real d2 = 0;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const real v = vel[3 * i + a] + hdt * (F[3 * i + a] * im);
            const real x = pos[3 * i + a] + dt * v;
            vel[3 * i + a] = v;
            pos[3 * i + a] = x;
            if (TRIGGER) {
                const real d = x - ref[3 * i + a];
                d2 += d * d;
            }
        }
        if (TRIGGER) {
            m = d2 > m ? d2 : m;
            if (!(d2 == d2)) m = (real)INFINITY;  // NaN -> force a rebuild
        }
    }
    if (TRIGGER) trigger_reduce_and_flag<real>(m, thr2, state, flag);
}

// step 5:  v += (dt/2) F / m
template <typename real>
__global__ void vv_kick_kernel(real* __restrict__ vel, const real* __restrict__ F, const real* __restrict__ inv_mass,
                               int64_t N, real dt)
{
    const real hdt = (real)0.5 * dt;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
        const real s = hdt * inv_mass[i];
#pragma unroll
        for (int a = 0; a < 3; ++a) vel[3 * i + a] += F[3 * i + a] * s;
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// Step 3 for rigid three-site water (PAPER.md:281-292 step 3; PAPER.md:327 names SETTLE): the analytic solution of the
// three distance constraints, one thread per molecule.  Notation of Miyamoto & Kollman: subscript 0 = positions before the
// drift (rigid), 1 = after the unconstrained drift, 3 = constrained; all relative to the old oxygen, so that fp32
// coordinates only ever enter as differences.  The constraint forces lie in the old molecular plane, hence the component
// along its normal Z is unchanged and the rest is three rotations (phi, psi, theta) of the canonical triangle.
template <typename real>
__global__ void settle_kernel(const real* __restrict__ pos_old, real* __restrict__ pos, real* __restrict__ vel,
                              const int32_t* __restrict__ water, int64_t n_w, real wO, real wH, real ra, real rb, real rc,
                              real d_hh2, real inv_dt)
{
    for (int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; w < n_w; w += (int64_t)gridDim.x * blockDim.x) {
        const int64_t ia = water[3 * w], ib = water[3 * w + 1], ic = water[3 * w + 2];
        real a0[3], b0[3], c0[3], A[3], B[3], C[3], com[3], a1[3], b1[3], c1[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            a0[k] = pos_old[3 * ia + k];
            b0[k] = pos_old[3 * ib + k] - a0[k];
            c0[k] = pos_old[3 * ic + k] - a0[k];
            A[k] = pos[3 * ia + k] - a0[k];
            B[k] = pos[3 * ib + k] - a0[k];
            C[k] = pos[3 * ic + k] - a0[k];
            com[k] = wO * A[k] + wH * (B[k] + C[k]);  // wO = m_O / M, wH = m_H / M
            a1[k] = A[k] - com[k];
            b1[k] = B[k] - com[k];
            c1[k] = C[k] - com[k];
        }
        // orthonormal frame: Z normal to the old plane, X = a1 x Z, Y = Z x X
        real Z[3] = {b0[1] * c0[2] - b0[2] * c0[1], b0[2] * c0[0] - b0[0] * c0[2], b0[0] * c0[1] - b0[1] * c0[0]};
        real X[3] = {a1[1] * Z[2] - a1[2] * Z[1], a1[2] * Z[0] - a1[0] * Z[2], a1[0] * Z[1] - a1[1] * Z[0]};
        real Y[3] = {Z[1] * X[2] - Z[2] * X[1], Z[2] * X[0] - Z[0] * X[2], Z[0] * X[1] - Z[1] * X[0]};
        const real nz = rsqrt(Z[0] * Z[0] + Z[1] * Z[1] + Z[2] * Z[2]);
        const real nx = rsqrt(X[0] * X[0] + X[1] * X[1] + X[2] * X[2]);
        const real ny = rsqrt(Y[0] * Y[0] + Y[1] * Y[1] + Y[2] * Y[2]);
#pragma unroll
        for (int k = 0; k < 3; ++k) { X[k] *= nx; Y[k] *= ny; Z[k] *= nz; }
        auto dot = [](const real* u, const real* v) { return u[0] * v[0] + u[1] * v[1] + u[2] * v[2]; };
        const real xb0 = dot(b0, X), yb0 = dot(b0, Y), xc0 = dot(c0, X), yc0 = dot(c0, Y);
        const real za1 = dot(a1, Z);
        const real xb1 = dot(b1, X), yb1 = dot(b1, Y), zb1 = dot(b1, Z);
        const real xc1 = dot(c1, X), yc1 = dot(c1, Y), zc1 = dot(c1, Z);
        // tilt angles from the unchanged normal components
        const real sinphi = za1 / ra;
        const real cosphi = sqrt((real)1 - sinphi * sinphi);
        const real sinpsi = (zb1 - zc1) / ((real)2 * rc * cosphi);
        const real cospsi = sqrt((real)1 - sinpsi * sinpsi);
        const real ya2 = ra * cosphi;
        real xb2 = -rc * cospsi;
        const real yb2 = -rb * cosphi - rc * sinpsi * sinphi;
        const real yc2 = -rb * cosphi + rc * sinpsi * sinphi;
        // re-impose |bc| = d_HH on xb2 (zero in exact arithmetic; removes the rounding of the two square roots)
        const real dy = yb2 - yc2, dz = zb1 - zc1;
        xb2 = (real)-0.5 * sqrt(fmax(d_hh2 - dy * dy - dz * dz, (real)0));
        // in-plane rotation theta from the zero-torque condition about Z
        const real alpha = xb2 * (xb0 - xc0) + yb0 * yb2 + yc0 * yc2;
        const real beta = xb2 * (yc0 - yb0) + xb0 * yb2 + xc0 * yc2;
        const real gamma = xb0 * yb1 - xb1 * yb0 + xc0 * yc1 - xc1 * yc0;
        const real al2be2 = alpha * alpha + beta * beta;
        const real sintheta = (alpha * gamma - beta * sqrt(fmax(al2be2 - gamma * gamma, (real)0))) / al2be2;
        const real costheta = sqrt((real)1 - sintheta * sintheta);
        const real a3[3] = {-ya2 * sintheta, ya2 * costheta, za1};
        const real b3[3] = {xb2 * costheta - yb2 * sintheta, xb2 * sintheta + yb2 * costheta, zb1};
        const real c3[3] = {-xb2 * costheta - yc2 * sintheta, -xb2 * sintheta + yc2 * costheta, zc1};
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const real na = com[k] + X[k] * a3[0] + Y[k] * a3[1] + Z[k] * a3[2];
            const real nb = com[k] + X[k] * b3[0] + Y[k] * b3[1] + Z[k] * b3[2];
            const real nc = com[k] + X[k] * c3[0] + Y[k] * c3[1] + Z[k] * c3[2];
            if (vel) {  // the constraint displacement is a velocity change over dt
                vel[3 * ia + k] += (na - A[k]) * inv_dt;
                vel[3 * ib + k] += (nb - B[k]) * inv_dt;
                vel[3 * ic + k] += (nc - C[k]) * inv_dt;
            }
            pos[3 * ia + k] = a0[k] + na;
            pos[3 * ib + k] = a0[k] + nb;
            pos[3 * ic + k] = a0[k] + nc;
        }
    }
}

// Step 6 for rigid three-site water (PAPER.md:281-292 step 6): remove the relative velocity along the three bonds with
// impulses mu_k r_k shared by inverse mass.  Bonds k = (O,H1), (O,H2), (H1,H2) with r_k = x_i - x_j; the multipliers solve
// the 3 x 3 system  sum_k c_lk (r_l . r_k) mu_k = -(v_i - v_j)_l . r_l,  c_lk = sum_a s_l(a) s_k(a) / m_a  (s = +1, -1 on the
// two ends of a bond), directly (Cramer), one thread per molecule.
template <typename real>
__global__ void settle_vel_kernel(const real* __restrict__ pos, real* __restrict__ vel, const int32_t* __restrict__ water,
                                  int64_t n_w, real imO, real imH)
{
    for (int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; w < n_w; w += (int64_t)gridDim.x * blockDim.x) {
        const int64_t ia = water[3 * w], ib = water[3 * w + 1], ic = water[3 * w + 2];
        real r0[3], r1[3], r2[3], va[3], vb[3], vc[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const real xa = pos[3 * ia + k], xb = pos[3 * ib + k], xc = pos[3 * ic + k];
            r0[k] = xa - xb;
            r1[k] = xa - xc;
            r2[k] = xb - xc;
            va[k] = vel[3 * ia + k];
            vb[k] = vel[3 * ib + k];
            vc[k] = vel[3 * ic + k];
        }
        auto dot = [](const real* u, const real* v) { return u[0] * v[0] + u[1] * v[1] + u[2] * v[2]; };
        const real a00 = (imO + imH) * dot(r0, r0), a11 = (imO + imH) * dot(r1, r1), a22 = (imH + imH) * dot(r2, r2);
        const real a01 = imO * dot(r0, r1), a02 = -imH * dot(r0, r2), a12 = imH * dot(r1, r2);
        real b0 = 0, b1 = 0, b2 = 0;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            b0 -= (va[k] - vb[k]) * r0[k];
            b1 -= (va[k] - vc[k]) * r1[k];
            b2 -= (vb[k] - vc[k]) * r2[k];
        }
        // symmetric 3 x 3 solve by cofactors
        const real c00 = a11 * a22 - a12 * a12, c01 = a02 * a12 - a01 * a22, c02 = a01 * a12 - a02 * a11;
        const real c11 = a00 * a22 - a02 * a02, c12 = a01 * a02 - a00 * a12, c22 = a00 * a11 - a01 * a01;
        const real idet = (real)1 / (a00 * c00 + a01 * c01 + a02 * c02);
        const real mu0 = (c00 * b0 + c01 * b1 + c02 * b2) * idet;
        const real mu1 = (c01 * b0 + c11 * b1 + c12 * b2) * idet;
        const real mu2 = (c02 * b0 + c12 * b1 + c22 * b2) * idet;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            vel[3 * ia + k] = va[k] + imO * (mu0 * r0[k] + mu1 * r1[k]);
            vel[3 * ib + k] = vb[k] + imH * (mu2 * r2[k] - mu0 * r0[k]);
            vel[3 * ic + k] = vc[k] - imH * (mu1 * r1[k] + mu2 * r2[k]);
        }
    }
}

// Step 7 (Berendsen rescaling).  kinetic_energy: K = 1/2 sum m v^2, products in `real`,
// accumulated in fp64 per thread, warp shuffle, one fp64 atomic per block.  berendsen_scale: every thread derives lambda
// from the device-resident K (no host round trip) and scales its velocities.
template <typename real>
__global__ void kinetic_energy_kernel(const real* __restrict__ vel, const real* __restrict__ inv_mass, int64_t N,
                                      double* __restrict__ ke)
{
    double acc = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
        const real vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
        acc += (double)(vx * vx + vy * vy + vz * vz) / (double)inv_mass[i];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    __shared__ double sh[8];
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += sh[w];
        atomicAdd(ke, 0.5 * t);
    }
}

template <typename real>
__global__ void berendsen_scale_kernel(real* __restrict__ vel, int64_t n3, const double* __restrict__ ke, double two_over_dof_kb,
                                       double T0, double dt_over_tau)
{
    const double T = *ke * two_over_dof_kb;
    const real lam = (real)sqrt(1.0 + dt_over_tau * (T0 / T - 1.0));
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n3; i += (int64_t)gridDim.x * blockDim.x) vel[i] *= lam;
}

// bounding box of all positions (virtual box of a non-periodic system): ordered-int atomics on 6 words
__device__ __forceinline__ unsigned ordered_bits(float f)
{
    const unsigned u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
template <typename real>
__global__ void bbox_kernel(const real* __restrict__ pos, int64_t N, unsigned* __restrict__ out /* min[3], max[3], bad */)
{
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    bool bad = false;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const real x = pos[3 * i + a];
            if (!isfinite(x)) bad = true;
            // round outwards to fp32 so that the fp32 bounds enclose an fp64 coordinate
            const float xl = __double2float_rd((double)x), xh = __double2float_ru((double)x);
            lo[a] = fminf(lo[a], xl);
            hi[a] = fmaxf(hi[a], xh);
        }
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
            hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
        }
    if ((threadIdx.x & 31) == 0)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            atomicMin(&out[a], ordered_bits(lo[a]));
            atomicMax(&out[3 + a], ordered_bits(hi[a]));
        }
    if (bad) out[6] = 1u;
}

int bbox_impl(Ctx* ctx, const void* pos, int64_t N, unsigned* out_dev, cudaStream_t s)
{
    int blocks = (int)((N + 255) / 256);
    const int maxb = ctx->sm_count * 8;
    if (blocks > maxb) blocks = maxb;
    if (blocks < 1) blocks = 1;
    if (ctx->precision == DIMOS_F64) bbox_kernel<double><<<blocks, 256, 0, s>>>((const double*)pos, N, out_dev);
    else bbox_kernel<float><<<blocks, 256, 0, s>>>((const float*)pos, N, out_dev);
    DIMOS_LAUNCH_CHECK(ctx, "bbox");
    return DIMOS_OK;
}

// histogram of the LJ types (dispersion correction): block-local counts in shared memory, then atomics
__global__ void type_histogram_kernel(const int* __restrict__ type, int64_t N, int nt, unsigned long long* __restrict__ counts,
                                      int* __restrict__ bad)
{
    __shared__ unsigned sh[MAX_TYPES];
    for (int t = threadIdx.x; t < nt; t += blockDim.x) sh[t] = 0u;
    __syncthreads();
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
        const int t = type[i];
        if (t < 0 || t >= nt) *bad = 1;
        else atomicAdd(&sh[t], 1u);
    }
    __syncthreads();
    for (int t = threadIdx.x; t < nt; t += blockDim.x)
        if (sh[t]) atomicAdd(&counts[t], (unsigned long long)sh[t]);
}

int type_histogram_impl(Ctx* ctx, const int32_t* type, int64_t N, int nt, unsigned long long* counts_dev, int* bad_dev,
                        cudaStream_t s)
{
    int blocks = (int)((N + 255) / 256);
    const int maxb = ctx->sm_count * 8;
    if (blocks > maxb) blocks = maxb;
    if (blocks < 1) blocks = 1;
    type_histogram_kernel<<<blocks, 256, 0, s>>>(type, N, nt, counts_dev, bad_dev);
    DIMOS_LAUNCH_CHECK(ctx, "type_histogram");
    return DIMOS_OK;
}

static int grid_for(const Ctx* ctx, int64_t N)
{
    int blocks = (int)((N + 255) / 256);
    const int maxb = ctx->sm_count * 8;
    if (blocks > maxb) blocks = maxb;
    return blocks < 1 ? 1 : blocks;
}

template <typename real>
static void launch_kick_drift(Ctx* ctx, void* pos, void* vel, const void* F, const void* inv_mass, int64_t N, double dt,
                              const void* ref, double skin, int32_t* flag_dev, cudaStream_t s)
{
    const int blocks = grid_for(ctx, N);
    const real h = (real)0.5 * (real)skin;
    if (ref && flag_dev)
        vv_kick_drift_kernel<real, true><<<blocks, 256, 0, s>>>((real*)pos, (real*)vel, (const real*)F, (const real*)inv_mass, N,
                                                                 (real)dt, (const real*)ref, h * h, ctx->d_rebuild_state, flag_dev);
    else
        vv_kick_drift_kernel<real, false><<<blocks, 256, 0, s>>>((real*)pos, (real*)vel, (const real*)F, (const real*)inv_mass,
                                                                  N, (real)dt, nullptr, (real)0, nullptr, nullptr);
}

int vv_kick_drift_impl(Ctx* ctx, void* pos, void* vel, const void* F, const void* inv_mass, int64_t N, double dt,
                       const void* pos_at_build, double skin, int32_t* flag_dev, cudaStream_t s)
{
    if (ctx->precision == DIMOS_F64) launch_kick_drift<double>(ctx, pos, vel, F, inv_mass, N, dt, pos_at_build, skin, flag_dev, s);
    else launch_kick_drift<float>(ctx, pos, vel, F, inv_mass, N, dt, pos_at_build, skin, flag_dev, s);
    DIMOS_LAUNCH_CHECK(ctx, "vv_kick_drift");
    return DIMOS_OK;
}

int vv_kick_impl(Ctx* ctx, void* vel, const void* F, const void* inv_mass, int64_t N, double dt, cudaStream_t s)
{
    const int blocks = grid_for(ctx, N);
    if (ctx->precision == DIMOS_F64)
        vv_kick_kernel<double><<<blocks, 256, 0, s>>>((double*)vel, (const double*)F, (const double*)inv_mass, N, dt);
    else
        vv_kick_kernel<float><<<blocks, 256, 0, s>>>((float*)vel, (const float*)F, (const float*)inv_mass, N, (float)dt);
    DIMOS_LAUNCH_CHECK(ctx, "vv_kick");
    return DIMOS_OK;
}

int settle_impl(Ctx* ctx, const void* pos_old, void* pos, void* vel, const int32_t* water, int64_t n_w, double m_O,
                double m_H, double d_OH, double d_HH, double dt, cudaStream_t s)
{
    const double M = m_O + 2.0 * m_H, rc = 0.5 * d_HH, h = sqrt(d_OH * d_OH - rc * rc);
    const double ra = h * 2.0 * m_H / M, rb = h - ra;  // O and the HH midpoint from the centre of mass
    const double inv_dt = dt > 0 ? 1.0 / dt : 0.0;
    const int blocks = grid_for(ctx, n_w);
    if (ctx->precision == DIMOS_F64)
        settle_kernel<double><<<blocks, 256, 0, s>>>((const double*)pos_old, (double*)pos, (double*)vel, water, n_w, m_O / M,
                                                     m_H / M, ra, rb, rc, d_HH * d_HH, inv_dt);
    else
        settle_kernel<float><<<blocks, 256, 0, s>>>((const float*)pos_old, (float*)pos, (float*)vel, water, n_w,
                                                    (float)(m_O / M), (float)(m_H / M), (float)ra, (float)rb, (float)rc,
                                                    (float)(d_HH * d_HH), (float)inv_dt);
    DIMOS_LAUNCH_CHECK(ctx, "settle");
    return DIMOS_OK;
}

int settle_vel_impl(Ctx* ctx, const void* pos, void* vel, const int32_t* water, int64_t n_w, double m_O, double m_H,
                    cudaStream_t s)
{
    const int blocks = grid_for(ctx, n_w);
    if (ctx->precision == DIMOS_F64)
        settle_vel_kernel<double><<<blocks, 256, 0, s>>>((const double*)pos, (double*)vel, water, n_w, 1.0 / m_O, 1.0 / m_H);
    else
        settle_vel_kernel<float><<<blocks, 256, 0, s>>>((const float*)pos, (float*)vel, water, n_w, (float)(1.0 / m_O),
                                                        (float)(1.0 / m_H));
    DIMOS_LAUNCH_CHECK(ctx, "settle_velocities");
    return DIMOS_OK;
}

int kinetic_energy_impl(Ctx* ctx, const void* vel, const void* inv_mass, int64_t N, double* ke_dev, cudaStream_t s)
{
    DIMOS_CUDA_TRY(ctx, cudaMemsetAsync(ke_dev, 0, sizeof(double), s));
    const int blocks = grid_for(ctx, N);
    if (ctx->precision == DIMOS_F64)
        kinetic_energy_kernel<double><<<blocks, 256, 0, s>>>((const double*)vel, (const double*)inv_mass, N, ke_dev);
    else
        kinetic_energy_kernel<float><<<blocks, 256, 0, s>>>((const float*)vel, (const float*)inv_mass, N, ke_dev);
    DIMOS_LAUNCH_CHECK(ctx, "kinetic_energy");
    return DIMOS_OK;
}

int berendsen_scale_impl(Ctx* ctx, void* vel, int64_t N, const double* ke_dev, double two_over_dof_kb, double T0,
                         double dt_over_tau, cudaStream_t s)
{
    const int blocks = grid_for(ctx, 3 * N);
    if (ctx->precision == DIMOS_F64)
        berendsen_scale_kernel<double><<<blocks, 256, 0, s>>>((double*)vel, 3 * N, ke_dev, two_over_dof_kb, T0, dt_over_tau);
    else
        berendsen_scale_kernel<float><<<blocks, 256, 0, s>>>((float*)vel, 3 * N, ke_dev, two_over_dof_kb, T0, dt_over_tau);
    DIMOS_LAUNCH_CHECK(ctx, "berendsen_scale");
    return DIMOS_OK;
}

}  // namespace dimos
