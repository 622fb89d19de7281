// integrator.cu -- velocity-Verlet update (steps 1, 2 and 5), with the
// skin-displacement rebuild trigger (row A3) fused into the position update: the drift kernel already
// holds every new position in registers, so max |x - x_at_build|^2 costs one more 12-byte read per atom and saves
// the separate needs_rebuild pass.  Below: SETTLE for rigid water (steps 3, 6), the Berendsen thermostat (step 7) and
// the two fused per-molecule passes that run steps 1-3 and 5-6 for a water system.
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
                               int64_t N, real dt, const int* __restrict__ skip)
{
    if (skip != nullptr && *skip != 0) return;  // the caller's list is stale (see dimos_nb_params.skip_flag): this step is finished by the host
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
struct SettleGeom {
    real wO, wH;      // m_O / M, m_H / M
    real ra, rb, rc;  // O and the HH midpoint from the centre of mass, half the HH distance
    real d_hh2;
};

// b0, c0: old hydrogens relative to the old oxygen; A, B, C: unconstrained new atoms relative to the old oxygen;
// overwritten with the constrained new atoms in the same frame
template <typename real>
__device__ __forceinline__ void settle_molecule(const real* b0, const real* c0, real* A, real* B, real* C, const SettleGeom<real>& g)
{
    const real ra = g.ra, rb = g.rb, rc = g.rc, d_hh2 = g.d_hh2;
    real com[3], a1[3], b1[3], c1[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        com[k] = g.wO * A[k] + g.wH * (B[k] + C[k]);
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
    const real cosphi = sqrt(fmax((real)1 - sinphi * sinphi, (real)0));  // a molecule distorted beyond recovery gives 0, not NaN
    const real sinpsi = (zb1 - zc1) / ((real)2 * rc * cosphi);
    const real cospsi = sqrt(fmax((real)1 - sinpsi * sinpsi, (real)0));
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
    const real costheta = sqrt(fmax((real)1 - sintheta * sintheta, (real)0));
    const real a3[3] = {-ya2 * sintheta, ya2 * costheta, za1};
    const real b3[3] = {xb2 * costheta - yb2 * sintheta, xb2 * sintheta + yb2 * costheta, zb1};
    const real c3[3] = {-xb2 * costheta - yc2 * sintheta, -xb2 * sintheta + yc2 * costheta, zc1};
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        A[k] = com[k] + X[k] * a3[0] + Y[k] * a3[1] + Z[k] * a3[2];
        B[k] = com[k] + X[k] * b3[0] + Y[k] * b3[1] + Z[k] * b3[2];
        C[k] = com[k] + X[k] * c3[0] + Y[k] * c3[1] + Z[k] * c3[2];
    }
}

template <typename real>
__global__ void settle_kernel(const real* __restrict__ pos_old, real* __restrict__ pos, real* __restrict__ vel,
                              const int32_t* __restrict__ water, int64_t n_w, SettleGeom<real> g, real inv_dt)
{
    for (int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; w < n_w; w += (int64_t)gridDim.x * blockDim.x) {
        const int64_t ia = water[3 * w], ib = water[3 * w + 1], ic = water[3 * w + 2];
        real a0[3], b0[3], c0[3], A[3], B[3], C[3], Au[3], Bu[3], Cu[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            a0[k] = pos_old[3 * ia + k];
            b0[k] = pos_old[3 * ib + k] - a0[k];
            c0[k] = pos_old[3 * ic + k] - a0[k];
            Au[k] = A[k] = pos[3 * ia + k] - a0[k];
            Bu[k] = B[k] = pos[3 * ib + k] - a0[k];
            Cu[k] = C[k] = pos[3 * ic + k] - a0[k];
        }
        settle_molecule<real>(b0, c0, A, B, C, g);
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            if (vel) {  // the constraint displacement is a velocity change over dt
                vel[3 * ia + k] += (A[k] - Au[k]) * inv_dt;
                vel[3 * ib + k] += (B[k] - Bu[k]) * inv_dt;
                vel[3 * ic + k] += (C[k] - Cu[k]) * inv_dt;
            }
            pos[3 * ia + k] = a0[k] + A[k];
            pos[3 * ib + k] = a0[k] + B[k];
            pos[3 * ic + k] = a0[k] + C[k];
        }
    }
}

// Steps 1 + 2 + 3 for a system of rigid waters in one pass: kick, drift, SETTLE, the constraint's velocity change, and the
// rebuild trigger on the constrained positions.  The old positions live in registers, so no copy of them is needed.
template <typename real, bool TRIGGER>
__global__ void water_kick_drift_settle_kernel(real* __restrict__ pos, real* __restrict__ vel, const real* __restrict__ F,
                                               const int32_t* __restrict__ water, int64_t n_w, SettleGeom<real> g, real imO,
                                               real imH, real dt, const real* __restrict__ ref, real thr2,
                                               unsigned long long* __restrict__ state, int* __restrict__ flag)
{
    real m = 0;
    const real hdt = (real)0.5 * dt, inv_dt = (real)1 / dt;
    for (int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; w < n_w; w += (int64_t)gridDim.x * blockDim.x) {
        const int64_t id[3] = {water[3 * w], water[3 * w + 1], water[3 * w + 2]};
        real a0[3], b0[3], c0[3], P[3][3], U[3][3], V[3][3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            a0[k] = pos[3 * id[0] + k];
            b0[k] = pos[3 * id[1] + k] - a0[k];
            c0[k] = pos[3 * id[2] + k] - a0[k];
        }
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const real im = a == 0 ? imO : imH;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                V[a][k] = vel[3 * id[a] + k] + hdt * (F[3 * id[a] + k] * im);
                const real rel0 = a == 0 ? (real)0 : (a == 1 ? b0[k] : c0[k]);
                U[a][k] = P[a][k] = rel0 + dt * V[a][k];
            }
        }
        settle_molecule<real>(b0, c0, P[0], P[1], P[2], g);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            real d2 = 0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const real x = a0[k] + P[a][k];
                vel[3 * id[a] + k] = V[a][k] + (P[a][k] - U[a][k]) * inv_dt;
                pos[3 * id[a] + k] = x;
                if (TRIGGER) {
                    const real d = x - ref[3 * id[a] + k];
                    d2 += d * d;
                }
            }
            if (TRIGGER) {
                m = d2 > m ? d2 : m;
                if (!(d2 == d2)) m = (real)INFINITY;
            }
        }
    }
    if (TRIGGER) trigger_reduce_and_flag<real>(m, thr2, state, flag);
}

// Step 6 for rigid three-site water (PAPER.md:281-292 step 6): remove the relative velocity along the three bonds with
// impulses mu_k r_k shared by inverse mass.  Bonds k = (O,H1), (O,H2), (H1,H2) with r_k = x_i - x_j; the multipliers solve
// the 3 x 3 system  sum_k c_lk (r_l . r_k) mu_k = -(v_i - v_j)_l . r_l,  c_lk = sum_a s_l(a) s_k(a) / m_a  (s = +1, -1 on the
// two ends of a bond), directly (Cramer), one thread per molecule.
// x: positions of O, H1, H2 (any common origin); v: their velocities, corrected in place
template <typename real>
__device__ __forceinline__ void settle_vel_molecule(const real (*x)[3], real (*v)[3], real imO, real imH)
{
    real r0[3], r1[3], r2[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        r0[k] = x[0][k] - x[1][k];
        r1[k] = x[0][k] - x[2][k];
        r2[k] = x[1][k] - x[2][k];
    }
    auto dot = [](const real* u, const real* w) { return u[0] * w[0] + u[1] * w[1] + u[2] * w[2]; };
    const real a00 = (imO + imH) * dot(r0, r0), a11 = (imO + imH) * dot(r1, r1), a22 = (imH + imH) * dot(r2, r2);
    const real a01 = imO * dot(r0, r1), a02 = -imH * dot(r0, r2), a12 = imH * dot(r1, r2);
    real b0 = 0, b1 = 0, b2 = 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        b0 -= (v[0][k] - v[1][k]) * r0[k];
        b1 -= (v[0][k] - v[2][k]) * r1[k];
        b2 -= (v[1][k] - v[2][k]) * r2[k];
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
        v[0][k] += imO * (mu0 * r0[k] + mu1 * r1[k]);
        v[1][k] += imH * (mu2 * r2[k] - mu0 * r0[k]);
        v[2][k] -= imH * (mu1 * r1[k] + mu2 * r2[k]);
    }
}

// KICK: first v += (dt/2) F / m (step 5), then the velocity constraint (step 6); ke (if not NULL) accumulates the kinetic
// energy of the constrained velocities (step 8), fp64, one atomic per block
template <typename real, bool KICK>
__global__ void settle_vel_kernel(const real* __restrict__ pos, real* __restrict__ vel, const real* __restrict__ F,
                                  const int32_t* __restrict__ water, int64_t n_w, real imO, real imH, real hdt,
                                  double* __restrict__ ke, const int* __restrict__ skip)
{
    if (skip != nullptr && *skip != 0) return;  // the caller's list is stale (see dimos_nb_params.skip_flag): this step is finished by the host
    double acc = 0.0;
    for (int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; w < n_w; w += (int64_t)gridDim.x * blockDim.x) {
        const int64_t id[3] = {water[3 * w], water[3 * w + 1], water[3 * w + 2]};
        real x[3][3], v[3][3];
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                x[a][k] = pos[3 * id[a] + k];
                v[a][k] = vel[3 * id[a] + k];
                if (KICK) v[a][k] += hdt * (F[3 * id[a] + k] * (a == 0 ? imO : imH));
            }
        settle_vel_molecule<real>(x, v, imO, imH);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
#pragma unroll
            for (int k = 0; k < 3; ++k) vel[3 * id[a] + k] = v[a][k];
            if (KICK) acc += (double)(v[a][0] * v[a][0] + v[a][1] * v[a][1] + v[a][2] * v[a][2]) / (double)(a == 0 ? imO : imH);
        }
    }
    if (KICK && ke) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        __shared__ double sh[8];
        if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
            for (int q = 0; q < (int)(blockDim.x >> 5); ++q) t += sh[q];
            atomicAdd(ke, 0.5 * t);
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
        const real im = inv_mass[i];
        if (im > (real)0) acc += (double)(vx * vx + vy * vy + vz * vz) / (double)im;  // inv_mass = 0: a frozen atom, no kinetic energy
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
    // a system at rest (T = 0) has nothing to rescale: lambda = 1 instead of a division by zero; the radicand is
    // kept non-negative (dt > tau with T far above T0 would otherwise give NaN velocities)
    const double rad = T > 0.0 ? 1.0 + dt_over_tau * (T0 / T - 1.0) : 1.0;
    const real lam = (real)sqrt(rad > 0.0 ? rad : 0.0);
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
                                                                 (real)dt, (const real*)ref, h * h, next_trigger_state(ctx), flag_dev);
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

// Langevin dynamics, reading C-26: exact Ornstein-Uhlenbeck velocity update v <- a v + sqrt((1 - a^2) k_B T / m) xi
template <typename real>
__global__ void langevin_ou_kernel(real* __restrict__ vel, const real* __restrict__ inv_mass, const real* __restrict__ xi, int64_t N,
                                   real a, real b2 /* (1 - a^2) k_B T */)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
        const real sg = sqrt(b2 * inv_mass[i]);
#pragma unroll
        for (int c = 0; c < 3; ++c) vel[3 * i + c] = a * vel[3 * i + c] + sg * xi[3 * i + c];
    }
}

int langevin_ou_impl(Ctx* ctx, void* vel, const void* inv_mass, const void* xi, int64_t N, double gamma, double dt, double T, cudaStream_t s)
{
    const int blocks = grid_for(ctx, N);
    const double a = exp(-gamma * dt), b2 = (1.0 - a * a) * 8.314462618e-3 * T;
    if (ctx->precision == DIMOS_F64)
        langevin_ou_kernel<double><<<blocks, 256, 0, s>>>((double*)vel, (const double*)inv_mass, (const double*)xi, N, a, b2);
    else
        langevin_ou_kernel<float><<<blocks, 256, 0, s>>>((float*)vel, (const float*)inv_mass, (const float*)xi, N, (float)a, (float)b2);
    DIMOS_LAUNCH_CHECK(ctx, "langevin_ou");
    return DIMOS_OK;
}

int vv_kick_impl(Ctx* ctx, void* vel, const void* F, const void* inv_mass, int64_t N, double dt, const int32_t* skip, cudaStream_t s)
{
    const int blocks = grid_for(ctx, N);
    if (ctx->precision == DIMOS_F64)
        vv_kick_kernel<double><<<blocks, 256, 0, s>>>((double*)vel, (const double*)F, (const double*)inv_mass, N, dt, skip);
    else
        vv_kick_kernel<float><<<blocks, 256, 0, s>>>((float*)vel, (const float*)F, (const float*)inv_mass, N, (float)dt, skip);
    DIMOS_LAUNCH_CHECK(ctx, "vv_kick");
    return DIMOS_OK;
}

template <typename real>
static SettleGeom<real> settle_geom(double m_O, double m_H, double d_OH, double d_HH)
{
    const double M = m_O + 2.0 * m_H, rc = 0.5 * d_HH, h = sqrt(d_OH * d_OH - rc * rc);
    const double ra = h * 2.0 * m_H / M;
    return SettleGeom<real>{(real)(m_O / M), (real)(m_H / M), (real)ra, (real)(h - ra), (real)rc, (real)(d_HH * d_HH)};
}

int settle_impl(Ctx* ctx, const void* pos_old, void* pos, void* vel, const int32_t* water, int64_t n_w, double m_O,
                double m_H, double d_OH, double d_HH, double dt, cudaStream_t s)
{
    const double inv_dt = dt > 0 ? 1.0 / dt : 0.0;
    const int blocks = grid_for(ctx, n_w);
    if (ctx->precision == DIMOS_F64)
        settle_kernel<double><<<blocks, 256, 0, s>>>((const double*)pos_old, (double*)pos, (double*)vel, water, n_w,
                                                     settle_geom<double>(m_O, m_H, d_OH, d_HH), inv_dt);
    else
        settle_kernel<float><<<blocks, 256, 0, s>>>((const float*)pos_old, (float*)pos, (float*)vel, water, n_w,
                                                    settle_geom<float>(m_O, m_H, d_OH, d_HH), (float)inv_dt);
    DIMOS_LAUNCH_CHECK(ctx, "settle");
    return DIMOS_OK;
}

int settle_vel_impl(Ctx* ctx, const void* pos, void* vel, const int32_t* water, int64_t n_w, double m_O, double m_H,
                    cudaStream_t s)
{
    const int blocks = grid_for(ctx, n_w);
    if (ctx->precision == DIMOS_F64)
        settle_vel_kernel<double, false><<<blocks, 256, 0, s>>>((const double*)pos, (double*)vel, nullptr, water, n_w, 1.0 / m_O,
                                                                1.0 / m_H, 0.0, nullptr, nullptr);
    else
        settle_vel_kernel<float, false><<<blocks, 256, 0, s>>>((const float*)pos, (float*)vel, nullptr, water, n_w,
                                                               (float)(1.0 / m_O), (float)(1.0 / m_H), 0.f, nullptr, nullptr);
    DIMOS_LAUNCH_CHECK(ctx, "settle_velocities");
    return DIMOS_OK;
}

template <typename real>
static void launch_water_a(Ctx* ctx, void* pos, void* vel, const void* F, const int32_t* water, int64_t n_w, double m_O,
                           double m_H, double d_OH, double d_HH, double dt, const void* ref, double skin, int32_t* flag_dev,
                           cudaStream_t s)
{
    const int blocks = grid_for(ctx, n_w);
    const real h = (real)0.5 * (real)skin;
    const SettleGeom<real> g = settle_geom<real>(m_O, m_H, d_OH, d_HH);
    if (ref && flag_dev)
        water_kick_drift_settle_kernel<real, true><<<blocks, 256, 0, s>>>((real*)pos, (real*)vel, (const real*)F, water, n_w, g,
                                                                          (real)(1.0 / m_O), (real)(1.0 / m_H), (real)dt,
                                                                          (const real*)ref, h * h, next_trigger_state(ctx), flag_dev);
    else
        water_kick_drift_settle_kernel<real, false><<<blocks, 256, 0, s>>>((real*)pos, (real*)vel, (const real*)F, water, n_w, g,
                                                                           (real)(1.0 / m_O), (real)(1.0 / m_H), (real)dt, nullptr,
                                                                           (real)0, nullptr, nullptr);
}

int water_step_a_impl(Ctx* ctx, void* pos, void* vel, const void* F, const int32_t* water, int64_t n_w, double m_O, double m_H,
                      double d_OH, double d_HH, double dt, const void* ref, double skin, int32_t* flag_dev, cudaStream_t s)
{
    if (ctx->precision == DIMOS_F64) launch_water_a<double>(ctx, pos, vel, F, water, n_w, m_O, m_H, d_OH, d_HH, dt, ref, skin, flag_dev, s);
    else launch_water_a<float>(ctx, pos, vel, F, water, n_w, m_O, m_H, d_OH, d_HH, dt, ref, skin, flag_dev, s);
    DIMOS_LAUNCH_CHECK(ctx, "water_kick_drift_settle");
    return DIMOS_OK;
}

int water_step_b_impl(Ctx* ctx, const void* pos, void* vel, const void* F, const int32_t* water, int64_t n_w, double m_O,
                      double m_H, double dt, double* ke_dev, const int32_t* skip, cudaStream_t s)
{
    if (ke_dev) DIMOS_CUDA_TRY(ctx, cudaMemsetAsync(ke_dev, 0, sizeof(double), s));
    const int blocks = grid_for(ctx, n_w);
    if (ctx->precision == DIMOS_F64)
        settle_vel_kernel<double, true><<<blocks, 256, 0, s>>>((const double*)pos, (double*)vel, (const double*)F, water, n_w,
                                                               1.0 / m_O, 1.0 / m_H, 0.5 * dt, ke_dev, skip);
    else
        settle_vel_kernel<float, true><<<blocks, 256, 0, s>>>((const float*)pos, (float*)vel, (const float*)F, water, n_w,
                                                              (float)(1.0 / m_O), (float)(1.0 / m_H), (float)(0.5 * dt), ke_dev, skip);
    DIMOS_LAUNCH_CHECK(ctx, "water_kick_settle_velocities");
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
