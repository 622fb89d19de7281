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

}  // namespace dimos
