// trigger.cuh -- tail of the skin-displacement rebuild trigger: the grid-wide
// maximum of the squared displacements and the flag  max > (skin/2)^2, shared by needs_rebuild_kernel (nonbonded.cu)
// and the fused velocity-Verlet kick + drift kernel (integrator.cu).
#pragma once

#include "common.cuh"

namespace dimos {

// m: this thread's maximum of |pos - pos_at_build|^2 (INFINITY for a NaN).  Warp shuffle -> block -> one atomicMax per
// block on state[0] (non-negative doubles order like their bit patterns); the last block (ticket in state[1]) writes
// the flag and resets the state for the next call.  Must be reached by every thread of the block.
template <typename real>
__device__ __forceinline__ void trigger_reduce_and_flag(real m, real thr2, unsigned long long* __restrict__ state,
                                                        int* __restrict__ flag)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        real y = __shfl_xor_sync(0xffffffffu, m, o);
        m = y > m ? y : m;
    }
    __shared__ real wmax[32];
    __shared__ bool last;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) wmax[w] = m;
    __syncthreads();
    if (w == 0) {
        m = lane < (blockDim.x >> 5) ? wmax[lane] : (real)0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            real y = __shfl_xor_sync(0xffffffffu, m, o);
            m = y > m ? y : m;
        }
        if (lane == 0) {
            atomicMax(&state[0], (unsigned long long)__double_as_longlong((double)m));
            __threadfence();
            unsigned long long t = atomicAdd(&state[1], 1ull);
            last = (t == (unsigned long long)gridDim.x - 1);
        }
    }
    __syncthreads();
    if (last && threadIdx.x == 0) {
        __threadfence();
        unsigned long long bits = atomicExch(&state[0], 0ull);
        state[1] = 0ull;
        double mx = __longlong_as_double((long long)bits);
        *flag = mx > (double)thr2 ? 1 : 0;
    }
}

}  // namespace dimos
