// pair_common.cuh -- declarations shared by the pair-force kernels (nonbonded.cu: generic fp32/fp64/mixed kernel;
// pair_f32x2.cu: packed-FP32 kernel for the fp32 / cell-image-shift case).
#pragma once

#include "common.cuh"

#ifndef F64_MIN_CTAS
#define F64_MIN_CTAS 3  // resident CTAs per SM the fp64 pair kernel is compiled (80 registers) and launched for
#endif

namespace dimos {

__device__ __forceinline__ float4 mk4(float x, float y, float z, float w) { return make_float4(x, y, z, w); }
__device__ __forceinline__ double4 mk4(double x, double y, double z, double w) { return make_double4(x, y, z, w); }

// one vector reduction per j-atom (REDG.E.ADD.F32x4 on sm_100a); fp64 falls back to three scalar REDs
__device__ __forceinline__ void red_add_xyz(float4* p, float x, float y, float z)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(x), "f"(y), "f"(z), "f"(0.0f) : "memory");
}
__device__ __forceinline__ void red_add_xyz(double4* p, double x, double y, double z)
{
    atomicAdd(&p->x, x);
    atomicAdd(&p->y, y);
    atomicAdd(&p->z, z);
}

constexpr int PF_WARPS = 8;
constexpr int STYPE_ACTIVE = 1 << 30;  // stype[] bit: the atom's type has non-zero LJ partners
constexpr int STYPE_MASK = 0xFFFF;
constexpr int FX_WARPS = 8;  // packed-FP32 kernel: warps per CTA
constexpr int FX_CTAS_PER_SM = 2;
constexpr int N_PART = 9;  // E_lj, E_coul, Wxx, Wxy, Wxz, Wyy, Wyz, Wzz, E_excl

template <typename real>
struct ForceParams {
    using real4 = typename vec4<real>::type;
    int64_t n_units, n_slots;
    int row_cap, m_res, nt;
    int row_words;  // packed kernel: words per shared-memory row buffer (row capacity + slack, multiple of 32)
    const real4* xyzq;
    const int* stype;
    const unsigned* entry;        // slot | code << 27
    const unsigned char* emask;   // i-mask per entry (read for the masked chunks)
    const int2* row_info;         // {chunks | partial << 16, nA | nM << 16}
    const typename vec4<real>::type* lj4;  // (c6, c12, 6 c6, 12 c12) per type pair
    unsigned long long* unit_counter;      // dynamic unit scheduling (zeroed by gather_kernel)
    const int* row_active;   // per type: any non-zero LJ partner
    const int* order_stale;  // != 0: an atom the builder assumed LJ-free has LJ partners (evaluate LJ everywhere)
    const int* skip;         // dimos_nb_params.skip_flag: NULL, or a device word; != 0 when the kernel runs: do nothing
    real4* Facc;
    real4* Fown;
    double* partials;        // [gridDim.x][N_PART]
    real rc2, ke, krf, m2krf, crf, alpha, two_a_sqrtpi;
    real rs, inv_sw;  // LJ switch (Eq. 6): r_s and 1/(r_c - r_s)
    int sw_on;
    int erfc_fast;  // fp64 Ewald: alpha r_cut <= 3.6, erfc from the Chebyshev series (nonbonded.cu)
    // fp64 copies for the energy of small fp32 boxes (generic kernel, per-pair minimum image)
    double d_ke, d_krf, d_crf, d_alpha, d_rs, d_inv_sw, d_L[3];
    real L[3], invL[3], h[3];
};

// reduce-scatter of 8 values over the 32 lanes: on return lane l holds, in v[0], the warp-wide sum of
// element ((l>>4)&1)*4 + ((l>>3)&1)*2 + ((l>>2)&1)   (9 shuffles instead of 40)
template <typename T>
__device__ __forceinline__ T reduce8_scatter(T (&v)[8], int lane)
{
    const unsigned FULL = 0xffffffffu;
    const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
    T a[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        T send = b4 ? v[k] : v[k + 4];
        T keep = b4 ? v[k + 4] : v[k];
        a[k] = keep + __shfl_xor_sync(FULL, send, 16);
    }
    T b[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        T send = b3 ? a[k] : a[k + 2];
        T keep = b3 ? a[k + 2] : a[k];
        b[k] = keep + __shfl_xor_sync(FULL, send, 8);
    }
    T send = b2 ? b[0] : b[1];
    T keep = b2 ? b[1] : b[0];
    T c = keep + __shfl_xor_sync(FULL, send, 4);
    c += __shfl_xor_sync(FULL, c, 2);
    c += __shfl_xor_sync(FULL, c, 1);
    return c;
}

// packed-FP32 pair kernel (pair_f32x2.cu); returns false when the case is not covered (caller uses the generic kernel)
// rolled fp64 kernel (pair_f64.cu); false = not covered
bool launch_pair_force_f64(const ForceParams<double>& P, int method, int pbc, unsigned nb, cudaStream_t s);
bool launch_pair_force_f32x2(const ForceParams<float>& P, int method, unsigned nb, size_t dyn, cudaStream_t s);

}  // namespace dimos
