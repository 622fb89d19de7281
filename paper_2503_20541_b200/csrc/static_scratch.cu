// static_scratch.cu -- dimos_nl_needs_rebuild_static: the rebuild trigger (reading C-5)
// for callers that must not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// The ordinary trigger (needs_rebuild_kernel, nonbonded.cu) keeps its reduction state in a buffer dimos_create allocates.
// This variant keeps ALL of its scratch -- one block maximum per 1,024 atoms and the ticket that elects the last block --
// in a file-scope __device__ array of fixed size, so the call allocates nothing: no cudaMalloc / cudaFree, no allocator
// callback, no library routine that allocates.  Every GPU that loads the library holds the array (STATIC_SCRATCH_BYTES =
// 64.25 KiB) until the process exits.  The array bounds the problem size: N <= DIMOS_STATIC_MAX_ATOMS.
//
// In host code the array's name is a host-side stand-in, not a device address; the address the kernel gets comes from
// cudaGetSymbolAddress, resolved once per device with that device current (cached below).
#include <math.h>

#include <mutex>

#include "common.cuh"

namespace dimos {

namespace {

constexpr int SS_THREADS = 256;
constexpr int SS_ATOMS_PER_THREAD = 4;
constexpr int SS_ATOMS_PER_BLOCK = SS_THREADS * SS_ATOMS_PER_THREAD;  // 1,024
constexpr int SS_MAX_BLOCKS = 8192;
constexpr size_t SS_HEADER_BYTES = 256;  // [0, 8): ticket (unsigned long long); the rest of the header is padding
constexpr size_t STATIC_SCRATCH_BYTES = SS_HEADER_BYTES + (size_t)SS_MAX_BLOCKS * sizeof(double);
static_assert((int64_t)SS_MAX_BLOCKS * SS_ATOMS_PER_BLOCK == DIMOS_STATIC_MAX_ATOMS, "dimos.h states the limit of this file");

static __device__ __align__(256) unsigned char g_static_scratch[STATIC_SCRATCH_BYTES];

// Block b takes atoms [1024 b, 1024 (b + 1)): thread t the atoms 1024 b + t + 256 k, k = 0..3 (consecutive threads read
// consecutive atoms).  Block maximum -> scratch (as double: exact for float), ticket; the last block to arrive reduces the
// block maxima of the whole grid and writes the flag and, if asked, the maximum itself.
template <typename real>
__global__ __launch_bounds__(SS_THREADS) void needs_rebuild_static_kernel(const real* __restrict__ pos, const real* __restrict__ ref,
                                                                          int64_t N, real thr2, unsigned char* __restrict__ scratch,
                                                                          int* __restrict__ flag, double* __restrict__ max_disp2)
{
    unsigned long long* ticket = reinterpret_cast<unsigned long long*>(scratch);
    double* block_max = reinterpret_cast<double*>(scratch + SS_HEADER_BYTES);
    __shared__ double wmax[SS_THREADS / 32];
    __shared__ bool last;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;

    real m = 0;
    const int64_t base = (int64_t)blockIdx.x * SS_ATOMS_PER_BLOCK + threadIdx.x;
#pragma unroll
    for (int k = 0; k < SS_ATOMS_PER_THREAD; ++k) {
        const int64_t i = base + (int64_t)k * SS_THREADS;
        if (i < N) {
            const real dx = pos[3 * i] - ref[3 * i];
            const real dy = pos[3 * i + 1] - ref[3 * i + 1];
            const real dz = pos[3 * i + 2] - ref[3 * i + 2];
            const real d2 = dx * dx + dy * dy + dz * dz;  // same expression as needs_rebuild_kernel: same rounding
            m = d2 > m ? d2 : m;
            if (!(d2 == d2)) m = (real)INFINITY;  // NaN -> force a rebuild
        }
    }
    double md = (double)m;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) md = fmax(md, __shfl_xor_sync(0xffffffffu, md, o));
    if (lane == 0) wmax[w] = md;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < SS_THREADS / 32; ++k) md = fmax(md, wmax[k]);
        block_max[blockIdx.x] = md;
        __threadfence();
        const unsigned long long t = atomicAdd(ticket, 1ull);
        last = (t == (unsigned long long)gridDim.x - 1);
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double g = 0.0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += SS_THREADS) g = fmax(g, __ldcg(block_max + b));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) g = fmax(g, __shfl_xor_sync(0xffffffffu, g, o));
    __syncthreads();  // wmax is reused
    if (lane == 0) wmax[w] = g;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < SS_THREADS / 32; ++k) g = fmax(g, wmax[k]);
        *flag = g > (double)thr2 ? 1 : 0;
        if (max_disp2) *max_disp2 = g;
        *ticket = 0ull;  // the host clears it before every launch as well
    }
}

// device address of g_static_scratch on `device` (current when called); resolved once per device
int static_scratch_address(Ctx* ctx, unsigned char** out)
{
    constexpr int MAX_DEV = 64;
    static std::mutex mtx;
    static unsigned char* cache[MAX_DEV] = {};
    const int d = ctx->device;
    std::lock_guard<std::mutex> lock(mtx);
    if (d >= 0 && d < MAX_DEV && cache[d]) {
        *out = cache[d];
        return DIMOS_OK;
    }
    unsigned char* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
    if (e != cudaSuccess || !p)
        return set_error(ctx, DIMOS_ECUDA, std::string("cudaGetSymbolAddress(static scratch): ") + cudaGetErrorString(e));
    if (d >= 0 && d < MAX_DEV) cache[d] = p;
    *out = p;
    return DIMOS_OK;
}

}  // namespace

}  // namespace dimos

using namespace dimos;

extern "C" DIMOS_API int dimos_nl_needs_rebuild_static(dimos_ctx* c, const void* pos, const void* pos_at_build, int64_t N, double skin,
                                                       int32_t* flag_dev, double* max_disp2_dev, void* stream)
{
    if (!c) return DIMOS_EINVAL;
    Ctx* ctx = reinterpret_cast<Ctx*>(c);
    if (!pos || !pos_at_build || !flag_dev) return set_error(ctx, DIMOS_EINVAL, "NULL argument");
    if (N <= 0 || !(skin >= 0)) return set_error(ctx, DIMOS_EINVAL, "bad N or skin");
    if (N > (int64_t)DIMOS_STATIC_MAX_ATOMS)
        return set_error(ctx, DIMOS_EOVERFLOW,
                         "dimos_nl_needs_rebuild_static: N = " + std::to_string(N) + " exceeds DIMOS_STATIC_MAX_ATOMS = " +
                             std::to_string((int64_t)DIMOS_STATIC_MAX_ATOMS) + " (the static scratch holds one block maximum per 1024 atoms); "
                             "use dimos_nl_needs_rebuild");
    if (cudaSetDevice(ctx->device) != cudaSuccess) return set_error(ctx, DIMOS_ECUDA, "cudaSetDevice failed");
    unsigned char* scratch = nullptr;
    int rc = static_scratch_address(ctx, &scratch);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    // the array keeps the last call's contents: the ticket must start at zero (the block maxima are all rewritten)
    DIMOS_CUDA_TRY(ctx, cudaMemsetAsync(scratch, 0, SS_HEADER_BYTES, s));
    const unsigned blocks = (unsigned)((N + SS_ATOMS_PER_BLOCK - 1) / SS_ATOMS_PER_BLOCK);
    if (ctx->precision == DIMOS_F64) {
        const double h = 0.5 * skin;
        needs_rebuild_static_kernel<double><<<blocks, SS_THREADS, 0, s>>>((const double*)pos, (const double*)pos_at_build, N, h * h, scratch,
                                                                          flag_dev, max_disp2_dev);
    } else {
        const float h = 0.5f * (float)skin;
        needs_rebuild_static_kernel<float><<<blocks, SS_THREADS, 0, s>>>((const float*)pos, (const float*)pos_at_build, N, h * h, scratch,
                                                                         flag_dev, max_disp2_dev);
    }
    DIMOS_LAUNCH_CHECK(ctx, "needs_rebuild_static");
    return DIMOS_OK;
}
