// nl_build.cu -- neighbour-list construction.
//
//   A1  cell binning by counting sort: bin_atoms (histogram) -> block-scan exclusive prefix sum ->
//       scatter; then, per cell, a k-d bisection in shared memory orders the cell's atoms so that
//       every 8 consecutive atoms form a spatially compact "unit" (i-cluster).
//   A2  cluster-pair list: one warp per unit gathers, from the (de-duplicated) 27-cell stencil,
//       first the units whose bounding box is within r_nl of its own, then the individual j-atoms
//       of those units that have at least one unit atom within r_nl.  Every unordered atom pair is
//       owned by exactly one unit (circular half-ordering of unit indices; triangular mask inside a
//       unit).  An entry is one 32-bit word (slot | stencil code selecting the periodic image); its
//       8-bit i-mask (exclusions, intra-unit half, padding) goes to a byte array that only the masked
//       chunks read.  A row is written in the three-phase layout the force kernels walk: j-atoms
//       assumed LJ-active (the flags of the last force call) upwards from the row's start, the
//       others downwards from the end of its capacity, masked entries and leftovers in between.
//
// All coordinates used here are cell-relative (x - cell origin - wrap*L, formed in fp64 and rounded
// once), so fp32 distance tests across the periodic seam keep ~1e-7 nm absolute accuracy at any L.
#include <math.h>

#include <algorithm>

#include "common.cuh"

namespace dimos {

// ------------------------------------------------------------------------------------------------
// small device helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned ordered_u32(float f)
{
    unsigned u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float4 make4(float x, float y, float z, float w) { return make_float4(x, y, z, w); }
__device__ __forceinline__ double4 make4(double x, double y, double z, double w) { return make_double4(x, y, z, w); }

__device__ __forceinline__ float rint_r(float x) { return rintf(x); }
__device__ __forceinline__ double rint_r(double x) { return rint(x); }

// ------------------------------------------------------------------------------------------------
// A1a: cell index of every atom + histogram ("each atom is assigned to one of the cells")
// ------------------------------------------------------------------------------------------------
template <typename real>
__global__ void bin_atoms_kernel(const real* __restrict__ pos, int64_t N, Grid g, int* __restrict__ cell_count,
                                 int* __restrict__ atom_cell, int* __restrict__ atom_rank,
                                 real* __restrict__ pos_at_build, int* __restrict__ flags)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int c[3];
    bool bad = false;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        real xr = pos[3 * i + a];
        pos_at_build[3 * i + a] = xr;
        double x = (double)xr;
        if (!isfinite(x)) { bad = true; x = 0.0; }
        double f = x / g.L[a];
        f -= floor(f);  // fractional coordinate in [0,1)
        int ci = (int)(f * g.n[a]);
        ci = ci < 0 ? 0 : (ci >= g.n[a] ? g.n[a] - 1 : ci);  // reading C-18
        c[a] = ci;
    }
    if (bad) atomicOr(&flags[0], FLAG_NONFINITE);
    int cell = (c[0] * g.n[1] + c[1]) * g.n[2] + c[2];
    atom_cell[i] = cell;
    atom_rank[i] = atomicAdd(&cell_count[cell], 1);
}

// ------------------------------------------------------------------------------------------------
// generic exclusive prefix sum of int32 (block scan, three phases); out has n+1 elements
// ------------------------------------------------------------------------------------------------
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 4;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

__device__ __forceinline__ int block_exclusive_scan(int v, int* total, int* warp_sums)
{
    // inclusive warp scan
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) warp_sums[w] = x;
    __syncthreads();
    if (w == 0) {
        int s = lane < (SCAN_THREADS / 32) ? warp_sums[lane] : 0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= o) s += y;
        }
        if (lane < (SCAN_THREADS / 32)) warp_sums[lane] = s;  // inclusive warp totals
    }
    __syncthreads();
    int base = w > 0 ? warp_sums[w - 1] : 0;
    *total = warp_sums[SCAN_THREADS / 32 - 1];
    __syncthreads();
    return base + x - v;
}

__global__ void scan_reduce_kernel(const int* __restrict__ in, int64_t n, int* __restrict__ block_sums)
{
    __shared__ int warp_sums[SCAN_THREADS / 32];
    int64_t base = (int64_t)blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    int s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k)
        if (base + k < n) s += in[base + k];
    int total;
    block_exclusive_scan(s, &total, warp_sums);
    if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
}

__global__ void scan_block_sums_kernel(int* __restrict__ block_sums, int nb)
{
    __shared__ int warp_sums[SCAN_THREADS / 32];
    __shared__ int carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int t0 = 0; t0 < nb; t0 += SCAN_THREADS) {
        int idx = t0 + threadIdx.x;
        int v = idx < nb ? block_sums[idx] : 0;
        int total;
        int ex = block_exclusive_scan(v, &total, warp_sums);
        int carry = carry_s;
        if (idx < nb) block_sums[idx] = ex + carry;
        __syncthreads();
        if (threadIdx.x == 0) carry_s = carry + total;
        __syncthreads();
    }
    if (threadIdx.x == 0) block_sums[nb] = carry_s;  // grand total
}

__global__ void scan_apply_kernel(const int* __restrict__ in, int64_t n, const int* __restrict__ block_sums,
                                  int nb, int* __restrict__ out)
{
    __shared__ int warp_sums[SCAN_THREADS / 32];
    int64_t base = (int64_t)blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    int v[SCAN_ITEMS];
    int s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        v[k] = (base + k < n) ? in[base + k] : 0;
        s += v[k];
    }
    int total;
    int ex = block_exclusive_scan(s, &total, warp_sums) + block_sums[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < n) out[base + k] = ex;
        ex += v[k];
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) out[n] = block_sums[nb];
}

static int exclusive_scan(Ctx* ctx, const int* in, int* out, int64_t n, int* tmp, cudaStream_t s)
{
    int nb = (int)((n + SCAN_TILE - 1) / SCAN_TILE);
    if (nb < 1) nb = 1;
    scan_reduce_kernel<<<nb, SCAN_THREADS, 0, s>>>(in, n, tmp);
    DIMOS_LAUNCH_CHECK(ctx, "scan_reduce");
    scan_block_sums_kernel<<<1, SCAN_THREADS, 0, s>>>(tmp, nb);
    DIMOS_LAUNCH_CHECK(ctx, "scan_block_sums");
    scan_apply_kernel<<<nb, SCAN_THREADS, 0, s>>>(in, n, tmp, nb, out);
    DIMOS_LAUNCH_CHECK(ctx, "scan_apply");
    return DIMOS_OK;
}
static size_t scan_tmp_ints(int64_t n) { return (size_t)((n + SCAN_TILE - 1) / SCAN_TILE) + 2; }

// units per cell = ceil(count / UNIT); also records the maximum cell population
__global__ void cell_units_kernel(const int* __restrict__ cell_count, int64_t ncells, int* __restrict__ unit_count,
                                  int* __restrict__ flags)
{
    int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int n = c < ncells ? cell_count[c] : 0;
    if (c < ncells) unit_count[c] = (n + UNIT - 1) / UNIT;
    int m = n;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(&flags[1], m);
}

// A1c: scatter atoms into cell order (counting sort; order inside a cell is fixed later by the k-d sort)
__global__ void scatter_atoms_kernel(int64_t N, const int* __restrict__ atom_cell, const int* __restrict__ atom_rank,
                                     const int* __restrict__ cell_start, int* __restrict__ cell_atoms)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    cell_atoms[cell_start[atom_cell[i]] + atom_rank[i]] = (int)i;
}

// ------------------------------------------------------------------------------------------------
// A1d: per-cell k-d bisection -> compact units of 8 atoms
// ------------------------------------------------------------------------------------------------
// Rank sort inside segments: position p (< n) carries local id Kin[p] and the 32-bit key KEY[p]; if its segment
// [st, st + cnt) is to be sorted (`sort_it`), p moves to st + #{q in the segment: KEY[q] < KEY[p], or equal and q < p}.
// One pass, no barrier inside, ~3 instructions per comparison: a cell of ~150 atoms needs ~450 comparisons per thread
// over all levels of the bisection, where full bitonic sorts of the padded cell cost six times 36 barrier-separated stages.
__device__ __forceinline__ void rank_scatter(const unsigned short* __restrict__ Lin, unsigned short* __restrict__ Lout,
                                             const unsigned* __restrict__ KEY, int p, int st, int cnt, bool sort_it)
{
    int dst = p;
    if (sort_it) {
        const unsigned kp = KEY[p];
        int r = 0;
        for (int q = st; q < st + cnt; ++q) {
            const unsigned kq = KEY[q];
            r += (kq < kp || (kq == kp && q < p)) ? 1 : 0;
        }
        dst = st + r;
    }
    Lout[dst] = Lin[p];
}

// segment arrays of the k-d bisection: a cell of npad (power of two) atoms ends in at most npad / UNIT segments; twice
// that is allocated (the split step writes children 2s, 2s+1)
__host__ __device__ inline int kd_segs(int npad_max) { return 2 * (npad_max / UNIT) < 8 ? 8 : 2 * (npad_max / UNIT); }

template <typename real>
__global__ void kd_cluster_kernel(const real* __restrict__ pos, Grid g, const int* __restrict__ cell_start,
                                  const int* __restrict__ unit_start, const int* __restrict__ cell_atoms,
                                  int* __restrict__ perm, int* __restrict__ inv_perm, double* __restrict__ ref,
                                  typename vec4<real>::type* __restrict__ xyz_build,
                                  typename vec4<real>::type* __restrict__ bb_lo,
                                  typename vec4<real>::type* __restrict__ bb_hi, int* __restrict__ unit_cell,
                                  int npad_max, const unsigned char* __restrict__ atom_active,
                                  unsigned char* __restrict__ slot_hint)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int cell = blockIdx.x;
    const int a0 = cell_start[cell];
    const int n = cell_start[cell + 1] - a0;
    if (n == 0) return;
    int npad = 32;
    while (npad < n) npad <<= 1;

    const int KS = kd_segs(npad_max);
    unsigned* KEY = reinterpret_cast<unsigned*>(smem_raw);                       // sort key of the atom at a position
    unsigned short* LA = reinterpret_cast<unsigned short*>(KEY + npad_max);      // position -> local id, two buffers
    unsigned short* LB = LA + npad_max;
    real* X = reinterpret_cast<real*>(smem_raw + (size_t)npad_max * 8);
    real* Y = X + npad_max;
    real* Z = Y + npad_max;
    int* ID = reinterpret_cast<int*>(Z + npad_max);
    int* segS = ID + npad_max;
    int* segN = segS + KS;
    int* segS2 = segN + KS;
    int* segN2 = segS2 + KS;
    int* segAxis = segN2 + KS;
    int* bbmin = segAxis + KS;  // [3][KS]
    int* bbmax = bbmin + 3 * KS;
    unsigned short* SEG = reinterpret_cast<unsigned short*>(bbmax + 3 * KS);
    __shared__ int any_big;

    // canonical order: by original atom index (makes the units independent of the order the binning atomics produced)
    for (int p = threadIdx.x; p < n; p += blockDim.x) { KEY[p] = (unsigned)cell_atoms[a0 + p]; LA[p] = (unsigned short)p; }
    __syncthreads();
    for (int p = threadIdx.x; p < n; p += blockDim.x) rank_scatter(LA, LB, KEY, p, 0, n, true);
    __syncthreads();

    const int cz = cell % g.n[2];
    const int cy = (cell / g.n[2]) % g.n[1];
    const int cx = cell / (g.n[2] * g.n[1]);
    const double org[3] = {cx * g.h[0], cy * g.h[1], cz * g.h[2]};

    for (int p = threadIdx.x; p < n; p += blockDim.x) {  // local id = canonical rank
        const int id = cell_atoms[a0 + LB[p]];
        ID[p] = id;
        double r[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            double x = (double)pos[3 * (int64_t)id + a];
            if (!isfinite(x)) x = 0.0;
            double k = floor(x / g.L[a]);
            r[a] = x - (org[a] + k * g.L[a]);
        }
        X[p] = (real)r[0];
        Y[p] = (real)r[1];
        Z[p] = (real)r[2];
        SEG[p] = 0;
    }
    __syncthreads();
    for (int p = threadIdx.x; p < n; p += blockDim.x) LA[p] = (unsigned short)p;  // position -> local id
    if (threadIdx.x == 0) { segS[0] = 0; segN[0] = n; }
    __syncthreads();

    int nseg = 1;
    int *cS = segS, *cN = segN, *nS = segS2, *nN = segN2;
    unsigned short *Lc = LA, *Ln = LB;
    for (int level = 0; level < 10; ++level) {
        if (threadIdx.x == 0) any_big = 0;
        __syncthreads();
        for (int s = threadIdx.x; s < nseg; s += blockDim.x) {
            if (cN[s] > UNIT) any_big = 1;
            bbmin[s] = bbmin[KS + s] = bbmin[2 * KS + s] = 0x7fffffff;
            bbmax[s] = bbmax[KS + s] = bbmax[2 * KS + s] = (int)0x80000000;
        }
        __syncthreads();
        if (!any_big) break;
        // bounding box of every segment that will be split (ordered-int atomics in shared memory)
        for (int p = threadIdx.x; p < n; p += blockDim.x) {
            int s = SEG[p];
            if (cN[s] > UNIT) {
                int lid = Lc[p];
                int ox = (int)(ordered_u32((float)X[lid]) ^ 0x80000000u);
                int oy = (int)(ordered_u32((float)Y[lid]) ^ 0x80000000u);
                int oz = (int)(ordered_u32((float)Z[lid]) ^ 0x80000000u);
                atomicMin(&bbmin[s], ox); atomicMax(&bbmax[s], ox);
                atomicMin(&bbmin[KS + s], oy); atomicMax(&bbmax[KS + s], oy);
                atomicMin(&bbmin[2 * KS + s], oz); atomicMax(&bbmax[2 * KS + s], oz);
            }
        }
        __syncthreads();
        for (int s = threadIdx.x; s < nseg; s += blockDim.x) {
            int ax = 0;
            if (cN[s] > UNIT) {
                float ext[3];
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    unsigned lo = (unsigned)bbmin[a * KS + s] ^ 0x80000000u;
                    unsigned hi = (unsigned)bbmax[a * KS + s] ^ 0x80000000u;
                    // undo ordered_u32
                    float flo = __uint_as_float((lo & 0x80000000u) ? (lo & 0x7fffffffu) : ~lo);
                    float fhi = __uint_as_float((hi & 0x80000000u) ? (hi & 0x7fffffffu) : ~hi);
                    ext[a] = fhi - flo;
                }
                if (ext[1] > ext[ax]) ax = 1;
                if (ext[2] > ext[ax]) ax = 2;
            }
            segAxis[s] = ax;
        }
        __syncthreads();
        // key of every atom of a segment to be split: its coordinate along the segment's longest axis
        for (int p = threadIdx.x; p < n; p += blockDim.x) {
            const int s = SEG[p];
            if (cN[s] > UNIT) {
                const int lid = Lc[p], ax = segAxis[s];
                const float v = ax == 0 ? (float)X[lid] : (ax == 1 ? (float)Y[lid] : (float)Z[lid]);
                KEY[p] = ordered_u32(v);
            }
        }
        __syncthreads();
        for (int p = threadIdx.x; p < n; p += blockDim.x) {
            const int s = SEG[p];
            rank_scatter(Lc, Ln, KEY, p, cS[s], cN[s], cN[s] > UNIT);
        }
        // split every big segment: the left child takes a multiple of UNIT atoms
        for (int s = threadIdx.x; s < nseg; s += blockDim.x) {
            int cnt = cN[s], st = cS[s];
            if (cnt > UNIT) {
                int u = (cnt + UNIT - 1) / UNIT;
                int nl = UNIT * ((u + 1) / 2);
                nS[2 * s] = st; nN[2 * s] = nl;
                nS[2 * s + 1] = st + nl; nN[2 * s + 1] = cnt - nl;
            } else {
                nS[2 * s] = st; nN[2 * s] = cnt;
                nS[2 * s + 1] = st + cnt; nN[2 * s + 1] = 0;
            }
        }
        __syncthreads();
        for (int p = threadIdx.x; p < n; p += blockDim.x) {  // segments are position ranges: the scatter stayed inside them
            int s = SEG[p];
            int child = 2 * s;
            if (cN[s] > UNIT && p >= nS[2 * s + 1]) child = 2 * s + 1;
            SEG[p] = (unsigned short)child;
        }
        __syncthreads();
        int* t;
        t = cS; cS = nS; nS = t;
        t = cN; cN = nN; nN = t;
        unsigned short* tl = Lc; Lc = Ln; Ln = tl;
        nseg *= 2;
    }

    // write the cell's atoms in their final order; position p -> slot u0*UNIT + p
    const int u0 = unit_start[cell];
    const int nu = (n + UNIT - 1) / UNIT;
    using real4 = typename vec4<real>::type;
    // LJ-activity hint of every position (remembered from the last force call; all active without one).  Inside a unit the
    // atoms with LJ partners come first, so that they share as few of the pair kernel's i-atom pairs as possible; the
    // list builder files j-atoms by the same flag.  Both are optimisations: the pair kernel checks the real types.
    for (int p = threadIdx.x; p < n; p += blockDim.x) SEG[p] = atom_active ? (unsigned short)(atom_active[ID[Lc[p]]] != 0) : (unsigned short)1;
    __syncthreads();
    for (int p = threadIdx.x; p < n; p += blockDim.x) {  // stable partition of every unit's atoms: active first
        const int b = p & ~(UNIT - 1), e = min(b + UNIT, n);
        const int mine = SEG[p];
        int n_act = 0, before_same = 0;
        for (int k = b; k < e; ++k) {
            n_act += SEG[k];
            before_same += (k < p && SEG[k] == mine) ? 1 : 0;
        }
        const int dst = b + (mine ? before_same : n_act + before_same);
        Ln[dst] = Lc[p];
        KEY[dst] = (unsigned)mine;
    }
    __syncthreads();
    for (int p = threadIdx.x; p < nu * UNIT; p += blockDim.x) {
        const int q = p < n ? p : n - 1;  // padding slots mirror the cell's last atom
        int lid = Ln[q];
        int id = ID[lid];
        int64_t slot = (int64_t)u0 * UNIT + p;
        perm[slot] = p < n ? id : ~id;
        if (p < n) inv_perm[id] = (int)slot;
        const int act = p < n ? (int)KEY[q] : 0;
        slot_hint[slot] = (unsigned char)act;
        // w: 0 = padding slot, 1 = real atom assumed without LJ partners, 2 = real atom assumed with
        xyz_build[slot] = make4(X[lid], Y[lid], Z[lid], p < n ? (real)(1 + act) : (real)0);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            double x = (double)pos[3 * (int64_t)id + a];
            if (!isfinite(x)) x = 0.0;
            double k = floor(x / g.L[a]);
            ref[3 * slot + a] = org[a] + k * g.L[a];
        }
    }
    for (int u = threadIdx.x; u < nu; u += blockDim.x) {
        real lo[3] = {(real)1e30, (real)1e30, (real)1e30}, hi[3] = {(real)-1e30, (real)-1e30, (real)-1e30};
        for (int k = 0; k < UNIT; ++k) {
            int p = u * UNIT + k;
            if (p >= n) break;
            int lid = Lc[p];
            real v[3] = {X[lid], Y[lid], Z[lid]};
#pragma unroll
            for (int a = 0; a < 3; ++a) { lo[a] = v[a] < lo[a] ? v[a] : lo[a]; hi[a] = v[a] > hi[a] ? v[a] : hi[a]; }
        }
        bb_lo[u0 + u] = make4(lo[0], lo[1], lo[2], (real)0);
        bb_hi[u0 + u] = make4(hi[0], hi[1], hi[2], (real)0);
        unit_cell[u0 + u] = cell;
    }
}

static size_t kd_smem_bytes(int npad_max, size_t real_size)
{
    return (size_t)npad_max * (8 + 3 * real_size + 4 + 2) + (size_t)kd_segs(npad_max) * 4 * (5 + 6) + 64;
}

// ------------------------------------------------------------------------------------------------
// exclusion adjacency (CSR over both directions)
// ------------------------------------------------------------------------------------------------
__global__ void excl_degree_kernel(const int2* __restrict__ pairs, int64_t n_excl, int64_t N, int* __restrict__ deg,
                                   int* __restrict__ flags)
{
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_excl) return;
    int2 p = pairs[k];
    if (p.x < 0 || p.y < 0 || p.x >= N || p.y >= N || p.x >= p.y) { atomicOr(&flags[0], FLAG_EXCL_RANGE); return; }
    int a = atomicAdd(&deg[p.x], 1);
    int b = atomicAdd(&deg[p.y], 1);
    if (a >= MAX_EXCL_PER_ATOM || b >= MAX_EXCL_PER_ATOM) atomicOr(&flags[0], FLAG_EXCL_OVERFLOW);
}
__global__ void excl_fill_kernel(const int2* __restrict__ pairs, int64_t n_excl, int64_t N,
                                 const int* __restrict__ start, int* __restrict__ cursor, int* __restrict__ adj)
{
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_excl) return;
    int2 p = pairs[k];
    if (p.x < 0 || p.y < 0 || p.x >= N || p.y >= N || p.x >= p.y) return;
    adj[start[p.x] + atomicAdd(&cursor[p.x], 1)] = p.y;
    adj[start[p.y] + atomicAdd(&cursor[p.y], 1)] = p.x;
}
// every pair must be listed once (reading C-17): a duplicate would be corrected twice by the Ewald exclusion correction
__global__ void excl_unique_kernel(const int2* __restrict__ pairs, int64_t n_excl, int64_t N, const int* __restrict__ start,
                                   const int* __restrict__ adj, int* __restrict__ flags)
{
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_excl) return;
    int2 p = pairs[k];
    if (p.x < 0 || p.y < 0 || p.x >= N || p.y >= N || p.x >= p.y) return;
    int seen = 0;
    const int e = min(start[p.x + 1], start[p.x] + MAX_EXCL_PER_ATOM);
    for (int q = start[p.x]; q < e; ++q) seen += adj[q] == p.y ? 1 : 0;
    if (seen > 1) atomicOr(&flags[0], FLAG_EXCL_DUP);
}
__global__ void zero_int_kernel(int* __restrict__ p, int64_t n)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = 0;
}

// ------------------------------------------------------------------------------------------------
// A2: list build, one warp per unit
// ------------------------------------------------------------------------------------------------
constexpr int BL_WARPS = 4;
constexpr int CAND_MAX = 256;  // candidate units buffered per warp before the atom-level pass
constexpr int EX_MAX = UNIT * MAX_EXCL_PER_ATOM;

template <typename real>
struct BuildParams {
    using real4 = typename vec4<real>::type;
    Grid g;
    int64_t n_units;
    int row_cap, m_res;
    real rnl2;
    real L[3], h[3];
    const int* unit_start;
    const int* unit_cell;
    const int* perm;
    const int* inv_perm;
    const real4* xyz;
    const real4* bb_lo;
    const real4* bb_hi;
    const int* excl_start;
    const int* excl_adj;
    unsigned* entry;
    unsigned char* emask;
    int2* row_info;
    int* flags;
};

// does unit U own the pairs between U and V (U != V)?  Circular half-ordering: balanced rows.
__device__ __forceinline__ bool owns(int64_t U, int64_t V, int64_t n_units)
{
    int64_t d = V - U;
    if (d < 0) d += n_units;
    if (2 * d < n_units) return true;
    if (2 * d == n_units) return U < V;
    return false;
}

template <typename real, int PBC>
__device__ __forceinline__ real axis_gap(real lo1, real hi1, real lo2, real hi2, real L)
{
    real g = fmax((real)0, fmax(lo1 - hi2, lo2 - hi1));
    if (PBC == 1) {
        real g1 = fmax((real)0, fmax(lo1 - (hi2 + L), (lo2 + L) - hi1));
        real g2 = fmax((real)0, fmax(lo1 - (hi2 - L), (lo2 - L) - hi1));
        g = fmin(g, fmin(g1, g2));
    }
    return g;
}

#ifndef BL_MIN_CTAS
#define BL_MIN_CTAS 7  // 72 registers: 28 warps per SM (6 CTAs at 80+ registers measured 8 % slower, 8 CTAs spill)
#endif
template <typename real, int PBC>
__global__ __launch_bounds__(BL_WARPS * 32, (sizeof(real) == 4 && PBC == 0) ? BL_MIN_CTAS : 1) void build_list_kernel(BuildParams<real> P)
{
    using real4 = typename vec4<real>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31;
    const int wib = threadIdx.x >> 5;
    const int64_t U = (int64_t)blockIdx.x * BL_WARPS + wib;
    __shared__ real4 code_off[27];  // image offset of every stencil code (saves the divisions by 9 and 3 per candidate)
    if (threadIdx.x < 27) {
        const int c = threadIdx.x;
        code_off[c] = make4((real)(c / 9 - 1) * P.h[0], (real)((c / 3) % 3 - 1) * P.h[1], (real)(c % 3 - 1) * P.h[2], (real)0);
    }
    __syncthreads();
    if (U >= P.n_units) return;  // no block-wide barriers below
    const unsigned FULL = 0xffffffffu;
    const unsigned lt_mask = (1u << lane) - 1u;

    // per-warp shared-memory carve-up
    const size_t per_warp = (size_t)CAND_MAX * 4 + CAND_MAX + (size_t)P.m_res * 4 + (size_t)P.m_res * 2 +
                            (size_t)EX_MAX * 4 + EX_MAX;
    unsigned char* base = smem_raw + (size_t)wib * ((per_warp + 15) & ~(size_t)15);
    int* cand_unit = reinterpret_cast<int*>(base);
    int* st_j = cand_unit + CAND_MAX;
    int* ex_slot = st_j + P.m_res;
    unsigned short* st_meta = reinterpret_cast<unsigned short*>(ex_slot + EX_MAX);
    unsigned char* cand_code = reinterpret_cast<unsigned char*>(st_meta + P.m_res);
    unsigned char* ex_i = cand_code + CAND_MAX;

    // ---- the unit's own atoms, broadcast to every lane ----
    real xi[UNIT], yi[UNIT], zi[UNIT];
    int my_perm = -1;
    real4 mine = make4((real)0, (real)0, (real)0, (real)0);
    if (lane < UNIT) { mine = P.xyz[U * UNIT + lane]; my_perm = P.perm[U * UNIT + lane]; }
#pragma unroll
    for (int i = 0; i < UNIT; ++i) {
        xi[i] = __shfl_sync(FULL, mine.x, i);
        yi[i] = __shfl_sync(FULL, mine.y, i);
        zi[i] = __shfl_sync(FULL, mine.z, i);
    }
    const unsigned valid_i = __ballot_sync(FULL, lane < UNIT && my_perm >= 0) & 0xFFu;
    const bool unit_full = valid_i == 0xFFu;
    const real4 ulo = P.bb_lo[U], uhi = P.bb_hi[U];

    // ---- exclusion partners of the unit's atoms, as (slot, i) pairs in shared memory ----
    int deg = 0, es = 0;
    if (lane < UNIT && my_perm >= 0) { es = P.excl_start[my_perm]; deg = min(P.excl_start[my_perm + 1] - es, MAX_EXCL_PER_ATOM); }
    int off_ex = deg;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(FULL, off_ex, o);
        if (lane >= o) off_ex += y;
    }
    const int n_ex = __shfl_sync(FULL, off_ex, 31);
    off_ex -= deg;
    int ex_lo = 0x7fffffff, ex_hi = -1;
    for (int k = 0; k < deg; ++k) {
        int s = P.inv_perm[P.excl_adj[es + k]];
        ex_slot[off_ex + k] = s;
        ex_i[off_ex + k] = (unsigned char)lane;
        ex_lo = min(ex_lo, s);
        ex_hi = max(ex_hi, s);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        ex_lo = min(ex_lo, __shfl_xor_sync(FULL, ex_lo, o));
        ex_hi = max(ex_hi, __shfl_xor_sync(FULL, ex_hi, o));
    }
    __syncwarp();

    const int64_t row = U * (int64_t)P.row_cap;
    int nm = 0;   // masked entries staged
    int nua = 0;  // mask-free entries of j-atoms assumed LJ-active: written upwards from the start of the row
    int nub = 0;  // mask-free entries of the others: written downwards from the end of the row's capacity
    bool lost = false;  // warp-uniform: the cursors met
    const int nu_cap = P.row_cap - P.m_res;
    // the row's mask-free region: A upwards from [0], B downwards from [nu_cap - 1].  The pointer goes through an opaque
    // move so that it stays ONE 64-bit register pair (ptxas otherwise re-adds row, m_res and the base for every store)
    unsigned* row_up;
    {
        unsigned* t = P.entry + row + P.m_res;
        asm volatile("mov.b64 %0, %1;" : "=l"(row_up) : "l"(t));
    }

    // append one warp-wide batch of entries; cls_b: the j-atom is assumed to have no LJ partners
    auto append = [&](bool accept, unsigned mask, int j, int code, bool cls_b) {
        const bool is_masked = accept && mask != 0xFFu;
        const bool is_a = accept && !is_masked && !cls_b;
        const bool is_b = accept && !is_masked && cls_b;
        const unsigned ba = __ballot_sync(FULL, is_a), bb = __ballot_sync(FULL, is_b);
        const unsigned e = entry_pack(j, code);
        if (__any_sync(FULL, is_masked)) {  // rare: a j-atom with an exclusion partner in the unit
            const unsigned bm = __ballot_sync(FULL, is_masked);
            if (is_masked) {
                const int pos = nm + __popc(bm & lt_mask);
                if (pos < P.m_res) { st_j[pos] = (int)e; st_meta[pos] = (unsigned short)mask; }
            }
            nm += __popc(bm);
        }
        // the two cursors never write into each other's current batch; once they would, nothing more is written and
        // the row is reported as overflowed (the host grows row_cap and rebuilds)
        if (nua + nub + 64 > nu_cap) lost = true;
        if (is_a && !lost) row_up[nua + __popc(ba & lt_mask)] = e;
        if (is_b && !lost) row_up[nu_cap - 1 - (nub + __popc(bb & lt_mask))] = e;
        nua += __popc(ba);
        nub += __popc(bb);
    };
    // Partial units (fewer than UNIT real atoms, one per cell) keep every entry, with its mask, in the upward region:
    // the force kernels run them through their masked path.
    auto append_any = [&](bool accept, unsigned mask, int j, int code, bool cls_b) {
        if (unit_full) { append(accept, mask, j, code, cls_b); return; }
        unsigned bp = __ballot_sync(FULL, accept);
        if (accept) {
            int pos = nua + __popc(bp & lt_mask);
            if (pos < nu_cap) {
                P.entry[row + P.m_res + pos] = entry_pack(j, code);
                P.emask[row + P.m_res + pos] = (unsigned char)mask;
            }
        }
        nua += __popc(bp);
    };

    // i-mask bits of the unit's atoms that exclude the atom in `slot`
    auto excl_bits = [&](int slot) -> unsigned {
        unsigned ex = 0;
        for (int k = 0; k < n_ex; ++k)
            if (ex_slot[k] == slot) ex |= 1u << ex_i[k];
        return ex;
    };
    const int ex_ulo = ex_lo >> 3, ex_uhi = ex_hi >> 3;  // range of the units that hold an exclusion partner (empty: lo > hi)

    // ---- own-unit entries: the i < j half ----
    {
        bool acc = lane < UNIT && my_perm >= 0;
        int slot = (int)(U * UNIT + lane);
        unsigned mask = 0;
        if (acc) {
            mask = ((1u << lane) - 1u) & valid_i & ~excl_bits(slot);
            acc = mask != 0;
        }
        append_any(acc, mask, slot, SELF_CODE, false);
    }

    // ---- stencil: unique neighbour cells per axis (reading C-18) ----
    const int cell = P.unit_cell[U];
    const int ccz = cell % P.g.n[2];
    const int ccy = (cell / P.g.n[2]) % P.g.n[1];
    const int ccx = cell / (P.g.n[2] * P.g.n[1]);
    const int cc[3] = {ccx, ccy, ccz};
    int sc[3][3], sd[3][3], sn[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int n = P.g.n[a];
        if (n == 1) { sn[a] = 1; sc[a][0] = cc[a]; sd[a][0] = 0; }
        else if (n == 2) { sn[a] = 2; sc[a][0] = cc[a]; sd[a][0] = 0; sc[a][1] = 1 - cc[a]; sd[a][1] = 1 - 2 * cc[a]; }
        else {
            sn[a] = 3;
            for (int k = 0; k < 3; ++k) { int d = k - 1; sd[a][k] = d; sc[a][k] = (cc[a] + d + n) % n; }
        }
    }

    int ncand = 0;
    constexpr int CAND_EXCL = 0x20;  // cand_code bit: the candidate unit holds an exclusion partner of one of the unit's atoms
    // atom-level pass over the buffered candidate units: one j-atom per lane, the next batch's atoms requested before the
    // current batch is tested (the LDS -> LDG chain of a batch is as long as its arithmetic)
    auto flush = [&]() {
        const int T = ncand * UNIT;
        int slot_n = 0, code_n = SELF_CODE;
        real4 pj_n = make4((real)0, (real)0, (real)0, (real)0);  // w = 0: padding, never accepted
        auto fetch = [&](int t) {
            slot_n = 0;
            code_n = SELF_CODE;
            pj_n.w = (real)0;
            if (t < T) {
                code_n = cand_code[t >> 3];
                slot_n = cand_unit[t >> 3] * UNIT + (t & 7);
                pj_n = P.xyz[slot_n];
            }
        };
        fetch(lane);
        for (int t0 = 0; t0 < T; t0 += 32) {
            const int slot = slot_n, code_f = code_n;
            const real4 pj = pj_n;
            fetch(t0 + 32 + lane);
            const int code = code_f & 0x1F;
            bool acc = false;
            const bool cls_b = pj.w == (real)1;
            unsigned mask = valid_i;
            if (__any_sync(FULL, (code_f & CAND_EXCL) != 0)) {
                if (code_f & CAND_EXCL) mask &= ~excl_bits(slot);
            }
            const real4 co = code_off[code];
            const real px = pj.x + co.x, py = pj.y + co.y, pz = pj.z + co.z;
            if constexpr (sizeof(real) == 4 && PBC == 0) {
                // fp32, image from the cell offset: two i-atoms per packed instruction (FADD2/FMUL2/FFMA2); the common
                // case (every i-atom counts) only needs "any i-atom in range": the smallest of the 8 squared distances
                const float2 nx = make_float2(-(float)px, -(float)px), ny = make_float2(-(float)py, -(float)py),
                             nz = make_float2(-(float)pz, -(float)pz);
                float2 r2v[UNIT / 2];
                bool any = false;
#pragma unroll
                for (int q = 0; q < UNIT / 2; ++q) {
                    const float2 ddx = __fadd2_rn(make_float2((float)xi[2 * q], (float)xi[2 * q + 1]), nx);
                    const float2 ddy = __fadd2_rn(make_float2((float)yi[2 * q], (float)yi[2 * q + 1]), ny);
                    const float2 ddz = __fadd2_rn(make_float2((float)zi[2 * q], (float)zi[2 * q + 1]), nz);
                    float2 r2 = __fmul2_rn(ddx, ddx);
                    r2 = __ffma2_rn(ddy, ddy, r2);
                    r2 = __ffma2_rn(ddz, ddz, r2);
                    r2v[q] = r2;
                    any = any || r2.x < (float)P.rnl2 || r2.y < (float)P.rnl2;
                }
                any = any && pj.w != (real)0;
                if (mask == 0xFFu) {
                    acc = any;
                } else if (any) {  // exclusions or missing i-atoms: which i-atoms are in range matters
                    unsigned bits = 0;
#pragma unroll
                    for (int q = 0; q < UNIT / 2; ++q) {
                        bits |= (r2v[q].x < (float)P.rnl2 ? 1u : 0u) << (2 * q);
                        bits |= (r2v[q].y < (float)P.rnl2 ? 1u : 0u) << (2 * q + 1);
                    }
                    acc = (bits & mask) != 0;
                }
            } else {
                unsigned bits = 0;
#pragma unroll
                for (int i = 0; i < UNIT; ++i) {
                    real ddx = xi[i] - px, ddy = yi[i] - py, ddz = zi[i] - pz;
                    if (PBC == 1) {
                        ddx -= P.L[0] * rint_r(ddx / P.L[0]);
                        ddy -= P.L[1] * rint_r(ddy / P.L[1]);
                        ddz -= P.L[2] * rint_r(ddz / P.L[2]);
                    }
                    real r2 = ddx * ddx + ddy * ddy + ddz * ddz;
                    bits |= (r2 < P.rnl2 ? 1u : 0u) << i;
                }
                acc = (bits & mask) != 0 && pj.w != (real)0;
            }
            append_any(acc, mask, slot, code, cls_b);
        }
        ncand = 0;
    };

    // Stencil table, one lane per (de-duplicated) stencil cell: the range of its units that U owns, and the image code.
    // Ownership (owns()) is an arc of unit indices, U + 1 .. U + d_max modulo n_units, and a cell's units are consecutive
    // indices, so the owned units of a cell are the cell's range clipped to the arc: the scan below then visits owned
    // units only and needs no ownership test.  A range that meets both pieces of a wrapped arc (possible only when one
    // cell holds about half of all units) is kept whole and the test is made per candidate (`test_owns`).
    const int n_u = (int)P.n_units;  // n_slots <= 2^27 (checked by the host): unit indices fit in an int
    const int iU = (int)U;
    int my_us = 0, my_cnt = 0, my_code = SELF_CODE;
    bool both = false;
    {
        const int ns = sn[0] * sn[1] * sn[2];
        if (lane < ns) {
            const int iz = lane % sn[2], iy = (lane / sn[2]) % sn[1], ix = lane / (sn[2] * sn[1]);
            int scx = 0, scy = 0, scz = 0, sdx = 0, sdy = 0, sdz = 0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                if (k == ix) { scx = sc[0][k]; sdx = sd[0][k]; }
                if (k == iy) { scy = sc[1][k]; sdy = sd[1][k]; }
                if (k == iz) { scz = sc[2][k]; sdz = sd[2][k]; }
            }
            const int c2 = (scx * P.g.n[1] + scy) * P.g.n[2] + scz;
            my_code = stencil_code(sdx, sdy, sdz);
            const int us = P.unit_start[c2], ue = P.unit_start[c2 + 1];
            const int d_max = (n_u - 1) / 2 + (((n_u & 1) == 0 && iU < n_u / 2) ? 1 : 0);
            const int a_hi = iU + d_max;  // last index of the arc, before wrapping
            const int lo1 = max(us, iU + 1), hi1 = min(ue, min(a_hi, n_u - 1) + 1);  // [U + 1, min(a_hi, n - 1)]
            const int lo2 = us, hi2 = a_hi >= n_u ? min(ue, a_hi - n_u + 1) : us;       // [0, a_hi - n]
            const bool p1 = hi1 > lo1, p2 = hi2 > lo2;
            both = p1 && p2;
            if (both) { my_us = us; my_cnt = ue - us; }
            else if (p1) { my_us = lo1; my_cnt = hi1 - lo1; }
            else if (p2) { my_us = lo2; my_cnt = hi2 - lo2; }
        }
    }
    const bool test_owns = __any_sync(FULL, both);
    int my_pre = my_cnt;  // exclusive prefix sum of the unit counts over the stencil lanes
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(FULL, my_pre, o);
        if (lane >= o) my_pre += y;
    }
    const int n_scan = __shfl_sync(FULL, my_pre, 31);
    my_pre -= my_cnt;

    // flat scan over the candidate units of all stencil cells, 32 per batch
    for (int f0 = 0; f0 < n_scan; f0 += 32) {
        if (ncand + 32 > CAND_MAX) flush();
        const int f = f0 + lane;
        // stencil lane of flat index f: the largest c with prefix[c] <= f (binary search over the lanes' prefixes)
        int c = 0;
#pragma unroll
        for (int step = 16; step > 0; step >>= 1) {
            const int t = c + step;
            const int pt = __shfl_sync(FULL, my_pre, t & 31);
            if (t < 32 && pt <= f) c = t;
        }
        const int c_us = __shfl_sync(FULL, my_us, c), c_pre = __shfl_sync(FULL, my_pre, c);
        int code = __shfl_sync(FULL, my_code, c);
        const int v = c_us + (f - c_pre);
        bool acc = f < n_scan;
        if (test_owns) acc = acc && v != iU && owns(U, v, P.n_units);
        if (acc) {
            const real4 co = code_off[code];
            real4 lo = P.bb_lo[v], hi = P.bb_hi[v];
            real gx = axis_gap<real, PBC>(ulo.x, uhi.x, lo.x + co.x, hi.x + co.x, P.L[0]);
            real gy = axis_gap<real, PBC>(ulo.y, uhi.y, lo.y + co.y, hi.y + co.y, P.L[1]);
            real gz = axis_gap<real, PBC>(ulo.z, uhi.z, lo.z + co.z, hi.z + co.z, P.L[2]);
            acc = gx * gx + gy * gy + gz * gz < P.rnl2;
            if (acc && v >= ex_ulo && v <= ex_uhi) {  // does this unit hold an exclusion partner?
                for (int k = 0; k < n_ex; ++k)
                    if ((ex_slot[k] >> 3) == v) code |= CAND_EXCL;
            }
        }
        unsigned b = __ballot_sync(FULL, acc);
        if (acc) {
            int pos = ncand + __popc(b & lt_mask);
            cand_unit[pos] = v;
            cand_code[pos] = (unsigned char)code;
        }
        ncand += __popc(b);
        __syncwarp();
    }
    flush();
    __syncwarp();

    // ---- finish the row ----
    if (nm > P.m_res) {
        if (lane == 0) { atomicOr(&P.flags[0], FLAG_MASKED_OVERFLOW); atomicMax(&P.flags[7], nm); }
        nm = P.m_res;
    }
    // Row layout (what the force kernels' three phases walk):
    //   [ A: whole chunks of mask-free entries, LJ-active j ][ M: the chunks that read their i-masks ] ... gap ... [ B: whole
    //   chunks of mask-free entries, LJ-free j, ending at the row's capacity ]
    // M holds A's leftover entries (already in place behind A's last whole chunk), the staged masked entries, B's
    // leftover entries (the last ones written, at the low end of the downward region) and padding up to a chunk.
    int full_a = unit_full ? (nua & ~31) : 0, full_b = nub & ~31;
    const int rem_a = nua - full_a, rem_b = nub - full_b;
    int n_mpad = (rem_a + nm + rem_b + 31) & ~31;
    if (lost || full_a + n_mpad + full_b > nu_cap) {
        if (lane == 0) { atomicOr(&P.flags[0], FLAG_ROW_OVERFLOW); atomicMax(&P.flags[6], nua + nub + nm + 160); }
        full_a = full_b = n_mpad = 0;  // the row is unusable; the host grows row_cap and rebuilds
        nm = 0;
    } else if (unit_full) {
        unsigned wb = 0;
        if (lane < rem_b) wb = P.entry[row + P.m_res + (nu_cap - nub) + lane];  // read B's leftovers before M may overwrite them
        __syncwarp();
        const int self = (int)(U * UNIT);
        for (int k = lane; k < n_mpad; k += 32) {
            const int64_t e = row + P.m_res + full_a + k;
            if (k < rem_a) {
                P.emask[e] = 0xFFu;
            } else if (k < rem_a + nm) {
                P.entry[e] = (unsigned)st_j[k - rem_a];
                P.emask[e] = (unsigned char)st_meta[k - rem_a];
            } else if (k < rem_a + nm + rem_b) {
                P.emask[e] = 0xFFu;  // the entry itself (one of B's leftovers) is written below
            } else {
                P.entry[e] = entry_pack(self, SELF_CODE);  // padding: the unit itself, mask 0
                P.emask[e] = 0;
            }
        }
        __syncwarp();
        if (lane < rem_b) P.entry[row + P.m_res + full_a + rem_a + nm + lane] = wb;
    } else {
        // partial unit: pad the upward region to a whole chunk; every chunk is a masked chunk
        const int self = (int)(U * UNIT);
        for (int k = nua + lane; k < n_mpad; k += 32) {
            P.entry[row + P.m_res + k] = entry_pack(self, SELF_CODE);
            P.emask[row + P.m_res + k] = 0;
        }
    }
    if (lane == 0) {
        const int total = (full_a + n_mpad + full_b) >> 5;
        P.row_info[U] = make_int2(total | (unit_full ? 0 : 0x10000), (full_a >> 5) | ((n_mpad >> 5) << 16));
        atomicAdd(reinterpret_cast<unsigned long long*>(&P.flags[2]), (unsigned long long)(nm + nua + nub));
        atomicAdd(reinterpret_cast<unsigned long long*>(&P.flags[4]), (unsigned long long)(total * 32));
    }
}

static size_t build_smem_bytes(int m_res)
{
    size_t per_warp = (size_t)CAND_MAX * 4 + CAND_MAX + (size_t)m_res * 4 + (size_t)m_res * 2 + (size_t)EX_MAX * 4 + EX_MAX;
    per_warp = (per_warp + 15) & ~(size_t)15;
    return per_warp * BL_WARPS;
}

// ------------------------------------------------------------------------------------------------
// export: expand the list to atom pairs at the build positions
// ------------------------------------------------------------------------------------------------
template <typename real, int PBC>
__global__ __launch_bounds__(128) void export_pairs_kernel(BuildParams<real> P, int2* __restrict__ pairs, int64_t cap,
                                                           unsigned long long* __restrict__ counter,
                                                           real* __restrict__ dvec, int* __restrict__ shift,
                                                           const double* __restrict__ ref)
{
    using real4 = typename vec4<real>::type;
    const int lane = threadIdx.x & 31;
    const int64_t U = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
    if (U >= P.n_units) return;
    const unsigned FULL = 0xffffffffu;
    real xi[UNIT], yi[UNIT], zi[UNIT];
    int pi[UNIT];
    int my_perm = -1;
    real4 mine = make4((real)0, (real)0, (real)0, (real)0);
    if (lane < UNIT) { mine = P.xyz[U * UNIT + lane]; my_perm = P.perm[U * UNIT + lane]; }
#pragma unroll
    for (int i = 0; i < UNIT; ++i) {
        xi[i] = __shfl_sync(FULL, mine.x, i);
        yi[i] = __shfl_sync(FULL, mine.y, i);
        zi[i] = __shfl_sync(FULL, mine.z, i);
        pi[i] = __shfl_sync(FULL, my_perm, i);
    }
    const int2 ri = P.row_info[U];
    const int nch = ri.x & 0xFFFF;  // chunks in the row
    const int n_a = ri.y & 0xFFFF, n_am = n_a + (int)((unsigned)ri.y >> 16);
    const int64_t row = U * (int64_t)P.row_cap + P.m_res;
    for (int c = 0; c < nch; ++c) {
        const int64_t e = row + row_chunk_offset(c, nch, n_am, P.row_cap - P.m_res) + lane;
        const unsigned wd = P.entry[e];
        const int j = (int)(wd & ENTRY_SLOT_MASK);
        const unsigned mask = (c >= n_a && c < n_am) ? (unsigned)P.emask[e] : 0xFFu;  // only the masked chunks store masks
        const int code = (int)(wd >> ENTRY_SLOT_BITS);
        real4 pj = P.xyz[j];
        const int pj_orig = P.perm[j];
        const int dx = code / 9 - 1, dy = (code / 3) % 3 - 1, dz = code % 3 - 1;
        const real px = pj.x + (real)dx * P.h[0], py = pj.y + (real)dy * P.h[1], pz = pj.z + (real)dz * P.h[2];
        unsigned bits = 0;
#pragma unroll
        for (int i = 0; i < UNIT; ++i) {
            real ddx = xi[i] - px, ddy = yi[i] - py, ddz = zi[i] - pz;
            if (PBC == 1) {
                ddx -= P.L[0] * rint_r(ddx / P.L[0]);
                ddy -= P.L[1] * rint_r(ddy / P.L[1]);
                ddz -= P.L[2] * rint_r(ddz / P.L[2]);
            }
            real r2 = ddx * ddx + ddy * ddy + ddz * ddz;
            bits |= (r2 < P.rnl2 ? 1u : 0u) << i;
        }
        bits &= mask;
        int cnt = __popc(bits);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(FULL, incl, o);
            if (lane >= o) incl += y;
        }
        int total = __shfl_sync(FULL, incl, 31);
        unsigned long long basep = 0;
        if (lane == 0 && total > 0) basep = atomicAdd(counter, (unsigned long long)total);
        basep = __shfl_sync(FULL, basep, 0);
        unsigned long long w = basep + (unsigned long long)(incl - cnt);
#pragma unroll
        for (int i = 0; i < UNIT; ++i) {
            if (bits & (1u << i)) {
                if ((int64_t)w < cap) {
                    int a = pi[i], b = pj_orig;
                    pairs[w] = a < b ? make_int2(a, b) : make_int2(b, a);
                    if (dvec || shift) {
                        // edge (a, b), a < b:  d = r_a - r_b - n L (minimum image), n = shift.  With raw = cell-relative +
                        // ref the image count follows from the origins: n L = (raw_i - raw_j) - d
                        real d[3] = {xi[i] - px, yi[i] - py, zi[i] - pz};
                        const real rel[3] = {xi[i] - pj.x, yi[i] - pj.y, zi[i] - pj.z};
                        const real sgn = a < b ? (real)1 : (real)-1;
#pragma unroll
                        for (int ax = 0; ax < 3; ++ax) {
                            if (PBC == 1) d[ax] -= P.L[ax] * rint_r(d[ax] / P.L[ax]);
                            const double raw = (ref[3 * (U * UNIT + i) + ax] - ref[3 * (int64_t)j + ax]) + (double)rel[ax];
                            const int n = (int)rint((raw - (double)d[ax]) / (double)P.g.L[ax]);
                            if (dvec) dvec[3 * w + ax] = sgn * d[ax];
                            if (shift) shift[3 * w + ax] = a < b ? n : -n;
                        }
                    }
                }
                ++w;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// host orchestration
// ------------------------------------------------------------------------------------------------
template <typename real>
static BuildParams<real> make_build_params(const NL* nl)
{
    using real4 = typename vec4<real>::type;
    BuildParams<real> P;
    P.g = nl->grid;
    P.n_units = nl->n_units;
    P.row_cap = nl->row_cap;
    P.m_res = nl->m_res;
    P.rnl2 = (real)nl->r_nl * (real)nl->r_nl;
    for (int a = 0; a < 3; ++a) { P.L[a] = (real)nl->grid.L[a]; P.h[a] = (real)nl->grid.h[a]; }
    P.unit_start = (const int*)nl->unit_start.p;
    P.unit_cell = (const int*)nl->unit_cell.p;
    P.perm = (const int*)nl->perm.p;
    P.inv_perm = (const int*)nl->inv_perm.p;
    P.xyz = (const real4*)nl->xyz_build.p;
    P.bb_lo = (const real4*)nl->bb_lo.p;
    P.bb_hi = (const real4*)nl->bb_hi.p;
    P.excl_start = (const int*)nl->excl_start.p;
    P.excl_adj = (const int*)nl->excl_adj.p;
    P.entry = (unsigned*)nl->entry.p;
    P.emask = (unsigned char*)nl->emask.p;
    P.row_info = (int2*)nl->row_info.p;
    P.flags = (int*)nl->flags.p;
    return P;
}

template <typename real>
static int nl_build_typed(Ctx* ctx, NL* nl, const real* pos, const int32_t* excl_pairs, int64_t n_excl,
                          real* pos_at_build, cudaStream_t s)
{
    using real4 = typename vec4<real>::type;
    const int64_t N = nl->N;
    const Grid& g = nl->grid;
    const int64_t ncells = g.ncells;
    int rc;
    // ---- workspace that depends only on N / ncells ----
    if ((rc = ensure(ctx, nl->cell_count, (ncells + 1) * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->cell_start, (ncells + 1) * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->unit_start, (ncells + 1) * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->scan_tmp, (scan_tmp_ints(std::max(ncells, N) + 1) + (size_t)ncells + 1 + (size_t)N + 1) * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->atom_cell, N * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->atom_rank, N * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->cell_atoms, N * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->inv_perm, N * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->flags, 16 * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->excl_start, (N + 1) * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->excl_adj, (size_t)std::max<int64_t>(2 * n_excl, 1) * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->excl_pairs, (size_t)std::max<int64_t>(n_excl, 1) * sizeof(int2), s))) return rc;
    if ((rc = ensure(ctx, nl->export_count, 8, s))) return rc;
    int* flags = (int*)nl->flags.p;
    int* scan_tmp = (int*)nl->scan_tmp.p;
    int* unit_count = scan_tmp + scan_tmp_ints(std::max(ncells, N) + 1);  // int[ncells+1]
    int* excl_deg = unit_count + ncells + 1;                               // int[N+1]
    const int T = 256;

    zero_int_kernel<<<1, 32, 0, s>>>(flags, 16);
    DIMOS_LAUNCH_CHECK(ctx, "zero_flags");
    zero_int_kernel<<<(unsigned)((ncells + 1 + T - 1) / T), T, 0, s>>>((int*)nl->cell_count.p, ncells + 1);
    DIMOS_LAUNCH_CHECK(ctx, "zero_cells");
    bin_atoms_kernel<real><<<(unsigned)((N + T - 1) / T), T, 0, s>>>(pos, N, g, (int*)nl->cell_count.p,
                                                                      (int*)nl->atom_cell.p, (int*)nl->atom_rank.p,
                                                                      pos_at_build, flags);
    DIMOS_LAUNCH_CHECK(ctx, "bin_atoms");
    cell_units_kernel<<<(unsigned)((ncells + T - 1) / T), T, 0, s>>>((const int*)nl->cell_count.p, ncells, unit_count, flags);
    DIMOS_LAUNCH_CHECK(ctx, "cell_units");
    if ((rc = exclusive_scan(ctx, (const int*)nl->cell_count.p, (int*)nl->cell_start.p, ncells, scan_tmp, s))) return rc;
    if ((rc = exclusive_scan(ctx, unit_count, (int*)nl->unit_start.p, ncells, scan_tmp, s))) return rc;
    scatter_atoms_kernel<<<(unsigned)((N + T - 1) / T), T, 0, s>>>(N, (const int*)nl->atom_cell.p, (const int*)nl->atom_rank.p,
                                                                   (const int*)nl->cell_start.p, (int*)nl->cell_atoms.p);
    DIMOS_LAUNCH_CHECK(ctx, "scatter_atoms");

    // exclusion CSR
    nl->n_excl = n_excl;
    zero_int_kernel<<<(unsigned)((N + 1 + T - 1) / T), T, 0, s>>>(excl_deg, N + 1);
    DIMOS_LAUNCH_CHECK(ctx, "zero_deg");
    if (n_excl > 0) {
        if ((const void*)excl_pairs != (const void*)nl->excl_pairs.p)  // dimos_step_host rebuilds from the retained copy
            DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(nl->excl_pairs.p, excl_pairs, n_excl * sizeof(int2), cudaMemcpyDeviceToDevice, s));
        excl_degree_kernel<<<(unsigned)((n_excl + T - 1) / T), T, 0, s>>>((const int2*)nl->excl_pairs.p, n_excl, N, excl_deg, flags);
        DIMOS_LAUNCH_CHECK(ctx, "excl_degree");
    }
    if ((rc = exclusive_scan(ctx, excl_deg, (int*)nl->excl_start.p, N, scan_tmp, s))) return rc;
    if (n_excl > 0) {
        zero_int_kernel<<<(unsigned)((N + 1 + T - 1) / T), T, 0, s>>>(excl_deg, N + 1);
        DIMOS_LAUNCH_CHECK(ctx, "zero_cursor");
        excl_fill_kernel<<<(unsigned)((n_excl + T - 1) / T), T, 0, s>>>((const int2*)nl->excl_pairs.p, n_excl, N,
                                                                        (const int*)nl->excl_start.p, excl_deg, (int*)nl->excl_adj.p);
        DIMOS_LAUNCH_CHECK(ctx, "excl_fill");
        excl_unique_kernel<<<(unsigned)((n_excl + T - 1) / T), T, 0, s>>>((const int2*)nl->excl_pairs.p, n_excl, N, (const int*)nl->excl_start.p,
                                                                          (const int*)nl->excl_adj.p, flags);
        DIMOS_LAUNCH_CHECK(ctx, "excl_unique");
    }

    // the 1-4 exceptions the list holds (dimos_nl_set_exceptions) survive a rebuild only if they still fit the system: indices
    // below the new N and every pair among the new excluded pairs; checked against the adjacency just built (flags[10])
    if (nl->n_exc > 0 && (rc = check_exceptions_impl(ctx, nl, (const int32_t*)nl->exc_pairs.p, nl->n_exc, flags + 10, s))) return rc;

    // ---- read back: number of units, max cell population, early error flags (sync #1) ----
    int* h = ctx->h_pinned;
    DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(h, flags, 2 * sizeof(int), cudaMemcpyDeviceToHost, s));
    DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(h + 2, (int*)nl->unit_start.p + ncells, sizeof(int), cudaMemcpyDeviceToHost, s));
    DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(h + 3, flags + 10, sizeof(int), cudaMemcpyDeviceToHost, s));
    DIMOS_CUDA_TRY(ctx, cudaStreamSynchronize(s));
    if (nl->n_exc > 0 && h[3] != 0) {
        nl->n_exc = 0;  // they cannot be used with this system; the handle itself stays usable for the next build
        return set_error(ctx, DIMOS_EINVAL,
                         "the list's 1-4 exceptions do not fit the system it is rebuilt for (index out of range, or a pair that is "
                         "not among the excluded pairs): they have been removed; set them again after the build");
    }
    if (h[0] & FLAG_NONFINITE) return set_error(ctx, DIMOS_EINVAL, "non-finite coordinate in pos");
    if (h[0] & FLAG_EXCL_RANGE) return set_error(ctx, DIMOS_EINVAL, "excl_pairs row out of range or not i<j");
    if (h[0] & FLAG_EXCL_OVERFLOW) return set_error(ctx, DIMOS_EINVAL, "an atom has more than 32 exclusion partners");
    if (h[0] & FLAG_EXCL_DUP) return set_error(ctx, DIMOS_EINVAL, "excl_pairs lists a pair more than once");
    nl->max_cell_count = h[1];
    if (h[1] > KD_MAX) return set_error(ctx, DIMOS_EOVERFLOW, "more than 4096 atoms in one cell (r_cut+skin too large for this density)");
    nl->n_units = h[2];
    nl->n_slots = nl->n_units * UNIT;
    if (nl->n_slots > (int64_t)ENTRY_SLOT_MASK) return set_error(ctx, DIMOS_EOVERFLOW, "more than 2^27 atom slots: list entries hold 27-bit slot indices");
    const int64_t nun = nl->n_units, nsl = nl->n_slots;

    if ((rc = ensure(ctx, nl->perm, nsl * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->ref, nsl * 3 * sizeof(double), s))) return rc;
    if ((rc = ensure(ctx, nl->xyz_build, nsl * sizeof(real4), s))) return rc;
    if ((rc = ensure(ctx, nl->bb_lo, nun * sizeof(real4), s))) return rc;
    if ((rc = ensure(ctx, nl->bb_hi, nun * sizeof(real4), s))) return rc;
    if ((rc = ensure(ctx, nl->unit_cell, nun * sizeof(int), s))) return rc;
    if ((rc = ensure(ctx, nl->row_info, nun * sizeof(int2), s))) return rc;
    if ((rc = ensure(ctx, nl->slot_hint, nsl, s))) return rc;

    int npad_max = 32;
    while (npad_max < nl->max_cell_count) npad_max <<= 1;
    const size_t kd_smem = kd_smem_bytes(npad_max, sizeof(real));
    DIMOS_CUDA_TRY(ctx, cudaFuncSetAttribute(kd_cluster_kernel<real>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kd_smem));
    kd_cluster_kernel<real><<<(unsigned)ncells, 256, kd_smem, s>>>(
        pos, g, (const int*)nl->cell_start.p, (const int*)nl->unit_start.p, (const int*)nl->cell_atoms.p, (int*)nl->perm.p,
        (int*)nl->inv_perm.p, (double*)nl->ref.p, (real4*)nl->xyz_build.p, (real4*)nl->bb_lo.p, (real4*)nl->bb_hi.p,
        (int*)nl->unit_cell.p, npad_max, nl->hint_valid ? (const unsigned char*)nl->atom_active.p : nullptr,
        (unsigned char*)nl->slot_hint.p);
    DIMOS_LAUNCH_CHECK(ctx, "kd_cluster");

    // ---- row capacity estimate (grown on overflow) ----
    if (nl->row_cap == 0) {
        const double vol = g.L[0] * g.L[1] * g.L[2];
        const double dens = (double)N / vol;
        const double ext = 0.75 * cbrt((double)UNIT / dens);
        const double rr = nl->r_nl + ext;
        double est = 0.5 * dens * (4.0 / 3.0) * M_PI * rr * rr * rr * 1.3 + 64;
        if (est > (double)N + 32) est = (double)N + 32;
        nl->row_cap = nl->m_res + (((int)est + 31) & ~31);
    }
    for (int attempt = 0; attempt < 6; ++attempt) {
        if ((rc = ensure(ctx, nl->entry, ((size_t)nun * nl->row_cap + LIST_SLACK) * sizeof(unsigned), s))) return rc;
        if ((rc = ensure(ctx, nl->emask, ((size_t)nun * nl->row_cap + LIST_SLACK) * sizeof(unsigned char), s))) return rc;
        zero_int_kernel<<<1, 32, 0, s>>>(flags + 2, 8);
        DIMOS_LAUNCH_CHECK(ctx, "zero_counters");
        BuildParams<real> P = make_build_params<real>(nl);
        const size_t smem = build_smem_bytes(nl->m_res);
        const unsigned nb = (unsigned)((nun + BL_WARPS - 1) / BL_WARPS);
        if (g.pbc_mode == 0) {
            DIMOS_CUDA_TRY(ctx, cudaFuncSetAttribute(build_list_kernel<real, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            build_list_kernel<real, 0><<<nb, BL_WARPS * 32, smem, s>>>(P);
        } else {
            DIMOS_CUDA_TRY(ctx, cudaFuncSetAttribute(build_list_kernel<real, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            build_list_kernel<real, 1><<<nb, BL_WARPS * 32, smem, s>>>(P);
        }
        DIMOS_LAUNCH_CHECK(ctx, "build_list");
        DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(h, flags, 8 * sizeof(int), cudaMemcpyDeviceToHost, s));
        DIMOS_CUDA_TRY(ctx, cudaStreamSynchronize(s));  // sync #2
        if (!(h[0] & (FLAG_ROW_OVERFLOW | FLAG_MASKED_OVERFLOW))) {
            unsigned long long ne, np;
            memcpy(&ne, h + 2, 8);
            memcpy(&np, h + 4, 8);
            nl->n_entries = (int64_t)ne;
            nl->n_entries_padded = (int64_t)np;
            return DIMOS_OK;
        }
        nl->n_grow++;
        if (h[0] & FLAG_MASKED_OVERFLOW) {
            int need = (h[7] + 31) & ~31;
            if (need > 4096) return set_error(ctx, DIMOS_EOVERFLOW, "too many masked entries per unit");
            nl->row_cap += need - nl->m_res;
            nl->m_res = need;
        }
        if (h[0] & FLAG_ROW_OVERFLOW) nl->row_cap = nl->m_res + (((int)(h[6] * 1.15) + 63) & ~31);
        zero_int_kernel<<<1, 32, 0, s>>>(flags, 1);
        DIMOS_LAUNCH_CHECK(ctx, "zero_flags");
        zero_int_kernel<<<1, 32, 0, s>>>(flags + 6, 2);
        DIMOS_LAUNCH_CHECK(ctx, "zero_flags");
    }
    return set_error(ctx, DIMOS_EOVERFLOW, "neighbour-list row capacity still exceeded after 6 growth attempts");
}

int nl_build_impl(Ctx* ctx, NL* nl, const void* pos, const int32_t* excl_pairs, int64_t n_excl, void* pos_at_build,
                  cudaStream_t s)
{
    if (ctx->precision == DIMOS_F64)
        return nl_build_typed<double>(ctx, nl, (const double*)pos, excl_pairs, n_excl, (double*)pos_at_build, s);
    return nl_build_typed<float>(ctx, nl, (const float*)pos, excl_pairs, n_excl, (float*)pos_at_build, s);
}

template <typename real>
static int nl_export_typed(Ctx* ctx, const NL* nl, int32_t* pairs, int64_t cap, int64_t* n_pairs_host, double radius, void* dvec,
                           int32_t* shift, cudaStream_t s)
{
    BuildParams<real> P = make_build_params<real>(nl);
    P.rnl2 = (real)radius * (real)radius;
    unsigned long long* counter = (unsigned long long*)nl->export_count.p;
    zero_int_kernel<<<1, 32, 0, s>>>((int*)counter, 2);
    DIMOS_LAUNCH_CHECK(ctx, "zero_counter");
    const unsigned nb = (unsigned)((nl->n_units + 3) / 4);
    if (nl->grid.pbc_mode == 0)
        export_pairs_kernel<real, 0><<<nb, 128, 0, s>>>(P, (int2*)pairs, pairs ? cap : 0, counter, (real*)dvec, shift, (const double*)nl->ref.p);
    else
        export_pairs_kernel<real, 1><<<nb, 128, 0, s>>>(P, (int2*)pairs, pairs ? cap : 0, counter, (real*)dvec, shift, (const double*)nl->ref.p);
    DIMOS_LAUNCH_CHECK(ctx, "export_pairs");
    unsigned long long* h = reinterpret_cast<unsigned long long*>(ctx->h_pinned + 16);
    DIMOS_CUDA_TRY(ctx, cudaMemcpyAsync(h, counter, 8, cudaMemcpyDeviceToHost, s));
    DIMOS_CUDA_TRY(ctx, cudaStreamSynchronize(s));
    *n_pairs_host = (int64_t)*h;
    if ((int64_t)*h > cap && pairs) return set_error(ctx, DIMOS_EOVERFLOW, "pairs buffer too small");
    return DIMOS_OK;
}

int nl_export_impl(Ctx* ctx, const NL* nl, int32_t* pairs, int64_t cap, int64_t* n_pairs_host, double radius, cudaStream_t s,
                   void* dvec, int32_t* shift)
{
    if (ctx->precision == DIMOS_F64) return nl_export_typed<double>(ctx, nl, pairs, cap, n_pairs_host, radius, dvec, shift, s);
    return nl_export_typed<float>(ctx, nl, pairs, cap, n_pairs_host, radius, dvec, shift, s);
}

}  // namespace dimos
