// pm_bin.cu -- cell sort: bin particles by mesh tile and boundary class (counting sort).
//
// Not in the paper (which only says "efficient CUDA implementations of scatter and gather", PAPER.md
// L496); named by BASELINE.json north_star ("particles cell-sorted ... each step").  The sort exists so
// that the CIC kernels (eq. 10) can work tile by tile out of shared memory:
//   key(j) = tile(j) * 8 + class(j),  class bit d = particle in the last cell layer of its tile along d
//   rec[slot] = {X, Y, Z, j}: absolute position in fixed point (cell << fbits | fraction) + particle id
// histogram (warp-aggregated global atomics) -> exclusive scan -> reorder (warp-aggregated cursors).
// The order of particles inside one key is arbitrary; nothing downstream depends on it (the scatter
// accumulates in integer fixed point, which is associative).
#include "pm_internal.cuh"

namespace pm {

struct BinGeom {
    unsigned long long M[3];      // N << fbits
    unsigned long long qstep[3];  // lattice spacing in fixed point
    int N[3], L[3], nt[3];
    int fbits;
    int pow2[3];                  // N power of two
};

__device__ __forceinline__ unsigned int wrap_fixed(long long v, unsigned long long M, int pow2)
{
    if (pow2) return (unsigned int)((unsigned long long)v & (M - 1ull));
    long long m = (long long)M;
    long long r = v % m;
    if (r < 0) r += m;
    return (unsigned int)r;
}

// absolute fixed-point position of particle j
template <bool FROM_STATE>
__device__ __forceinline__ void load_position(const BinGeom &g, long long j, const float *__restrict__ x,
                                              const int *__restrict__ s, unsigned int X[3])
{
    if (FROM_STATE) {
        long long jz = j % g.L[2], t = j / g.L[2];
        long long jy = t % g.L[1], jx = t / g.L[1];
        long long jj[3] = {jx, jy, jz};
#pragma unroll
        for (int d = 0; d < 3; d++) {
            long long v = (long long)(jj[d] * g.qstep[d]) + (long long)s[3 * j + d];
            X[d] = wrap_fixed(v, g.M[d], g.pow2[d]);
        }
    } else {
        const double sc = (double)(1u << g.fbits);
#pragma unroll
        for (int d = 0; d < 3; d++) {
            double xv = (double)x[3 * j + d] * sc;  // exact: power-of-two scaling of an fp32
            long long v = (long long)floor(xv);
            X[d] = wrap_fixed(v, g.M[d], g.pow2[d]);
        }
    }
}

__device__ __forceinline__ int key_of(const BinGeom &g, const unsigned int X[3])
{
    int c0 = (int)(X[0] >> g.fbits), c1 = (int)(X[1] >> g.fbits), c2 = (int)(X[2] >> g.fbits);
    int t0 = c0 / TX, t1 = c1 / TY, t2 = c2 / TZ;
    int e0 = min(t0 * TX + TX, g.N[0]) - 1, e1 = min(t1 * TY + TY, g.N[1]) - 1, e2 = min(t2 * TZ + TZ, g.N[2]) - 1;
    int cls = ((c0 == e0) << 2) | ((c1 == e1) << 1) | (int)(c2 == e2);
    return ((t0 * g.nt[1] + t1) * g.nt[2] + t2) * NCLS + cls;
}

// one atomic per distinct key in the warp; returns this lane's slot (base of its group + rank)
__device__ __forceinline__ int warp_aggregated_inc(int *ctr, int key, bool active)
{
    unsigned int act = __ballot_sync(0xffffffffu, active);
    if (!active) return 0;
    unsigned int peers = __match_any_sync(act, key);
    int lane = threadIdx.x & 31;
    int leader = __ffs(peers) - 1;
    int rank = __popc(peers & ((1u << lane) - 1u));
    int base = 0;
    if (lane == leader) base = atomicAdd(ctr + key, __popc(peers));
    base = __shfl_sync(peers, base, leader);
    return base + rank;
}

template <bool FROM_STATE>
__global__ void __launch_bounds__(256) bin_count_kernel(BinGeom g, long long np, const float *__restrict__ x,
                                                        const int *__restrict__ s, int *__restrict__ hist)
{
    long long stride = (long long)gridDim.x * blockDim.x;
    long long n_round = (np + 31) / 32 * 32;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < n_round; j += stride) {
        bool active = j < np;
        int key = 0;
        if (active) {
            unsigned int X[3];
            load_position<FROM_STATE>(g, j, x, s, X);
            key = key_of(g, X);
        }
        warp_aggregated_inc(hist, key, active);
    }
}

template <bool FROM_STATE>
__global__ void __launch_bounds__(256) bin_reorder_kernel(BinGeom g, long long np, const float *__restrict__ x,
                                                          const int *__restrict__ s, int *__restrict__ cursor,
                                                          uint4 *__restrict__ rec)
{
    long long stride = (long long)gridDim.x * blockDim.x;
    long long n_round = (np + 31) / 32 * 32;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < n_round; j += stride) {
        bool active = j < np;
        int key = 0;
        unsigned int X[3] = {0, 0, 0};
        if (active) {
            load_position<FROM_STATE>(g, j, x, s, X);
            key = key_of(g, X);
        }
        int slot = warp_aggregated_inc(cursor, key, active);
        if (active) rec[slot] = make_uint4(X[0], X[1], X[2], (unsigned int)j);
    }
}

// ---- exclusive scan of n ints: 3 kernels, 4096 elements per block ---------------------------------
constexpr int SCAN_T = 1024, SCAN_PER = 4, SCAN_CH = SCAN_T * SCAN_PER;

__device__ __forceinline__ int block_exclusive_scan(int v, int *total)
{
    __shared__ int wsum[32];
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    if (w == 0) {
        int ws = wsum[lane];
        int winc = ws;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += t;
        }
        wsum[lane] = winc - ws;  // exclusive warp offsets
        if (lane == 31) *total = winc;
    }
    __syncthreads();
    int r = wsum[w] + inc - v;
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(SCAN_T) scan_reduce_kernel(const int *__restrict__ in, int n, int *__restrict__ bsum)
{
    __shared__ int tot;
    int base = blockIdx.x * SCAN_CH + threadIdx.x * SCAN_PER;
    int v = 0;
#pragma unroll
    for (int k = 0; k < SCAN_PER; k++)
        if (base + k < n) v += in[base + k];
    block_exclusive_scan(v, &tot);
    if (threadIdx.x == 0) bsum[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(SCAN_T) scan_top_kernel(int *__restrict__ bsum, int nb)
{
    __shared__ int tot;
    __shared__ int carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nb; b0 += SCAN_T) {
        int i = b0 + threadIdx.x;
        int v = i < nb ? bsum[i] : 0;
        int ex = block_exclusive_scan(v, &tot);
        int carry = carry_s;
        if (i < nb) bsum[i] = ex + carry;
        __syncthreads();
        if (threadIdx.x == 0) carry_s = carry + tot;
        __syncthreads();
    }
}

// reads the histogram from `cursor`, writes the exclusive prefix to both offsets and cursor
__global__ void __launch_bounds__(SCAN_T) scan_final_kernel(int *__restrict__ cursor, int n, const int *__restrict__ bsum,
                                                            int *__restrict__ offsets)
{
    __shared__ int tot;
    int base = blockIdx.x * SCAN_CH + threadIdx.x * SCAN_PER;
    int v[SCAN_PER], sum = 0;
#pragma unroll
    for (int k = 0; k < SCAN_PER; k++) {
        v[k] = base + k < n ? cursor[base + k] : 0;
        sum += v[k];
    }
    int ex = block_exclusive_scan(sum, &tot) + bsum[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_PER; k++) {
        if (base + k < n) {
            offsets[base + k] = ex;
            cursor[base + k] = ex;
        }
        ex += v[k];
    }
}

static BinGeom make_bin_geom(const Geometry &g)
{
    BinGeom b;
    for (int d = 0; d < 3; d++) {
        b.M[d] = (unsigned long long)g.N[d] << g.fbits;
        b.qstep[d] = g.qstep[d];
        b.N[d] = g.N[d];
        b.L[d] = g.L[d];
        b.nt[d] = g.nt[d];
        b.pow2[d] = (g.N[d] & (g.N[d] - 1)) == 0;
    }
    b.fbits = g.fbits;
    return b;
}

int bin_particles(pm_ctx *c, long long np, const float *x)
{
    const Geometry &g = c->g;
    BinGeom b = make_bin_geom(g);
    int n = g.nkeys + 1;  // the extra entry makes offsets[nkeys] = np
    PM_CUDA(c, cudaMemsetAsync(c->cursor, 0, sizeof(int) * (size_t)n, c->stream));
    int blocks = (int)((np + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (blocks < 1) blocks = 1;
    {
        Timer t(c, TC_BIN_COUNT, 12.0 * np);
        if (x)
            bin_count_kernel<false><<<blocks, 256, 0, c->stream>>>(b, np, x, nullptr, c->cursor);
        else
            bin_count_kernel<true><<<blocks, 256, 0, c->stream>>>(b, np, nullptr, c->s, c->cursor);
        PM_LAUNCH_CHECK(c, "bin_count_kernel");
        t.stop();
    }
    {
        Timer t(c, TC_BIN_SCAN, 12.0 * n);
        int nb = (n + SCAN_CH - 1) / SCAN_CH;
        scan_reduce_kernel<<<nb, SCAN_T, 0, c->stream>>>(c->cursor, n, c->blocksum);
        scan_top_kernel<<<1, SCAN_T, 0, c->stream>>>(c->blocksum, nb);
        scan_final_kernel<<<nb, SCAN_T, 0, c->stream>>>(c->cursor, n, c->blocksum, c->offsets);
        PM_LAUNCH_CHECK(c, "scan kernels");
        c->n_own += 2;
        t.stop();
    }
    {
        Timer t(c, TC_BIN_REORDER, 28.0 * np);
        if (x)
            bin_reorder_kernel<false><<<blocks, 256, 0, c->stream>>>(b, np, x, nullptr, c->cursor, c->rec);
        else
            bin_reorder_kernel<true><<<blocks, 256, 0, c->stream>>>(b, np, nullptr, c->s, c->cursor, c->rec);
        PM_LAUNCH_CHECK(c, "bin_reorder_kernel");
        t.stop();
    }
    return PM_OK;
}

}  // namespace pm
