// pm_bin.cu -- cell sort: bin particles by mesh tile and boundary class (counting sort).
//
// Not in the paper (which only says "efficient CUDA implementations of scatter and gather", PAPER.md
// L496); named by BASELINE.json north_star ("particles cell-sorted ... each step").  The sort exists so
// that the CIC kernels (eq. 10) can work tile by tile out of shared memory:
//   key(j) = tile(j) * 8 + class(j),  class bit d = particle in the last cell layer of its tile along d
//   rec[slot] = {X, Y, Z, j}: absolute position in fixed point (cell << fbits | fraction) + particle id
// histogram (warp-aggregated global atomics; normally produced by the kernel that moved the particles: the
// fused gather + kick + drift of pm_cic.cu or kick_drift of pm_integrate.cu) -> exclusive scan -> reorder
// (warp-aggregated cursors).
// The order of particles inside one key is arbitrary; nothing downstream depends on it (the scatter
// accumulates in integer fixed point, which is associative).
#include "pm_pos.cuh"

namespace pm {

PosGeom make_pos_geom(const Geometry &g)
{
    PosGeom b;
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

// record coordinate of particle j: from the integrator state (FROM_STATE) or from absolute float positions
template <bool FROM_STATE>
__device__ __forceinline__ void load_position(const PosGeom &g, long long j, const float *__restrict__ x,
                                              const long long *__restrict__ xs, unsigned int X[3])
{
    if (FROM_STATE) {
#pragma unroll
        for (int d = 0; d < 3; d++) X[d] = record_coord(g, xs[3 * j + d], d);
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
__global__ void __launch_bounds__(256) bin_count_kernel(PosGeom g, long long np, const float *__restrict__ x,
                                                        const long long *__restrict__ xs, int *__restrict__ hist)
{
    pdl_enter();
    long long stride = (long long)gridDim.x * blockDim.x;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < np; j += stride) {
        unsigned int X[3];
        load_position<FROM_STATE>(g, j, x, xs, X);
        hist_add(hist, key_of(g, X));
    }
}

template <bool FROM_STATE>
__global__ void __launch_bounds__(256) bin_reorder_kernel(PosGeom g, long long np, const float *__restrict__ x,
                                                          const long long *__restrict__ xs, int *__restrict__ cursor,
                                                          uint4 *__restrict__ rec)
{
    pdl_enter();
    long long stride = (long long)gridDim.x * blockDim.x;
    long long n_round = (np + 31) / 32 * 32;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < n_round; j += stride) {
        bool active = j < np;
        int key = 0;
        unsigned int X[3] = {0, 0, 0};
        if (active) {
            load_position<FROM_STATE>(g, j, x, xs, X);
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

// Single-pass exclusive scan with decoupled look-back: block b publishes its total tagged with the launch's
// epoch (one 64-bit word, so tag and value arrive together; no reset between launches), then adds up the totals
// of all lower blocks.  A block waits only on lower-numbered blocks, which the hardware dispatches first.
// Reads (and clears) the histogram, writes the exclusive prefix to both offsets and cursor.
__global__ void __launch_bounds__(SCAN_T) scan_kernel(int *__restrict__ hist, int n, int *__restrict__ offsets,
                                                      int *__restrict__ cursor, unsigned long long *agg, unsigned int epoch)
{
    __shared__ int tot;
    __shared__ int base_s;
    pdl_enter();
    const int base = blockIdx.x * SCAN_CH + threadIdx.x * SCAN_PER;
    int v[SCAN_PER], sum = 0;
    if (base + SCAN_PER <= n) {
        int4 h = *reinterpret_cast<const int4 *>(hist + base);
        v[0] = h.x; v[1] = h.y; v[2] = h.z; v[3] = h.w;
    } else {
#pragma unroll
        for (int k = 0; k < SCAN_PER; k++) v[k] = base + k < n ? hist[base + k] : 0;
    }
#pragma unroll
    for (int k = 0; k < SCAN_PER; k++) sum += v[k];
    int ex = block_exclusive_scan(sum, &tot);
    if (threadIdx.x == 0) {
        unsigned long long w = ((unsigned long long)epoch << 32) | (unsigned int)tot;
        asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(agg + blockIdx.x), "l"(w) : "memory");
    }
    if (threadIdx.x < 32) {
        int acc = 0;
        for (int b = threadIdx.x; b < (int)blockIdx.x; b += 32) {
            unsigned long long w;
            do {
                asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(w) : "l"(agg + b) : "memory");
            } while ((unsigned int)(w >> 32) != epoch);
            acc += (int)(unsigned int)w;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (threadIdx.x == 0) base_s = acc;
    }
    __syncthreads();
    ex += base_s;
    int o[SCAN_PER];
#pragma unroll
    for (int k = 0; k < SCAN_PER; k++) { o[k] = ex; ex += v[k]; }
    if (base + SCAN_PER <= n) {
        *reinterpret_cast<int4 *>(offsets + base) = make_int4(o[0], o[1], o[2], o[3]);
        *reinterpret_cast<int4 *>(cursor + base) = make_int4(o[0], o[1], o[2], o[3]);
        *reinterpret_cast<int4 *>(hist + base) = make_int4(0, 0, 0, 0);
    } else {
#pragma unroll
        for (int k = 0; k < SCAN_PER; k++)
            if (base + k < n) { offsets[base + k] = o[k]; cursor[base + k] = o[k]; hist[base + k] = 0; }
    }
}

static int bin_blocks(long long np)
{
    long long blocks = (np + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (blocks < 1) blocks = 1;
    return (int)blocks;
}

// key histogram of np particles (absolute float positions x, or the ctx state when x == NULL) into c->hist,
// which must be all zero on entry (it is between sorts: the scan clears it)
int bin_count(pm_ctx *c, long long np, const float *x)
{
    PosGeom b = make_pos_geom(c->g);
    Timer t(c, TC_BIN_COUNT, (x ? 12.0 : 24.0) * np);
    if (x)
        PM_CUDA(c, launch_pdl(bin_count_kernel<false>, dim3(bin_blocks(np)), dim3(256), 0, c->stream, b, np, x, nullptr, c->hist));
    else
        PM_CUDA(c, launch_pdl(bin_count_kernel<true>, dim3(bin_blocks(np)), dim3(256), 0, c->stream, b, np, nullptr, c->x, c->hist));
    PM_LAUNCH_CHECK(c, "bin_count_kernel");
    t.stop();
    return PM_OK;
}

// c->hist -> offsets (exclusive scan) -> sorted records; leaves c->hist zero
int bin_sort(pm_ctx *c, long long np, const float *x)
{
    const Geometry &g = c->g;
    PosGeom b = make_pos_geom(g);
    int n = g.nkeys + 1;  // the extra entry makes offsets[nkeys] = np
    {
        Timer t(c, TC_BIN_SCAN, 16.0 * n);
        int nb = (n + SCAN_CH - 1) / SCAN_CH;
        c->scan_epoch++;
        if (c->scan_epoch == 0) c->scan_epoch = 1;  // 0 is the tag of the zero-initialised buffer
        PM_CUDA(c, launch_pdl(scan_kernel, dim3(nb), dim3(SCAN_T), 0, c->stream, c->hist, n, c->offsets, c->cursor, c->scan_agg, c->scan_epoch));
        PM_LAUNCH_CHECK(c, "scan kernels");
        t.stop();
    }
    {
        Timer t(c, TC_BIN_REORDER, (x ? 28.0 : 40.0) * np);
        if (x)
            PM_CUDA(c, launch_pdl(bin_reorder_kernel<false>, dim3(bin_blocks(np)), dim3(256), 0, c->stream, b, np, x, nullptr, c->cursor, c->rec));
        else
            PM_CUDA(c, launch_pdl(bin_reorder_kernel<true>, dim3(bin_blocks(np)), dim3(256), 0, c->stream, b, np, nullptr, c->x, c->cursor, c->rec));
        PM_LAUNCH_CHECK(c, "bin_reorder_kernel");
        t.stop();
    }
    return PM_OK;
}

}  // namespace pm
