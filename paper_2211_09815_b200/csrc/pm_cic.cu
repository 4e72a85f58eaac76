// pm_cic.cu -- cloud-in-cell scatter / gather / weight-gradient gather, tile by tile out of shared memory.
//
// PAPER.md eq. 10 (L121-125): W(x, x') = prod_d max(1 - |x_d - x'_d| / l, 0), l = 1 cell; the gather
// "interpolates ... from the same grid points with the same weights" (L133); their VJPs (L410) are a
// scatter of cotangents (value argument) and a weight-gradient gather (position argument).
// Cell i_d = floor(x_d), t_d = x_d - i_d in [0,1): weight (1 - t_d) at i_d, t_d at i_d + 1 (periodic),
// derivative -1 / +1 (floor convention, right derivative; R7).
//
// Input: the records sorted by (tile, class) of pm_bin.cu.  One CTA per mesh tile of TX x TY x TZ cells.
//
// scatter -- OUTPUT-STATIONARY: the CTA owns the mesh points of its tile, pulls the particles of its
//   own tile plus the last-cell-layer classes of its (up to 7) low-side neighbour tiles, accumulates in
//   shared memory with NATIVE int32 atomics (fp32 shared atomics are CAS loops on sm_100a) in fixed
//   point with a per-tile power-of-two scale chosen from sum|v| so that it cannot overflow, and writes
//   every mesh point exactly once with a plain coalesced store: no zero-fill pass, no global atomics,
//   and a result that does not depend on the order in which particles arrive (bit-reproducible).
// gather -- the CTA stages the (TX+1)(TY+1)(TZ+1) halo of each mesh in shared memory and interpolates
//   for the particles of its own tile; results go to out[j] in the caller's particle order.
#include "pm_internal.cuh"

namespace pm {

struct CicGeom {
    int N[3], nt[3];
    int fbits;
    int zs;        // floats per z-row
    long long ms;  // floats per mesh (component stride)
};

// the 14 contiguous class runs a tile pulls from itself (m = 0) and its low neighbours
// m: bit 2/1/0 = neighbour is one tile lower in x/y/z; classes [c0, c1)
__constant__ signed char kRuns[14][3] = {{0, 0, 8}, {4, 4, 8}, {2, 2, 4}, {2, 6, 8}, {1, 1, 2}, {1, 3, 4}, {1, 5, 6},
                                         {1, 7, 8}, {6, 6, 8}, {5, 5, 6}, {5, 7, 8}, {3, 3, 4}, {3, 7, 8}, {7, 7, 8}};
constexpr int NRUNS = 14;
constexpr int TILE_PTS = TX * TY * TZ;

__device__ __forceinline__ void tile_coords(const CicGeom &g, int tile, int t[3], int t0[3], int ext[3])
{
    t[2] = tile % g.nt[2];
    int r = tile / g.nt[2];
    t[1] = r % g.nt[1];
    t[0] = r / g.nt[1];
    t0[0] = t[0] * TX; t0[1] = t[1] * TY; t0[2] = t[2] * TZ;
    ext[0] = min(TX, g.N[0] - t0[0]);
    ext[1] = min(TY, g.N[1] - t0[1]);
    ext[2] = min(TZ, g.N[2] - t0[2]);
}

__device__ __forceinline__ float block_sum(float v, float *sh /*>= 32 floats*/)
{
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) sh[w] = v;
    __syncthreads();
    float r = 0.f;
    for (int k = 0; k < nw; k++) r += sh[k];  // same order in every thread
    __syncthreads();
    return r;
}

// --------------------------------------------------------------------------------------------------
// scatter
// --------------------------------------------------------------------------------------------------
template <int C, bool HAS_VAL>
__global__ void __launch_bounds__(256) scatter_kernel(CicGeom g, const uint4 *__restrict__ rec,
                                                      const int *__restrict__ offsets,
                                                      const float *__restrict__ val, float *__restrict__ mesh)
{
    __shared__ int tile_acc[C][TILE_PTS];
    __shared__ int run_start[NRUNS];
    __shared__ int run_prefix[NRUNS + 1];
    __shared__ float red[32];

    int t[3], t0[3], ext[3];
    tile_coords(g, blockIdx.x, t, t0, ext);

    for (int i = threadIdx.x; i < C * TILE_PTS; i += blockDim.x) (&tile_acc[0][0])[i] = 0;
    if (threadIdx.x < NRUNS) {
        int m = kRuns[threadIdx.x][0], c0 = kRuns[threadIdx.x][1], c1 = kRuns[threadIdx.x][2];
        bool valid = true;
        int n[3];
#pragma unroll
        for (int d = 0; d < 3; d++) {
            int low = (m >> (2 - d)) & 1;
            if (low && g.nt[d] == 1) valid = false;  // the only tile along d is its own neighbour
            n[d] = t[d] - low;
            if (n[d] < 0) n[d] += g.nt[d];
        }
        int key = ((n[0] * g.nt[1] + n[1]) * g.nt[2] + n[2]) * NCLS;
        int b = 0, e = 0;
        if (valid) { b = offsets[key + c0]; e = offsets[key + c1]; }
        run_start[threadIdx.x] = b;
        run_prefix[threadIdx.x + 1] = e - b;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        run_prefix[0] = 0;
        for (int r = 0; r < NRUNS; r++) run_prefix[r + 1] += run_prefix[r];
    }
    __syncthreads();
    const int total = run_prefix[NRUNS];

    // bound on the absolute sum any mesh point can reach -> power-of-two fixed-point scale
    float bound;
    if (HAS_VAL) {
        float part = 0.f;
        for (int i = threadIdx.x; i < total; i += blockDim.x) {
            int r = 0;
            while (i >= run_prefix[r + 1]) r++;
            unsigned int j = rec[run_start[r] + (i - run_prefix[r])].w;
            float m = 0.f;
#pragma unroll
            for (int c = 0; c < C; c++) m = fmaxf(m, fabsf(val[(size_t)j * C + c]));
            part += m;
        }
        bound = block_sum(part, red) * 1.0001f;  // margin for the fp32 summation itself
    } else {
        bound = (float)total;
    }
    int ex;
    frexpf(fmaxf(bound, 1e-37f), &ex);       // bound <= 2^ex
    int k = min(30 - ex, 96);
    const float scale = ldexpf(1.f, k), inv_scale = ldexpf(1.f, -k);
    const float fr = 1.f / (float)(1u << g.fbits);
    const unsigned int fmask = (1u << g.fbits) - 1u;

    for (int i = threadIdx.x; i < total; i += blockDim.x) {
        int r = 0;
        while (i >= run_prefix[r + 1]) r++;
        uint4 q = rec[run_start[r] + (i - run_prefix[r])];
        float v[C];
        if (HAS_VAL) {
#pragma unroll
            for (int c = 0; c < C; c++) v[c] = val[(size_t)q.w * C + c] * scale;
        } else {
#pragma unroll
            for (int c = 0; c < C; c++) v[c] = scale;
        }
        unsigned int X[3] = {q.x, q.y, q.z};
        int l[3][2];     // local mesh-point index of the two corners per axis, or -1 when not owned
        float w[3][2];
#pragma unroll
        for (int d = 0; d < 3; d++) {
            int cd = (int)(X[d] >> g.fbits);
            float td = (float)(X[d] & fmask) * fr;
            w[d][0] = 1.f - td;
            w[d][1] = td;
#pragma unroll
            for (int b = 0; b < 2; b++) {
                int gd = cd + b;
                if (gd == g.N[d]) gd = 0;
                int ld = gd - t0[d];
                if (ld < 0) ld += g.N[d];
                l[d][b] = (ld < ext[d]) ? ld : -1;
            }
        }
#pragma unroll
        for (int bx = 0; bx < 2; bx++)
#pragma unroll
            for (int by = 0; by < 2; by++)
#pragma unroll
                for (int bz = 0; bz < 2; bz++) {
                    if ((l[0][bx] | l[1][by] | l[2][bz]) < 0) continue;
                    float ww = w[0][bx] * w[1][by] * w[2][bz];
                    int idx = (l[0][bx] * TY + l[1][by]) * TZ + l[2][bz];
#pragma unroll
                    for (int c = 0; c < C; c++) atomicAdd(&tile_acc[c][idx], __float2int_rn(ww * v[c]));
                }
    }
    __syncthreads();

    for (int i = threadIdx.x; i < TILE_PTS; i += blockDim.x) {
        int lz = i % TZ, r = i / TZ;
        int ly = r % TY, lx = r / TY;
        if (lx < ext[0] && ly < ext[1] && lz < ext[2]) {
            size_t o = ((size_t)(t0[0] + lx) * g.N[1] + (t0[1] + ly)) * g.zs + (t0[2] + lz);
#pragma unroll
            for (int c = 0; c < C; c++) mesh[(size_t)c * g.ms + o] = (float)tile_acc[c][i] * inv_scale;
        }
    }
}

// --------------------------------------------------------------------------------------------------
// gathers
// --------------------------------------------------------------------------------------------------
constexpr int HX = TX + 1, HY = TY + 1, HZ = TZ + 1;
constexpr int HALO_PTS = HX * HY * HZ;
enum GatherMode { G_VALUE = 0, G_GRAD = 1, G_FUSED = 2 };

template <int C, int MODE, bool HAS_COT>
__global__ void __launch_bounds__(256) gather_kernel(CicGeom g, const uint4 *__restrict__ rec,
                                                     const int *__restrict__ offsets,
                                                     const float *__restrict__ mesh, const float *__restrict__ cot,
                                                     float cot_scale, float *__restrict__ out, float *__restrict__ out2)
{
    __shared__ float halo[C][HALO_PTS];
    int t[3], t0[3], ext[3];
    tile_coords(g, blockIdx.x, t, t0, ext);
    const int key0 = blockIdx.x * NCLS;
    const int beg = offsets[key0], end = offsets[key0 + NCLS];
    if (beg == end) return;

    for (int i = threadIdx.x; i < HALO_PTS; i += blockDim.x) {
        int lz = i % HZ, r = i / HZ;
        int ly = r % HY, lx = r / HY;
        if (lx <= ext[0] && ly <= ext[1] && lz <= ext[2]) {
            int gx = t0[0] + lx, gy = t0[1] + ly, gz = t0[2] + lz;
            if (gx >= g.N[0]) gx -= g.N[0];
            if (gy >= g.N[1]) gy -= g.N[1];
            if (gz >= g.N[2]) gz -= g.N[2];
            size_t o = ((size_t)gx * g.N[1] + gy) * g.zs + gz;
#pragma unroll
            for (int c = 0; c < C; c++) halo[c][i] = mesh[(size_t)c * g.ms + o];
        }
    }
    __syncthreads();

    const float fr = 1.f / (float)(1u << g.fbits);
    const unsigned int fmask = (1u << g.fbits) - 1u;
    for (int i = beg + threadIdx.x; i < end; i += blockDim.x) {
        uint4 q = rec[i];
        unsigned int X[3] = {q.x, q.y, q.z};
        int l[3];
        float w[3][2];
#pragma unroll
        for (int d = 0; d < 3; d++) {
            l[d] = (int)(X[d] >> g.fbits) - t0[d];
            float td = (float)(X[d] & fmask) * fr;
            w[d][0] = 1.f - td;
            w[d][1] = td;
        }
        const int base = (l[0] * HY + l[1]) * HZ + l[2];
        const size_t j = q.w;
        float cv[C];
        if (MODE == G_GRAD) {
#pragma unroll
            for (int c = 0; c < C; c++) cv[c] = HAS_COT ? cot[j * C + c] : 1.f;
        }
        if (MODE == G_FUSED) {
            cv[0] = 1.f;
#pragma unroll
            for (int c = 1; c < C; c++) cv[c] = cot[j * 3 + (c - 1)];
        }
        float val[C];
        float gr[3] = {0.f, 0.f, 0.f};
#pragma unroll
        for (int c = 0; c < C; c++) val[c] = 0.f;
#pragma unroll
        for (int bx = 0; bx < 2; bx++)
#pragma unroll
            for (int by = 0; by < 2; by++)
#pragma unroll
                for (int bz = 0; bz < 2; bz++) {
                    const int idx = base + (bx * HY + by) * HZ + bz;
                    const float W = w[0][bx] * w[1][by] * w[2][bz];
                    const float dWx = (bx ? 1.f : -1.f) * w[1][by] * w[2][bz];
                    const float dWy = (by ? 1.f : -1.f) * w[0][bx] * w[2][bz];
                    const float dWz = (bz ? 1.f : -1.f) * w[0][bx] * w[1][by];
                    float m = 0.f;  // cotangent-weighted mesh value at this corner
#pragma unroll
                    for (int c = 0; c < C; c++) {
                        float f = halo[c][idx];
                        if (MODE != G_GRAD) val[c] += W * f;
                        if (MODE != G_VALUE) m += cv[c] * f;
                    }
                    if (MODE != G_VALUE) {
                        gr[0] += dWx * m;
                        gr[1] += dWy * m;
                        gr[2] += dWz * m;
                    }
                }
        if (MODE == G_VALUE) {
#pragma unroll
            for (int c = 0; c < C; c++) out[j * C + c] = val[c];
        } else if (MODE == G_GRAD) {
#pragma unroll
            for (int e = 0; e < 3; e++) out[j * 3 + e] = gr[e] * cot_scale;
        } else {
#pragma unroll
            for (int e = 0; e < 3; e++) {
                out[j * 3 + e] = val[1 + e];
                out2[j * 3 + e] = gr[e];
            }
        }
    }
}

static CicGeom make_cic_geom(const Geometry &g, int zs, long long ms)
{
    CicGeom c;
    for (int d = 0; d < 3; d++) { c.N[d] = g.N[d]; c.nt[d] = g.nt[d]; }
    c.fbits = g.fbits;
    c.zs = zs;
    c.ms = ms;
    return c;
}

int scatter_sorted(pm_ctx *c, const float *val, int C, float *mesh, int zs, long long ms)
{
    CicGeom g = make_cic_geom(c->g, zs, ms);
    double np = (double)c->g.np, ng = (double)c->g.ng;
    if (C == 1 && !val) {
        Timer t(c, TC_SCATTER1, 12.0 * np + 4.0 * ng);
        scatter_kernel<1, false><<<c->g.ntiles, 256, 0, c->stream>>>(g, c->rec, c->offsets, nullptr, mesh);
        PM_LAUNCH_CHECK(c, "scatter_kernel<1>");
        t.stop();
    } else if (C == 1) {
        Timer t(c, TC_SCATTER1, 16.0 * np + 4.0 * ng);
        scatter_kernel<1, true><<<c->g.ntiles, 256, 0, c->stream>>>(g, c->rec, c->offsets, val, mesh);
        PM_LAUNCH_CHECK(c, "scatter_kernel<1,val>");
        t.stop();
    } else if (C == 3 && val) {
        Timer t(c, TC_SCATTER3, 24.0 * np + 12.0 * ng);
        scatter_kernel<3, true><<<c->g.ntiles, 256, 0, c->stream>>>(g, c->rec, c->offsets, val, mesh);
        PM_LAUNCH_CHECK(c, "scatter_kernel<3,val>");
        t.stop();
    } else {
        return fail(c, PM_EINVAL, "scatter", "C must be 1, or 3 with values");
    }
    return PM_OK;
}

int gather_sorted(pm_ctx *c, const float *mesh, int C, int zs, long long ms, float *out)
{
    CicGeom g = make_cic_geom(c->g, zs, ms);
    double np = (double)c->g.np, ng = (double)c->g.ng;
    if (C == 1) {
        Timer t(c, TC_GATHER3, 16.0 * np + 4.0 * ng);
        gather_kernel<1, G_VALUE, false><<<c->g.ntiles, 256, 0, c->stream>>>(g, c->rec, c->offsets, mesh, nullptr, 1.f, out, nullptr);
        PM_LAUNCH_CHECK(c, "gather_kernel<1>");
        t.stop();
    } else if (C == 3) {
        Timer t(c, TC_GATHER3, 24.0 * np + 12.0 * ng);
        gather_kernel<3, G_VALUE, false><<<c->g.ntiles, 256, 0, c->stream>>>(g, c->rec, c->offsets, mesh, nullptr, 1.f, out, nullptr);
        PM_LAUNCH_CHECK(c, "gather_kernel<3>");
        t.stop();
    } else {
        return fail(c, PM_EINVAL, "gather", "C must be 1 or 3");
    }
    return PM_OK;
}

int gather_grad_sorted(pm_ctx *c, const float *mesh, int C, int zs, long long ms, const float *cot, float cot_scale,
                       float *out)
{
    CicGeom g = make_cic_geom(c->g, zs, ms);
    double np = (double)c->g.np, ng = (double)c->g.ng;
    Timer t(c, TC_GATHER_GRAD, (24.0 + (cot ? 4.0 * C : 0.0)) * np + 4.0 * C * ng);
    if (C == 1 && !cot)
        gather_kernel<1, G_GRAD, false><<<c->g.ntiles, 256, 0, c->stream>>>(g, c->rec, c->offsets, mesh, nullptr, cot_scale, out, nullptr);
    else if (C == 1)
        gather_kernel<1, G_GRAD, true><<<c->g.ntiles, 256, 0, c->stream>>>(g, c->rec, c->offsets, mesh, cot, cot_scale, out, nullptr);
    else if (C == 3 && !cot)
        gather_kernel<3, G_GRAD, false><<<c->g.ntiles, 256, 0, c->stream>>>(g, c->rec, c->offsets, mesh, nullptr, cot_scale, out, nullptr);
    else if (C == 3)
        gather_kernel<3, G_GRAD, true><<<c->g.ntiles, 256, 0, c->stream>>>(g, c->rec, c->offsets, mesh, cot, cot_scale, out, nullptr);
    else
        return fail(c, PM_EINVAL, "gather_grad", "C must be 1 or 3");
    PM_LAUNCH_CHECK(c, "gather_kernel<grad>");
    t.stop();
    return PM_OK;
}

int gather_fused_sorted(pm_ctx *c, const float *mesh4, int zs, long long ms, const float *pi, float *acc, float *alpha)
{
    CicGeom g = make_cic_geom(c->g, zs, ms);
    double np = (double)c->g.np, ng = (double)c->g.ng;
    Timer t(c, TC_GATHER_FUSED, 48.0 * np + 16.0 * ng);
    gather_kernel<4, G_FUSED, true><<<c->g.ntiles, 256, 0, c->stream>>>(g, c->rec, c->offsets, mesh4, pi, 1.f, acc, alpha);
    PM_LAUNCH_CHECK(c, "gather_kernel<fused>");
    t.stop();
    return PM_OK;
}

}  // namespace pm
