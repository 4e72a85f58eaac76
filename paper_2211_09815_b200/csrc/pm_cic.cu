// pm_cic.cu -- cloud-in-cell scatter / gather / weight-gradient gather, tile by tile out of shared memory.
//
// PAPER.md eq. 10 (L121-125): W(x, x') = prod_d max(1 - |x_d - x'_d| / l, 0), l = 1 cell; the gather
// "interpolates ... from the same grid points with the same weights" (L133); their VJPs (L410) are a
// scatter of cotangents (value argument) and a weight-gradient gather (position argument).
// Cell i_d = floor(x_d), t_d = x_d - i_d in [0,1): weight (1 - t_d) at i_d, t_d at i_d + 1 (periodic),
// derivative -1 / +1 (floor convention, right derivative; R7).
//
// Input: the records sorted by (tile, class) of pm_bin.cu.  One CTA per mesh tile of TX x TY x TZ cells,
// grid = (tiles_z, tiles_y, tiles_x).
//
// scatter -- OUTPUT-STATIONARY: the CTA owns the mesh points of its tile, pulls the particles of its
//   own tile plus the last-cell-layer classes of its (up to 7) low-side neighbour tiles, accumulates in
//   shared memory with NATIVE int32 atomics (fp32 shared atomics are CAS loops on sm_100a) in fixed
//   point with a per-tile power-of-two scale chosen from sum|v| so that it cannot overflow, converts in
//   place and writes the tile with ONE TMA tensor store (cp.async.bulk.tensor, clipped at the mesh edge):
//   no zero-fill pass, no global atomics, every mesh point written exactly once, and a result that does
//   not depend on the order in which particles arrive (bit-reproducible).
// gather -- the halo box (TX+1)(TY+1)(TZ+4) of each mesh is brought into shared memory by TMA tensor
//   loads signalled on an mbarrier (tiles touching the upper mesh edge, whose halo wraps periodically,
//   and meshes whose layout TMA cannot address use plain coalesced row loads); the CTA then interpolates
//   for the particles of its own tile; results go to out[j] in the caller's particle order.
#include <cstdlib>

#include "pm_pos.cuh"

namespace pm {

struct CicGeom {
    int N[3], nt[3];
    int fbits;
    int zs;        // floats per z-row
    long long ms;  // floats per mesh (component stride)
    int use_tma;   // tensor map valid for this mesh
    int c0;        // first component (4th tensor-map coordinate)
    int kshift;    // debug: coarsen the scatter's fixed-point scale by this many bits (0 in production)
    double mean;   // unit-mass scatter only: constant subtracted from every mesh point IN INTEGER, before the
                   // int -> fp32 conversion (0 = plain density; nbar on the force path, whose k = 0 mode is zeroed
                   // anyway, so that fp32 rounding is relative to the fluctuation rho - nbar, not to rho)
};

constexpr int TILE_PTS = TX * TY * TZ;
constexpr int HX = TX + 1, HY = TY + 1, HZ = TZ + 1;
constexpr int HZP = TZ + 4;                               // halo row pitch: 144 bytes, a TMA-legal box width
constexpr int HALO_PTS = HX * HY * HZP;
constexpr int HALO_STRIDE = (HALO_PTS + 31) / 32 * 32;    // per-mesh stride in shared memory: 128-byte multiple

// ---- PTX wrappers: mbarrier + TMA (sm_90+/sm_100a) ----------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned phase)
{
    unsigned ok = 0;
    while (!ok) {
        asm volatile(
            "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(phase)
            : "memory");
    }
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *m, unsigned long long *bar, int z, int y, int x, int c)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(smem_u32(dst)), "l"((unsigned long long)m), "r"(smem_u32(bar)), "r"(z), "r"(y), "r"(x), "r"(c)
        : "memory");
}
__device__ __forceinline__ void tma_store_4d(const CUtensorMap *m, const void *src, int z, int y, int x, int c)
{
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5}], [%1];"
                 ::"l"((unsigned long long)m), "r"(smem_u32(src)), "r"(z), "r"(y), "r"(x), "r"(c)
                 : "memory");
}
__device__ __forceinline__ void tma_store_commit_and_wait()
{
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---- host: tensor maps ------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
        (void)cudaGetLastError();
    }
    return fn;
}

// 4-D view {z, y, x, component} of C meshes [Nx][Ny][zs] spaced ms floats apart; box = {bz, by, bx, 1}
static bool encode_mesh_map(CUtensorMap *out, const float *base, const int N[3], int C, int zs, long long ms, int bz,
                            int by, int bx)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    if (((uintptr_t)base & 15) || (zs & 3) || (ms & 3)) return false;  // 16-byte base and strides
    cuuint64_t dims[4] = {(cuuint64_t)N[2], (cuuint64_t)N[1], (cuuint64_t)N[0], (cuuint64_t)C};
    cuuint64_t strides[3] = {(cuuint64_t)zs * 4, (cuuint64_t)zs * 4 * (cuuint64_t)N[1], (cuuint64_t)ms * 4};
    cuuint32_t box[4] = {(cuuint32_t)bz, (cuuint32_t)by, (cuuint32_t)bx, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void *)base, dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

int cic_init_tensor_maps(pm_ctx *c)
{
    const Geometry &g = c->g;
    c->tma_ok = encode_mesh_map(&c->tmap_load, c->mesh[0], g.N, 7, g.zs, g.mesh_stride, HZP, HY, HX) &&
                encode_mesh_map(&c->tmap_store, c->mesh[0], g.N, 7, g.zs, g.mesh_stride, TZ, TY, TX);
    return PM_OK;
}

// picks the tensor map for a mesh pointer: the ctx's maps for internal meshes, a freshly encoded one otherwise
static CicGeom make_cic_geom(pm_ctx *c, const float *mesh, int C, int zs, long long ms, bool store, CUtensorMap *map)
{
    const Geometry &g = c->g;
    CicGeom r;
    for (int d = 0; d < 3; d++) { r.N[d] = g.N[d]; r.nt[d] = g.nt[d]; }
    r.fbits = g.fbits;
    r.zs = zs;
    r.ms = ms;
    r.use_tma = 0;
    r.c0 = 0;
    { const char *e = getenv("PM_DEBUG_KSHIFT"); r.kshift = e ? atoi(e) : 0; }
    r.mean = 0.0;
    memset(map, 0, sizeof(*map));
    long long off = mesh - c->mesh[0];
    bool internal = zs == g.zs && ms == g.mesh_stride && mesh >= c->mesh[0] && off % g.mesh_stride == 0 &&
                    off / g.mesh_stride + C <= 7;
    if (internal && c->tma_ok) {
        *map = store ? c->tmap_store : c->tmap_load;
        r.use_tma = 1;
        r.c0 = (int)(off / g.mesh_stride);
    } else if (!internal) {
        if (store ? encode_mesh_map(map, mesh, g.N, C, zs, ms, TZ, TY, TX) : encode_mesh_map(map, mesh, g.N, C, zs, ms, HZP, HY, HX))
            r.use_tma = 1;
    }
    return r;
}

__device__ __forceinline__ void tile_coords(const CicGeom &g, int t[3], int t0[3], int ext[3])
{
    t[0] = blockIdx.z; t[1] = blockIdx.y; t[2] = blockIdx.x;
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
// the 14 contiguous class runs a tile pulls from itself (m = 0) and its low neighbours
// m: bit 2/1/0 = neighbour is one tile lower in x/y/z; classes [c0, c1)
__constant__ signed char kRuns[14][3] = {{0, 0, 8}, {4, 4, 8}, {2, 2, 4}, {2, 6, 8}, {1, 1, 2}, {1, 3, 4}, {1, 5, 6},
                                         {1, 7, 8}, {6, 6, 8}, {5, 5, 6}, {5, 7, 8}, {3, 3, 4}, {3, 7, 8}, {7, 7, 8}};
constexpr int NRUNS = 14;

// predicated shared-memory integer reduction: no branch, no divergence region around the atomic
__device__ __forceinline__ void red_shared_if(int *addr, int v, bool ok)
{
    asm volatile("{\n .reg .pred p;\n setp.ne.s32 p, %2, 0;\n @p red.shared.add.s32 [%0], %1;\n}"
                 ::"r"(smem_u32(addr)), "r"(v), "r"((int)ok)
                 : "memory");
}

// deposit one particle into the CTA's tile: each of the 8 corners lands only if this tile owns that mesh point
template <int C, bool SIGNED>
__device__ __forceinline__ void deposit(const CicGeom &g, const int t0[3], const int ext[3], uint4 q, const float v[C],
                                        int (*tile_acc)[TILE_PTS], float fr, unsigned fmask)
{
    const unsigned X[3] = {q.x, q.y, q.z};
    int l[3][2];
    bool ok[3][2];
    float w[3][2];
#pragma unroll
    for (int d = 0; d < 3; d++) {
        int l0 = (int)(X[d] >> g.fbits) - t0[d];
        if (l0 < 0) l0 += g.N[d];          // particle of the low neighbour across the periodic edge
        int l1 = l0 + 1;
        if (l1 == g.N[d]) l1 = 0;          // the only tile along d is its own neighbour
        l[d][0] = l0;
        l[d][1] = l1;
        ok[d][0] = l0 < ext[d];
        ok[d][1] = l1 < ext[d];
        float td = (float)(X[d] & fmask) * fr;
        w[d][0] = 1.f - td;
        w[d][1] = td;
    }
#pragma unroll
    for (int bx = 0; bx < 2; bx++)
#pragma unroll
        for (int by = 0; by < 2; by++) {
            const float wxy = w[0][bx] * w[1][by];
            const int axy = (l[0][bx] * TY + l[1][by]) * TZ;
            const bool okxy = ok[0][bx] && ok[1][by];
#pragma unroll
            for (int bz = 0; bz < 2; bz++) {
                const float ww = wxy * w[2][bz];
                const bool o = okxy && ok[2][bz];
#pragma unroll
                for (int c = 0; c < C; c++)
                    red_shared_if(&tile_acc[c][axy + l[2][bz]], SIGNED ? __float2int_rn(ww * v[c]) : (int)__float2uint_rn(ww * v[c]), o);
            }
        }
}

template <int C, bool HAS_VAL>
__global__ void __launch_bounds__(256) scatter_kernel(const __grid_constant__ CUtensorMap tmap, CicGeom g,
                                                      const uint4 *__restrict__ rec, const int *__restrict__ offsets,
                                                      const float *__restrict__ val, float *__restrict__ mesh)
{
    __shared__ __align__(128) int tile_acc[C][TILE_PTS];
    __shared__ int run_start[NRUNS + 2];
    __shared__ int run_prefix[NRUNS + 2];
    __shared__ float red[32];

    int t[3], t0[3], ext[3];
    tile_coords(g, t, t0, ext);

    {
        int4 *z4 = reinterpret_cast<int4 *>(&tile_acc[0][0]);
        for (int i = threadIdx.x; i < C * TILE_PTS / 4; i += blockDim.x) z4[i] = make_int4(0, 0, 0, 0);
    }
    if (threadIdx.x < 32) {
        const int r = threadIdx.x;
        int b = 0, len = 0;
        if (r < NRUNS) {
            const int m = kRuns[r][0], c0 = kRuns[r][1], c1 = kRuns[r][2];
            bool valid = true;
            int n[3];
#pragma unroll
            for (int d = 0; d < 3; d++) {
                const int low = (m >> (2 - d)) & 1;
                if (low && g.nt[d] == 1) valid = false;  // the only tile along d is its own neighbour
                n[d] = t[d] - low;
                if (n[d] < 0) n[d] += g.nt[d];
            }
            if (valid) {
                const int key = ((n[0] * g.nt[1] + n[1]) * g.nt[2] + n[2]) * NCLS;
                b = offsets[key + c0];
                len = offsets[key + c1] - b;
            }
        }
        int inc = len;
#pragma unroll
        for (int o = 1; o < 16; o <<= 1) {
            int u = __shfl_up_sync(0xffffffffu, inc, o);
            if (r >= o) inc += u;
        }
        if (r < NRUNS) {
            run_start[r] = b - (inc - len);  // so that rec index = run_start[r] + flat index
            run_prefix[r + 1] = inc;
        }
        if (r == 0) run_prefix[0] = 0;
    }
    __syncthreads();
    const int own = run_prefix[1], total = run_prefix[NRUNS];

    // flat index -> record (+ values); the own tile is one contiguous run, the 13 neighbour runs are short
    auto fetch = [&](int i, uint4 &q, float v[C]) {
        int r = 0;
        if (i >= own) {
            r = 1;
            while (i >= run_prefix[r + 1]) r++;
        }
        q = rec[run_start[r] + i];
        if (HAS_VAL) {
#pragma unroll
            for (int c = 0; c < C; c++) v[c] = val[(size_t)q.w * C + c];
        }
    };

    // the first two rounds (all of a typical tile) are fetched up front and kept in registers
    const int i0 = threadIdx.x, i1 = threadIdx.x + blockDim.x;
    uint4 qa = make_uint4(0, 0, 0, 0), qb = qa;
    float va[C], vb[C];
#pragma unroll
    for (int c = 0; c < C; c++) va[c] = vb[c] = 0.f;
    if (i0 < total) fetch(i0, qa, va);
    if (i1 < total) fetch(i1, qb, vb);

    // bound on the absolute sum any mesh point can reach -> power-of-two fixed-point scale
    float bound;
    if (HAS_VAL) {
        float ma = 0.f, mb = 0.f;
#pragma unroll
        for (int c = 0; c < C; c++) { ma = fmaxf(ma, fabsf(va[c])); mb = fmaxf(mb, fabsf(vb[c])); }
        float part = ma + mb;
        for (int i = i1 + blockDim.x; i < total; i += blockDim.x) {
            uint4 q;
            float v[C];
            fetch(i, q, v);
            float m = 0.f;
#pragma unroll
            for (int c = 0; c < C; c++) m = fmaxf(m, fabsf(v[c]));
            part += m;
        }
        bound = block_sum(part, red) * 1.0001f;  // margin for the fp32 summation itself
    } else {
        bound = (float)total;
    }
    // fixed-point scale: the accumulators cannot overflow because |sum at any point| <= bound, and each of the
    // <= total deposits at a point rounds by <= 0.5.
    //   unit mass: deposits are >= 0 -> UNSIGNED accumulation with scale = (2^32 - headroom) / total.  total is an
    //              integer, so the scale (not a power of two: one extra fp32 rounding per deposit, 6e-8 relative,
    //              far below the quantum) is the same in every run: the density mesh stays bit-reproducible.
    //   values:    signed accumulation; bound is an fp32 sum whose last bits depend on the (arbitrary) order of
    //              the records, so only its exponent is used: scale = 2^(30 - ex) with bound <= 2^ex.
    float scale;
    if (HAS_VAL) {
        const int ex = (int)((__float_as_uint(fmaxf(bound, 1e-37f)) >> 23) & 255u) - 126;
        const int k = min(30 - ex, 96) - g.kshift;
        scale = __uint_as_float((unsigned)(127 + k) << 23);
    } else {
        const float room = fmaxf(4294967296.f * 0.99999f - (float)total, 1.f);
        scale = ldexpf(room / fmaxf(bound, 1.f), -g.kshift);
    }
    const float inv_scale = 1.f / scale;
    // mean subtraction (unit mass): mq quanta are removed exactly in integer, the sub-quantum rest in fp32
    long long mq = 0;
    float mrest = 0.f;
    if (!HAS_VAL && g.mean != 0.0) {
        const double m = g.mean * (double)scale;
        mq = __double2ll_rn(m);
        mrest = (float)((m - (double)mq) * (double)inv_scale);
    }
    const float fr = 1.f / (float)(1u << g.fbits);
    const unsigned fmask = (1u << g.fbits) - 1u;

    auto put = [&](uint4 q, const float vin[C]) {
        float v[C];
#pragma unroll
        for (int c = 0; c < C; c++) v[c] = HAS_VAL ? vin[c] * scale : scale;
        deposit<C, HAS_VAL>(g, t0, ext, q, v, tile_acc, fr, fmask);
    };
    if (i0 < total) put(qa, va);
    if (i1 < total) put(qb, vb);
    for (int i = i1 + blockDim.x; i < total; i += blockDim.x) {
        uint4 q;
        float v[C];
        fetch(i, q, v);
        put(q, v);
    }
    __syncthreads();

    if (g.use_tma) {
        // int -> float in place (same bytes), then one tensor store per component; TMA clips at the mesh edge
        int4 *a4 = reinterpret_cast<int4 *>(&tile_acc[0][0]);
        for (int i = threadIdx.x; i < C * TILE_PTS / 4; i += blockDim.x) {
            int4 a = a4[i];
            float4 f = HAS_VAL ? make_float4((float)a.x * inv_scale, (float)a.y * inv_scale, (float)a.z * inv_scale, (float)a.w * inv_scale)
                               : make_float4((float)((long long)(unsigned)a.x - mq) * inv_scale - mrest, (float)((long long)(unsigned)a.y - mq) * inv_scale - mrest,
                                             (float)((long long)(unsigned)a.z - mq) * inv_scale - mrest, (float)((long long)(unsigned)a.w - mq) * inv_scale - mrest);
            reinterpret_cast<float4 *>(a4)[i] = f;
        }
        fence_proxy_async_smem();
        __syncthreads();
        if (threadIdx.x == 0) {
#pragma unroll
            for (int c = 0; c < C; c++) tma_store_4d(&tmap, &tile_acc[c][0], t0[2], t0[1], t0[0], g.c0 + c);
            tma_store_commit_and_wait();
        }
    } else {
        // plain path: one warp per z-row
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
        for (int row = w; row < TX * TY; row += nw) {
            const int lx = row / TY, ly = row % TY;
            if (lx < ext[0] && ly < ext[1] && lane < ext[2]) {
                const size_t o = ((size_t)(t0[0] + lx) * g.N[1] + (t0[1] + ly)) * g.zs + (t0[2] + lane);
#pragma unroll
                for (int c = 0; c < C; c++) {
                    const int a = tile_acc[c][row * TZ + lane];
                    mesh[(size_t)c * g.ms + o] = HAS_VAL ? (float)a * inv_scale : (float)((long long)(unsigned)a - mq) * inv_scale - mrest;
                }
            }
        }
    }
}

// --------------------------------------------------------------------------------------------------
// gathers
// --------------------------------------------------------------------------------------------------
enum GatherMode { G_VALUE = 0, G_GRAD = 1, G_FUSED = 2 };

// KICK: the interpolated acc (and alpha) of a particle is applied on the spot -- p += rn(acc Ka) [+= rn(acc Kb)],
// x += rn(p D), and for the adjoint xi -= alpha K, pi -= xi D (eq. 16 L172 / eq. 49, same arithmetic and
// order as kick_drift_kernel) -- and the particle's new sort key is added to the histogram of the next sort, so
// a step needs no separate kick/drift and histogram passes and acc/alpha never travel through HBM.
template <int C, int MODE, bool HAS_COT, bool KICK>
__global__ void __launch_bounds__(256) gather_kernel(const __grid_constant__ CUtensorMap tmap, CicGeom g,
                                                     const uint4 *__restrict__ rec, const int *__restrict__ offsets,
                                                     const float *__restrict__ mesh, const float *cot,
                                                     float cot_scale, float *__restrict__ out, float *__restrict__ out2,
                                                     PosGeom pg, KickArgs ka)
{
    __shared__ __align__(128) float halo[C * HALO_STRIDE];
    __shared__ __align__(8) unsigned long long bar;
    int t[3], t0[3], ext[3];
    tile_coords(g, t, t0, ext);
    const int key0 = ((t[0] * g.nt[1] + t[1]) * g.nt[2] + t[2]) * NCLS;
    const int beg = offsets[key0], end = offsets[key0 + NCLS];
    if (beg == end) return;

    // the halo reaches one point past the tile: interior tiles never wrap and can take the TMA box as is
    const bool interior = g.use_tma && t0[0] + ext[0] < g.N[0] && t0[1] + ext[1] < g.N[1] && t0[2] + ext[2] < g.N[2];
    uint4 q = make_uint4(0, 0, 0, 0);
    if (interior) {
        if (threadIdx.x == 0) mbar_init(&bar, 1);
        __syncthreads();
        if (threadIdx.x == 0) {
            mbar_expect_tx(&bar, (unsigned)(C * HALO_PTS * sizeof(float)));
#pragma unroll
            for (int c = 0; c < C; c++) tma_load_4d(&halo[c * HALO_STRIDE], &tmap, &bar, t0[2], t0[1], t0[0], g.c0 + c);
        }
        if (beg + (int)threadIdx.x < end) q = rec[beg + threadIdx.x];  // overlaps the TMA flight
        mbar_wait(&bar, 0);
    } else {
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
        for (int row = w; row < C * HX * HY; row += nw) {
            const int c = row / (HX * HY), r2 = row % (HX * HY);
            const int lx = r2 / HY, ly = r2 % HY;
            if (lx <= ext[0] && ly <= ext[1]) {
                int gx = t0[0] + lx, gy = t0[1] + ly;
                if (gx >= g.N[0]) gx -= g.N[0];
                if (gy >= g.N[1]) gy -= g.N[1];
                const float *src = mesh + (size_t)c * g.ms + ((size_t)gx * g.N[1] + gy) * g.zs;
                float *dst = &halo[c * HALO_STRIDE + (lx * HY + ly) * HZP];
                if (lane <= ext[2]) {
                    int gz = t0[2] + lane;
                    if (gz >= g.N[2]) gz -= g.N[2];
                    dst[lane] = src[gz];
                }
                if (lane == 0 && ext[2] == TZ) {
                    int gz = t0[2] + TZ;
                    if (gz >= g.N[2]) gz -= g.N[2];
                    dst[TZ] = src[gz];
                }
            }
        }
        if (beg + (int)threadIdx.x < end) q = rec[beg + threadIdx.x];
        __syncthreads();
    }

    const float fr = 1.f / (float)(1u << g.fbits);
    const unsigned fmask = (1u << g.fbits) - 1u;
    for (int i = beg + threadIdx.x; i < end; i += blockDim.x) {
        if (i != beg + (int)threadIdx.x) q = rec[i];
        // KICK: the particle's state is fetched first (independent loads, in flight while the weights are formed)
        long long st_p[3], st_x[3];
        float st_xi[3];
        if (KICK) {
#pragma unroll
            for (int d = 0; d < 3; d++) {
                st_p[d] = ka.p[3 * (size_t)q.w + d];
                if (ka.Ds != 0.0) st_x[d] = ka.x[3 * (size_t)q.w + d];
                if (MODE == G_FUSED) st_xi[d] = ka.xi[3 * (size_t)q.w + d];
            }
        }
        const unsigned X[3] = {q.x, q.y, q.z};
        int l[3];
        float w[3][2];
#pragma unroll
        for (int d = 0; d < 3; d++) {
            l[d] = (int)(X[d] >> g.fbits) - t0[d];
            float td = (float)(X[d] & fmask) * fr;
            w[d][0] = 1.f - td;
            w[d][1] = td;
        }
        const int base = (l[0] * HY + l[1]) * HZP + l[2];
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
                    const int idx = base + (bx * HY + by) * HZP + bz;
                    const float W = w[0][bx] * w[1][by] * w[2][bz];
                    const float dWx = (bx ? 1.f : -1.f) * w[1][by] * w[2][bz];
                    const float dWy = (by ? 1.f : -1.f) * w[0][bx] * w[2][bz];
                    const float dWz = (bz ? 1.f : -1.f) * w[0][bx] * w[1][by];
                    float m = 0.f;  // cotangent-weighted mesh value at this corner
#pragma unroll
                    for (int c = 0; c < C; c++) {
                        const float f = halo[c * HALO_STRIDE + idx];
                        if (MODE != G_GRAD) val[c] += W * f;
                        if (MODE != G_VALUE) m += cv[c] * f;
                    }
                    if (MODE != G_VALUE) {
                        gr[0] += dWx * m;
                        gr[1] += dWy * m;
                        gr[2] += dWz * m;
                    }
                }
        if (KICK) {
            const float *a3 = MODE == G_FUSED ? &val[1] : &val[0];
            unsigned int Xn[3];
#pragma unroll
            for (int d = 0; d < 3; d++) {
                const size_t i = 3 * j + d;
                long long pv = st_p[d];
                if (ka.Ka != 0.0) pv += __double2ll_rn((double)a3[d] * ka.Ka);
                if (ka.Kb != 0.0) pv += __double2ll_rn((double)a3[d] * ka.Kb);
                ka.p[i] = pv;
                if (MODE == G_FUSED) {
                    float v = st_xi[d];
                    if (ka.Ka != 0.0) v = fmaf(-gr[d], ka.Kaf, v);
                    if (ka.Kb != 0.0) v = fmaf(-gr[d], ka.Kbf, v);
                    ka.xi[i] = v;
                    if (ka.Ds != 0.0) ka.pi[i] = fmaf(-v, ka.Df, cv[1 + d]);
                }
                if (ka.Ds != 0.0) {
                    const long long xv = st_x[d] + __double2ll_rn((double)pv * ka.Ds);
                    ka.x[i] = xv;
                    Xn[d] = record_coord(pg, xv, d);
                }
            }
            if (ka.Ds != 0.0) hist_add(ka.hist, key_of(pg, Xn));
            if (ka.store) {
#pragma unroll
                for (int e = 0; e < 3; e++) {
                    out[j * 3 + e] = a3[e];
                    if (MODE == G_FUSED) out2[j * 3 + e] = gr[e];
                }
            }
        } else if (MODE == G_VALUE) {
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

static dim3 tile_grid(const Geometry &g) { return dim3((unsigned)g.nt[2], (unsigned)g.nt[1], (unsigned)g.nt[0]); }
static int env_threads(const char *name, int dflt)
{
    const char *e = getenv(name);
    int v = e ? atoi(e) : dflt;
    return (v >= 32 && v <= 256 && v % 32 == 0) ? v : dflt;
}

int scatter_sorted(pm_ctx *c, const float *val, int C, float *mesh, int zs, long long ms, double mean)
{
    CUtensorMap map;
    CicGeom g = make_cic_geom(c, mesh, C, zs, ms, true, &map);
    g.mean = (C == 1 && !val) ? mean : 0.0;
    double np = (double)c->cur_np, ng = (double)c->g.ng;
    dim3 grid = tile_grid(c->g);
    if (C == 1 && !val) {
        Timer t(c, TC_SCATTER1, 12.0 * np + 4.0 * ng);
        scatter_kernel<1, false><<<grid, env_threads("PM_SCATTER_THREADS", 128), 0, c->stream>>>(map, g, c->rec, c->offsets, nullptr, mesh);
        PM_LAUNCH_CHECK(c, "scatter_kernel<1>");
        t.stop();
    } else if (C == 1) {
        Timer t(c, TC_SCATTER1, 16.0 * np + 4.0 * ng);
        scatter_kernel<1, true><<<grid, env_threads("PM_SCATTER_THREADS", 128), 0, c->stream>>>(map, g, c->rec, c->offsets, val, mesh);
        PM_LAUNCH_CHECK(c, "scatter_kernel<1,val>");
        t.stop();
    } else if (C == 3 && val) {
        Timer t(c, TC_SCATTER3, 24.0 * np + 12.0 * ng);
        scatter_kernel<3, true><<<grid, env_threads("PM_SCATTER_THREADS", 256), 0, c->stream>>>(map, g, c->rec, c->offsets, val, mesh);
        PM_LAUNCH_CHECK(c, "scatter_kernel<3,val>");
        t.stop();
    } else {
        return fail(c, PM_EINVAL, "scatter", "C must be 1, or 3 with values");
    }
    return PM_OK;
}

static double kick_bytes(const KickArgs *ka, bool adj)
{
    // per particle: p read + write, x read + write on a drift, xi read + write and pi write for the adjoint, stores
    double b = 48.0 + (ka->Ds != 0.0 ? 48.0 : 0.0) + (ka->store ? (adj ? 24.0 : 12.0) : 0.0);
    if (adj) b += 24.0 + (ka->Ds != 0.0 ? 12.0 : 0.0);
    return b;
}

int gather_sorted(pm_ctx *c, const float *mesh, int C, int zs, long long ms, float *out, const KickArgs *ka)
{
    CUtensorMap map;
    CicGeom g = make_cic_geom(c, mesh, C, zs, ms, false, &map);
    double np = (double)c->cur_np, ng = (double)c->g.ng;
    dim3 grid = tile_grid(c->g);
    PosGeom pg = make_pos_geom(c->g);
    KickArgs none;
    memset(&none, 0, sizeof none);
    if (ka && C != 3) return fail(c, PM_EINVAL, "gather", "internal: kick needs C = 3");
    if (C == 1) {
        Timer t(c, TC_GATHER3, 16.0 * np + 4.0 * ng);
        gather_kernel<1, G_VALUE, false, false><<<grid, env_threads("PM_GATHER_THREADS", 256), 0, c->stream>>>(map, g, c->rec, c->offsets, mesh, nullptr, 1.f, out, nullptr, pg, none);
        PM_LAUNCH_CHECK(c, "gather_kernel<1>");
        t.stop();
    } else if (C == 3 && !ka) {
        Timer t(c, TC_GATHER3, 24.0 * np + 12.0 * ng);
        gather_kernel<3, G_VALUE, false, false><<<grid, env_threads("PM_GATHER_THREADS", 256), 0, c->stream>>>(map, g, c->rec, c->offsets, mesh, nullptr, 1.f, out, nullptr, pg, none);
        PM_LAUNCH_CHECK(c, "gather_kernel<3>");
        t.stop();
    } else if (C == 3) {
        Timer t(c, TC_GATHER_KICK, (12.0 + kick_bytes(ka, false)) * np + 12.0 * ng);
        gather_kernel<3, G_VALUE, false, true><<<grid, env_threads("PM_GATHER_THREADS", 256), 0, c->stream>>>(map, g, c->rec, c->offsets, mesh, nullptr, 1.f, out, nullptr, pg, *ka);
        PM_LAUNCH_CHECK(c, "gather_kernel<3,kick>");
        t.stop();
    } else {
        return fail(c, PM_EINVAL, "gather", "C must be 1 or 3");
    }
    return PM_OK;
}

int gather_grad_sorted(pm_ctx *c, const float *mesh, int C, int zs, long long ms, const float *cot, float cot_scale,
                       float *out)
{
    CUtensorMap map;
    CicGeom g = make_cic_geom(c, mesh, C, zs, ms, false, &map);
    double np = (double)c->cur_np, ng = (double)c->g.ng;
    dim3 grid = tile_grid(c->g);
    PosGeom pg = make_pos_geom(c->g);
    KickArgs none;
    memset(&none, 0, sizeof none);
    const int th = env_threads("PM_GATHER_THREADS", 256);
    Timer t(c, TC_GATHER_GRAD, (24.0 + (cot ? 4.0 * C : 0.0)) * np + 4.0 * C * ng);
    if (C == 1 && !cot)
        gather_kernel<1, G_GRAD, false, false><<<grid, th, 0, c->stream>>>(map, g, c->rec, c->offsets, mesh, nullptr, cot_scale, out, nullptr, pg, none);
    else if (C == 1)
        gather_kernel<1, G_GRAD, true, false><<<grid, th, 0, c->stream>>>(map, g, c->rec, c->offsets, mesh, cot, cot_scale, out, nullptr, pg, none);
    else if (C == 3 && !cot)
        gather_kernel<3, G_GRAD, false, false><<<grid, th, 0, c->stream>>>(map, g, c->rec, c->offsets, mesh, nullptr, cot_scale, out, nullptr, pg, none);
    else if (C == 3)
        gather_kernel<3, G_GRAD, true, false><<<grid, th, 0, c->stream>>>(map, g, c->rec, c->offsets, mesh, cot, cot_scale, out, nullptr, pg, none);
    else
        return fail(c, PM_EINVAL, "gather_grad", "C must be 1 or 3");
    PM_LAUNCH_CHECK(c, "gather_kernel<grad>");
    t.stop();
    return PM_OK;
}

int gather_fused_sorted(pm_ctx *c, const float *mesh4, int zs, long long ms, const float *pi, float *acc, float *alpha,
                        const KickArgs *ka)
{
    CUtensorMap map;
    CicGeom g = make_cic_geom(c, mesh4, 4, zs, ms, false, &map);
    double np = (double)c->cur_np, ng = (double)c->g.ng;
    PosGeom pg = make_pos_geom(c->g);
    const int th = env_threads("PM_GATHER_THREADS", 256);
    if (!ka) {
        KickArgs none;
        memset(&none, 0, sizeof none);
        Timer t(c, TC_GATHER_FUSED, 48.0 * np + 16.0 * ng);
        gather_kernel<4, G_FUSED, true, false><<<tile_grid(c->g), th, 0, c->stream>>>(map, g, c->rec, c->offsets, mesh4, pi, 1.f, acc, alpha, pg, none);
        PM_LAUNCH_CHECK(c, "gather_kernel<fused>");
        t.stop();
    } else {
        Timer t(c, TC_GATHER_FUSED, (24.0 + kick_bytes(ka, true)) * np + 16.0 * ng);
        gather_kernel<4, G_FUSED, true, true><<<tile_grid(c->g), th, 0, c->stream>>>(map, g, c->rec, c->offsets, mesh4, pi, 1.f, acc, alpha, pg, *ka);
        PM_LAUNCH_CHECK(c, "gather_kernel<fused,kick>");
        t.stop();
    }
    return PM_OK;
}

}  // namespace pm
