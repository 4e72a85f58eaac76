// pm_cic.cu -- cloud-in-cell scatter / gather / weight-gradient gather, tile by tile out of shared memory.
//
// PAPER.md eq. 10 (L121-125): W(x, x') = prod_d max(1 - |x_d - x'_d| / l, 0), l = 1 cell; the gather
// "interpolates ... from the same grid points with the same weights" (L133); their VJPs (L410) are a
// scatter of cotangents (value argument) and a weight-gradient gather (position argument).
// Cell i_d = floor(x_d), t_d = x_d - i_d in [0,1): weight (1 - t_d) at i_d, t_d at i_d + 1 (periodic),
// derivative -1 / +1 (floor convention, right derivative; R7).
//
// Input: the records sorted by (tile, class) of pm_bin.cu; a tile is TX x TY x TZ cells.
//
// Both kernels are PERSISTENT: a few CTAs per SM draw tiles from a global counter (dense tiles do not stall a
// static schedule).  The scatter is WARP-SPECIALISED: one producer warp looks up the record runs of the next
// tiles and stages their records in a ring of NST shared-memory stages guarded by full / empty mbarriers (1-D
// bulk copies + 16-byte cp.async), NCW consumer warps accumulate.  The gather is a two-stage cp.async pipeline in
// which all 256 threads first start the 16-byte copies of the NEXT tile's halo rows and then interpolate for the
// particles of the current one (TMA tensor loads of these narrow 144-byte rows were measured slower and removed;
// TMA is kept for the scatter's tile stores).
//
// scatter -- OUTPUT-STATIONARY: the CTA owns the mesh points of the tile, takes the particles of the
//   tile itself plus the last-cell-layer classes of its (up to 7) low-side neighbour tiles, accumulates in
//   shared memory with NATIVE int32 atomics (fp32 and 64-bit shared atomics are CAS loops on sm_100a)
//   in fixed point with a per-tile scale that cannot overflow, converts in place and writes the tile
//   with ONE asynchronous TMA tensor store per mesh (clipped at the mesh edge) from a double-buffered
//   accumulator: no zero-fill pass, no global atomics, every mesh point written exactly once, and a
//   result that does not depend on the order in which particles arrive (bit-reproducible).
// gather -- the halo box (TX+1)(TY+1)(TZ+4) of each mesh sits in shared memory; the consumers
//   interpolate values / weight gradients / both for the particles of the tile and, in the KICK variants,
//   apply the kick(s) and the drift to the particle's fixed-point state on the spot (pm_pos.cuh).
#include <cstdlib>
#include <cstring>

#include "pm_pos.cuh"

#ifdef PM_DEBUG
#define PM_DBG(x) (x)
#else
#define PM_DBG(x) 0
#endif

namespace pm {

struct CicGeom {
    int N[3], nt[3];
    int fbits;
    int zs;        // floats per z-row
    long long ms;  // floats per mesh (component stride)
    int use_tma;   // scatter: tensor map valid for this mesh; gather: base and strides are 16-byte aligned (async row copies)
    int c0;        // first component (4th tensor-map coordinate)
    int dbg;       // probe build (-DPM_DEBUG) only: 1 = gather skips the particle loop, 2 = skips the halo copies, 8 = clock stamps
    int kshift;    // probe build only: coarsen the scatter's fixed-point scale by this many bits; both are 0 and unread in libpm.so
    int ntiles;
    double mean;   // unit-mass scatter only: constant subtracted from every mesh point IN INTEGER, before the
                   // int -> fp32 conversion (0 = plain density; nbar on the force path, whose k = 0 mode is zeroed
                   // anyway, so that fp32 rounding is relative to the fluctuation rho - nbar, not to rho)
    long long *dbgbuf;  // debug timeline (PM_DEBUG_CIC & 8): clock64 stamps of CTA 0
    int *spool_ctl;     // scatter pool: [0] next free accumulator, [16 + p] chunks of accumulator p that have arrived
    unsigned *spool;    // scatter pool: spool_n accumulators of TILE_PTS uint32, all zero between uses
    int *wq;       // work queue of this stream (wq_reserve / wq_pop below); items tagged with wq_epoch
    int wq_cap;    // items the queue holds
    int spool_n;   // accumulators in the scatter pool
    unsigned wq_epoch;
    int sh1, sh2;  // log2 of nt[1], nt[2] when they are powers of two (tile index -> coordinates without a division), else -1
    int *sched;    // [0] tile counter, [1] finished CTAs; both zero between launches (the last CTA resets them)
};

constexpr int TILE_PTS = TX * TY * TZ;
constexpr int HX = TX + 1, HY = TY + 1;
constexpr int HZP = TZ + 4;                               // halo row pitch: 144 bytes, a TMA-legal box width
constexpr int HALO_PTS = HX * HY * HZP;
constexpr int HALO_STRIDE = (HALO_PTS + 31) / 32 * 32;    // per-mesh stride in shared memory: 128-byte multiple
constexpr int NCW = 8;                                    // consumer warps
constexpr int NCT = NCW * 32;                             // consumer threads
constexpr int NTHREADS = NCT + 32;                        // + one producer warp
constexpr int SCHUNK = 2048;                               // scatter: records per chunk of a heavy tile
constexpr int SFAST = 1024;                               // valued scatter: tiles up to this many records take their bound from an integer sum
constexpr int RCAP = 512;                                 // records staged in shared memory per tile (the rest are read from global)

// ---- PTX wrappers: mbarrier + TMA (sm_90+/sm_100a) ----------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// expect-tx WITHOUT arriving (the thread arrives separately)
__device__ __forceinline__ void mbar_expect_tx_only(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// 16-byte asynchronous copy through the LSU path (no per-operation TMA cost: used for short / ragged pieces)
__device__ __forceinline__ void cp_async16(void *dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"((unsigned long long)src) : "memory");
}
// arrive on the barrier once all cp.async issued so far by this thread have landed (counts as this thread's arrival)
__device__ __forceinline__ void cp_async_arrive(unsigned long long *bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned phase)
{
    // try_wait with a suspend-time hint: a waiting warp sleeps in hardware instead of spinning through the issue slots
    asm volatile(
        "{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}"
        ::"r"(smem_u32(bar)), "r"(phase), "r"(20000u)
        : "memory");
}
// non-blocking: has the phase with this parity completed?
__device__ __forceinline__ bool mbar_test(unsigned long long *bar, unsigned phase)
{
    unsigned ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok)
                 : "r"(smem_u32(bar)), "r"(phase)
                 : "memory");
    return ok != 0;
}
__device__ __forceinline__ void bulk_load(void *dst, const void *src, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"((unsigned long long)src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void tma_store_4d(const CUtensorMap *m, const void *src, int z, int y, int x, int c)
{
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5}], [%1];"
                 ::"l"((unsigned long long)m), "r"(smem_u32(src)), "r"(z), "r"(y), "r"(x), "r"(c)
                 : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// barrier among the consumer warps only (the producer warp never joins it)
__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(NCT) : "memory"); }

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
    c->tma_ok = encode_mesh_map(&c->tmap_store, c->mesh[0], g.N, 7, g.zs, g.mesh_stride, TZ, TY, TX);
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
    r.kshift = 0;
    r.dbg = 0;
#ifdef PM_DEBUG
    // probe build only (python -m paper_2211_09815_b200.build --debug -> libpm_debug.so): knobs that change or skip work
    static const int env_kshift = [] { const char *e = getenv("PM_DEBUG_KSHIFT"); return e ? atoi(e) : 0; }();
    static const int env_dbg = [] { const char *e = getenv("PM_DEBUG_CIC"); return e ? atoi(e) : 0; }();
    r.kshift = env_kshift;
    r.dbg = env_dbg;
#endif
    r.mean = 0.0;
    r.ntiles = g.ntiles;
    r.sched = c->sched;
    r.wq = c->wq;
    r.wq_cap = (int)((c->wq_ints - 16) / 8);  // WQ_ITEM ints per item
    r.spool_n = c->spool_n;
    r.spool_ctl = c->spool_ctl;
    r.spool = c->spool;
    r.wq_epoch = ++c->wq_epoch ? c->wq_epoch : ++c->wq_epoch;  // never 0 (the cleared buffer's tag)
    r.sh1 = r.sh2 = -1;
    for (int k = 0; k < 31; k++) {
        if (g.nt[1] == (1 << k)) r.sh1 = k;
        if (g.nt[2] == (1 << k)) r.sh2 = k;
    }
    r.dbgbuf = reinterpret_cast<long long *>(c->scal);
    memset(map, 0, sizeof(*map));
    long long off = mesh - c->mesh[0];
    bool internal = zs == g.zs && ms == g.mesh_stride && mesh >= c->mesh[0] && off % g.mesh_stride == 0 &&
                    off / g.mesh_stride + C <= 7;
    if (!store) {
        // gathers copy halo rows in 16-byte pieces: all they need is a 16-byte aligned base and strides (no tensor map)
        r.use_tma = (((uintptr_t)mesh & 15) == 0 && (zs & 3) == 0 && (ms & 3) == 0) ? 1 : 0;
    } else if (internal && c->tma_ok) {
        *map = c->tmap_store;
        r.use_tma = 1;
        r.c0 = (int)(off / g.mesh_stride);
    } else if (!internal) {
        if (encode_mesh_map(map, mesh, g.N, C, zs, ms, TZ, TY, TX)) r.use_tma = 1;
    }
    return r;
}

// ---- tiles and scheduling -----------------------------------------------------------------------------
__device__ __forceinline__ void tile_coords(const CicGeom &g, int tile, int t[3], int t0[3], int ext[3])
{
    if (g.sh1 >= 0 && g.sh2 >= 0) {
        t[2] = tile & (g.nt[2] - 1);
        const int r = tile >> g.sh2;
        t[1] = r & (g.nt[1] - 1);
        t[0] = r >> g.sh1;
    } else {
        t[2] = tile % g.nt[2];
        const int r = tile / g.nt[2];
        t[1] = r % g.nt[1];
        t[0] = r / g.nt[1];
    }
    t0[0] = t[0] * TX; t0[1] = t[1] * TY; t0[2] = t[2] * TZ;
    ext[0] = min(TX, g.N[0] - t0[0]);
    ext[1] = min(TY, g.N[1] - t0[1]);
    ext[2] = min(TZ, g.N[2] - t0[2]);
}

// Tiles are drawn from the global counter TBATCH at a time (neighbouring tiles share halo lines in L2, and the
// atomic's round trip is paid once per batch); the next batch is requested one batch ahead.
constexpr int TBATCH = 1;
struct TileDraw {
    int base, next_base, pos;
    __device__ __forceinline__ void init(int *sched)
    {
        base = atomicAdd(&sched[0], TBATCH);
        next_base = atomicAdd(&sched[0], TBATCH);
        pos = 0;
    }
    // next tile index (may be >= ntiles: the caller stops there); uniform across the warp (lane 0 draws)
    __device__ __forceinline__ int next(int *sched)
    {
        if (pos == TBATCH) {
            base = next_base;
            next_base = atomicAdd(&sched[0], TBATCH);
            pos = 0;
        }
        return base + pos++;
    }
};

// called by one thread per CTA when it has drawn its last tile: the last CTA to finish re-arms the counters
__device__ __forceinline__ void sched_finish(int *sched, int *wq = nullptr, int *spool_ctl = nullptr)
{
    __threadfence();
    if (atomicAdd(&sched[1], 1) == (int)gridDim.x - 1) {
        sched[0] = 0;
        sched[1] = 0;
        if (wq) {
            wq[0] = 0;
            wq[1] = 0;
            wq[2] = 0;
        }
        if (spool_ctl) spool_ctl[0] = 0;
        __threadfence();
    }
}

// ---- global work queue for the chunks of heavy tiles (one queue per stream) ----------
// wq[0] = head, wq[1] = tail, wq[2] = tiles published so far; items of WQ_ITEM ints from wq + 16:
// {tile, lo, hi, pool, -, -, -, tag}.  ONE layout for the scatter and the gather kernels, so the tag word of an item only
// ever holds tags (the epoch of the launch that wrote it), never a payload that could be mistaken for one.
// Pusher (the thread that drew a heavy tile): reserve k items with one fetch-and-add on the tail, write the payloads,
// fence, write the tags.  The tail is NEVER taken back: when the reservation does not fit, the part below the capacity
// is published as no-op items (tile = -2) and the tile stays whole, so every reserved index below the capacity is
// eventually tagged.  Popper (a CTA whose tile counter is exhausted): fetch-and-add on the head; an index below the tail
// waits for its tag (its pusher is a resident CTA between two consecutive stores); an index at or beyond the tail waits
// until an item is pushed there or every tile has been published (wq[2] == ntiles: no push can follow), then the CTA is
// finished for good.  Every wait is on a CTA that has already drawn a tile, i.e. that is resident and itself waits on
// nobody, which is the forward-progress argument; a watchdog bounds the spins anyway and raises sched[8].
constexpr int WQ_ITEM = 8;
constexpr long long WQ_SPIN_CYCLES = 1ll << 33;  // ~4 s at 2 GHz: only a broken invariant gets here

__device__ __forceinline__ int wq_vload(const int *p) { return *reinterpret_cast<const volatile int *>(p); }
__device__ __forceinline__ void wq_watchdog_fire(const CicGeom &g) { atomicExch(&g.sched[8], 1); }

__device__ __forceinline__ void wq_write(const CicGeom &g, int idx, int tile, int lo, int hi, int pool)
{
    int *it = g.wq + 16 + WQ_ITEM * idx;
    it[0] = tile;
    it[1] = lo;
    it[2] = hi;
    it[3] = pool;
}
__device__ __forceinline__ void wq_tag(const CicGeom &g, int idx)
{
    *reinterpret_cast<volatile unsigned *>(g.wq + 16 + WQ_ITEM * idx + 7) = g.wq_epoch;
}
// one thread: reserves k items; returns their base, or -1 when they do not fit (no-op items published instead)
__device__ __forceinline__ int wq_reserve(const CicGeom &g, int k)
{
    const int base = atomicAdd(&g.wq[1], k);
    if (base + k <= g.wq_cap) return base;
    const int end = min(base + k, g.wq_cap);
    for (int i = base; i < end; i++) wq_write(g, i, -2, 0, 0, -1);
    __threadfence();
    for (int i = base; i < end; i++) wq_tag(g, i);
    __threadfence();
    return -1;
}
// one thread: next item of the queue; false = no more work for this CTA (it must then stay finished)
__device__ __forceinline__ bool wq_pop(const CicGeom &g, int &tile, int &lo, int &hi, int &pool)
{
    for (;;) {
        const int idx = atomicAdd(&g.wq[0], 1);
        const long long t_start = clock64();
        for (;;) {
            int t = wq_vload(&g.wq[1]);
            if (idx < t) break;
            if (wq_vload(&g.wq[2]) == g.ntiles) {
                __threadfence();
                t = wq_vload(&g.wq[1]);
                if (idx >= t) return false;
                break;
            }
            if (clock64() - t_start > WQ_SPIN_CYCLES) { wq_watchdog_fire(g); return false; }
        }
        if (idx >= g.wq_cap) return false;  // reservations beyond the capacity hold no items (their tiles stayed whole)
        const int *it = g.wq + 16 + WQ_ITEM * idx;
        while ((unsigned)wq_vload(it + 7) != g.wq_epoch) {
            if (clock64() - t_start > WQ_SPIN_CYCLES) { wq_watchdog_fire(g); return false; }
        }
        __threadfence();
        tile = wq_vload(it);
        lo = wq_vload(it + 1);
        hi = wq_vload(it + 2);
        pool = wq_vload(it + 3);
        if (tile >= 0) return true;
        // a no-op item: take the next one
    }
}

// CIC corners of one particle relative to a tile: local indices, ownership flags, weights.
// FAST: the particle is of the tile's own class 0 (no coordinate in the last cell layer): all 8 corners are inside.
template <bool FAST>
struct Corners {
    int l[3][2];
    bool ok[3][2];
    float w[3][2];
    __device__ __forceinline__ Corners(const CicGeom &g, const int t0[3], const int ext[3], uint4 q, float fr, unsigned fmask)
    {
        const unsigned X[3] = {q.x, q.y, q.z};
#pragma unroll
        for (int d = 0; d < 3; d++) {
            int l0 = (int)(X[d] >> g.fbits) - t0[d];
            int l1 = l0 + 1;
            if (!FAST) {
                if (l0 < 0) l0 += g.N[d];          // particle of the low neighbour across the periodic edge
                l1 = l0 + 1;
                if (l1 == g.N[d]) l1 = 0;          // the only tile along d is its own neighbour
            }
            l[d][0] = l0;
            l[d][1] = l1;
            ok[d][0] = FAST || l0 < ext[d];
            ok[d][1] = FAST || l1 < ext[d];
            const float td = (float)(X[d] & fmask) * fr;
            w[d][0] = 1.f - td;
            w[d][1] = td;
        }
    }
    // f(offset within the tile, weight, owned)
    template <class F>
    __device__ __forceinline__ void each(F f) const
    {
#pragma unroll
        for (int bx = 0; bx < 2; bx++)
#pragma unroll
            for (int by = 0; by < 2; by++) {
                const float wxy = w[0][bx] * w[1][by];
                const int axy = (l[0][bx] * TY + l[1][by]) * TZ;
                const bool okxy = ok[0][bx] && ok[1][by];
#pragma unroll
                for (int bz = 0; bz < 2; bz++) f(axy + l[2][bz], wxy * w[2][bz], okxy && ok[2][bz]);
            }
    }
};

// shared-memory integer reduction, predicated (no branch around the atomic) or not
__device__ __forceinline__ void red_shared(int *addr, int v, bool ok, bool always)
{
    if (always)
        asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(smem_u32(addr)), "r"(v) : "memory");
    else
        asm volatile("{\n .reg .pred p;\n setp.ne.s32 p, %2, 0;\n @p red.shared.add.s32 [%0], %1;\n}"
                     ::"r"(smem_u32(addr)), "r"(v), "r"((int)ok)
                     : "memory");
}

__device__ __forceinline__ float consumer_max(float v, float *sh /*NCW*/)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    consumer_sync();
    float r = sh[0];
#pragma unroll
    for (int k = 1; k < NCW; k++) r = fmaxf(r, sh[k]);
    consumer_sync();
    return r;
}

// power-of-two exponent e with v <= 2^e (v > 0, normal)
__device__ __forceinline__ int exp_above(float v) { return (int)((__float_as_uint(v) >> 23) & 255u) - 126; }

// --------------------------------------------------------------------------------------------------
// scatter
// --------------------------------------------------------------------------------------------------
// the 14 contiguous class runs a tile pulls from itself (m = 0) and its low neighbours
// m: bit 2/1/0 = neighbour is one tile lower in x/y/z; classes [c0, c1)
__constant__ signed char kRuns[14][3] = {{0, 0, 8}, {4, 4, 8}, {2, 2, 4}, {2, 6, 8}, {1, 1, 2}, {1, 3, 4}, {1, 5, 6},
                                         {1, 7, 8}, {6, 6, 8}, {5, 5, 6}, {5, 7, 8}, {3, 3, 4}, {3, 7, 8}, {7, 7, 8}};
constexpr int NRUNS = 14;

struct ScatterSlot {
    int tile;                   // -1: no more tiles
    int total;                  // records in all runs
    int n0;                     // leading records of the tile's own class 0 (all corners inside)
    int run_start[NRUNS];       // rec index = run_start[r] + flat index
    int run_prefix[NRUNS + 1];
    int lo, hi;                 // flat record range of this work item: [0, total) or one chunk of a heavy tile
    int pool;                   // heavy tile: slot of the global integer accumulator the chunks are combined in; else -1
};

// record stages: 3 for the scalar scatter (40 KB per CTA: five CTAs per SM at 40 registers), 2 for three components
// (64 KB: three CTAs per SM)
template <int C>
constexpr int scatter_stages() { return C == 1 ? 3 : 2; }
template <int C>
constexpr size_t scatter_smem_bytes() { return (size_t)2 * C * TILE_PTS * sizeof(int) + (size_t)scatter_stages<C>() * RCAP * sizeof(uint4); }

template <int C, bool HAS_VAL>
__global__ void __launch_bounds__(NTHREADS) scatter_kernel(const __grid_constant__ CUtensorMap tmap, CicGeom g,
                                                           const uint4 *__restrict__ rec, const int *__restrict__ offsets,
                                                           const float *__restrict__ val, float *__restrict__ mesh)
{
    constexpr int NST = C == 1 ? 3 : 2;  // = scatter_stages<C>()
    extern __shared__ __align__(128) unsigned char dsm[];
    typedef int AccBuf[C][TILE_PTS];
    AccBuf *acc = reinterpret_cast<AccBuf *>(dsm);                                        // [2]
    typedef uint4 RecBuf[RCAP];
    RecBuf *recbuf = reinterpret_cast<RecBuf *>(dsm + (size_t)2 * C * TILE_PTS * sizeof(int));  // [NST]
    __shared__ __align__(8) unsigned long long full[NST], empty[NST];
    __shared__ ScatterSlot slot[NST];
    __shared__ float redf[NCW];
    __shared__ unsigned redu[NCW];
    __shared__ int heavy_last;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < NST; s++) { mbar_init(&full[s], 32); mbar_init(&empty[s], NCW); }
        mbar_fence_init();
    }
    __syncthreads();
    pdl_enter();

    if (warp == NCW) {
        // ---------------- producer warp ----------------
        // run lookup of a tile: lanes 0..13 read the offsets of their run (the loads of tile n + 1 are issued before
        // tile n is published, so their latency hides behind the stage wait)
        auto lookup = [&](int tile, int &b, int &len, int &n0) {
            b = 0; len = 0; n0 = 0;
            if (tile < g.ntiles && lane < NRUNS) {
                int t[3], t0[3], ext[3];
                tile_coords(g, tile, t, t0, ext);
                const int m = kRuns[lane][0], c0 = kRuns[lane][1], c1 = kRuns[lane][2];
                bool valid = true;
                int nb[3];
#pragma unroll
                for (int d = 0; d < 3; d++) {
                    const int low = (m >> (2 - d)) & 1;
                    if (low && g.nt[d] == 1) valid = false;  // the only tile along d is its own neighbour
                    nb[d] = t[d] - low;
                    if (nb[d] < 0) nb[d] += g.nt[d];
                }
                if (valid) {
                    const int key = ((nb[0] * g.nt[1] + nb[1]) * g.nt[2] + nb[2]) * NCLS;
                    b = offsets[key + c0];
                    len = offsets[key + c1] - b;
                    if (lane == 0) n0 = offsets[key + 1] - b;
                }
            }
        };
        // Two register sets used by alternate iterations (the loop body is instantiated twice): the run lookup of tile
        // n + 2 is requested at the end of iteration n into the set iteration n has just finished with, so every lookup
        // has a whole iteration to complete and no value in flight is copied at the loop's back edge.
        TileDraw draw;
        if (lane == 0) draw.init(g.sched);
        auto draw_lookup = [&](int &tile, int &b, int &len, int &n0) {
            int t = 0;
            if (lane == 0) t = draw.next(g.sched);
            tile = __shfl_sync(0xffffffffu, t, 0);
            lookup(tile, b, len, n0);
        };
        int tileA, bA, lenA, n0A, tileB, bB, lenB, n0B;
        draw_lookup(tileA, bA, lenA, n0A);
        draw_lookup(tileB, bB, lenB, n0B);
        // publishes one work item into stage s: run table, flat range [lo, hi) and the staged records of that range
        // inclusive prefix of the run lengths over the lanes; returns the total
        auto run_scan = [&](int len, int &inc) {
            inc = len;
#pragma unroll
            for (int o = 1; o < 16; o <<= 1) {
                const int u = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += u;
            }
            return __shfl_sync(0xffffffffu, inc, NRUNS - 1);
        };
        auto publish = [&](int s, int tile, int b, int len, int inc, int total, int n0, int lo, int hi, int pool) {
            const int start = inc - len;
            if (hi < 0) hi = total;
            if (lane < NRUNS) {
                slot[s].run_start[lane] = b - start;
                slot[s].run_prefix[lane + 1] = inc;
            }
            // this lane's run restricted to [lo, min(hi, lo + RCAP)): staged at recbuf[flat - lo]
            const int s0 = max(start, lo), e0 = min(min(start + len, hi), lo + RCAP);
            const int cnt = lane < NRUNS ? max(e0 - s0, 0) : 0;
            if (lane == 0) {
                slot[s].run_prefix[0] = 0;
                slot[s].tile = tile;
                slot[s].total = total;
                slot[s].n0 = n0;
                slot[s].lo = lo;
                slot[s].hi = hi;
                slot[s].pool = pool;
                // the tile's own run: one bulk copy; the (short) neighbour runs: 16-byte async copies, one lane per run
                if (cnt > 0) {
                    mbar_expect_tx(&full[s], (unsigned)cnt * (unsigned)sizeof(uint4));
                    bulk_load(&recbuf[s][s0 - lo], rec + b + (s0 - start), (unsigned)cnt * (unsigned)sizeof(uint4), &full[s]);
                } else {
                    mbar_arrive(&full[s]);
                }
            } else {
                for (int k = 0; k < cnt; k++) cp_async16(&recbuf[s][s0 - lo + k], rec + b + (s0 - start) + k);
                cp_async_arrive(&full[s]);
            }
        };
        bool draw_done = false;
        auto body = [&](const int n, int &tile, int &b, int &len, int &n0) -> bool {
            const int s = n % NST;
            mbar_wait(&empty[s], ((n / NST) & 1) ^ 1);
            if (tile < g.ntiles) {
                // A heavy tile (unit mass only) is split into chunks of SCHUNK records that any CTA may take from the global
                // queue; the chunks add their integer accumulators into one global accumulator of the pool (same scale:
                // it depends on the tile's total only), and the last chunk to arrive converts and stores the tile.
                int inc;
                const int total = run_scan(len, inc);
                int lo = 0, hi = -1, pool = -1;
                if (!HAS_VAL && C == 1 && total > SCHUNK + SCHUNK / 2) {
                    const int k = (total + SCHUNK - 1) / SCHUNK;
                    int base = -1;
                    if (lane == 0) {
                        pool = atomicAdd(&g.spool_ctl[0], 1);
                        if (pool < g.spool_n) base = wq_reserve(g, k - 1);
                        if (base < 0) pool = -1;  // no accumulator or no room in the queue: the tile stays whole
                    }
                    pool = __shfl_sync(0xffffffffu, pool, 0);
                    base = __shfl_sync(0xffffffffu, base, 0);
                    if (pool >= 0) {
                        for (int i = lane; i < k - 1; i += 32) wq_write(g, base + i, tile, SCHUNK * (i + 1), min(total, SCHUNK * (i + 2)), pool);
                        __threadfence();
                        __syncwarp();
                        for (int i = lane; i < k - 1; i += 32) wq_tag(g, base + i);
                        __threadfence();
                        hi = SCHUNK;
                    }
                }
                publish(s, tile, b, len, inc, total, n0, lo, hi, pool);
                if (lane == 0) atomicAdd(&g.wq[2], 1);  // one more tile whose chunks (if any) are in the queue
                draw_lookup(tile, b, len, n0);  // for iteration n + 2
                return true;
            }
            // the tile counter is exhausted: chunks from the queue (fetch-and-add head; see the gather kernel), then finish
            int it_tile = -1, it_lo = 0, it_hi = 0, it_pool = -1;
            if (lane == 0 && !draw_done) {
                if (!wq_pop(g, it_tile, it_lo, it_hi, it_pool)) it_tile = -1;
            }
            it_tile = __shfl_sync(0xffffffffu, it_tile, 0);
            if (it_tile < 0) {
                draw_done = true;
                if (lane == 0) {
                    slot[s].tile = -1;
                    sched_finish(g.sched, g.wq, (!HAS_VAL && C == 1) ? g.spool_ctl : nullptr);
                }
                mbar_arrive(&full[s]);
                return false;
            }
            it_lo = __shfl_sync(0xffffffffu, it_lo, 0);
            it_hi = __shfl_sync(0xffffffffu, it_hi, 0);
            it_pool = __shfl_sync(0xffffffffu, it_pool, 0);
            int qb, qlen, qn0;
            lookup(it_tile, qb, qlen, qn0);
            int qinc;
            const int qtotal = run_scan(qlen, qinc);
            publish(s, it_tile, qb, qlen, qinc, qtotal, qn0, it_lo, it_hi, it_pool);
            return true;
        };
        for (int n = 0;; n += 2) {
            if (!body(n, tileA, bA, lenA, n0A)) break;
            if (!body(n + 1, tileB, bB, lenB, n0B)) break;
        }
        return;
    }

    // ---------------- consumer warps ----------------
    const int tid = threadIdx.x;
    {
        int4 *z4 = reinterpret_cast<int4 *>(&acc[0][0][0]);
        for (int i = tid; i < 2 * C * TILE_PTS / 4; i += NCT) z4[i] = make_int4(0, 0, 0, 0);
    }
    consumer_sync();
    const float fr = 1.f / (float)(1u << g.fbits);
    const unsigned fmask = (1u << g.fbits) - 1u;

    // valued scatter: records and values of the NEXT tile's first two rounds, requested while this tile is finished
    bool pre_ok = false;
    uint4 pqa = make_uint4(0, 0, 0, 0), pqb = pqa;
    float pva[C], pvb[C];
#pragma unroll
    for (int c = 0; c < C; c++) pva[c] = pvb[c] = 0.f;
    for (int n = 0;; n++) {
        const int s = n % NST, b = n & 1;
#define PM_SSTAMP(k) do { if (PM_DBG(g.dbg & 8) && blockIdx.x == 0 && n < 40 && (tid == 0 || tid == NCT - 1)) g.dbgbuf[((tid ? 1 : 0) * 40 + n) * 12 + (k)] = clock64(); } while (0)
        PM_SSTAMP(0);
        mbar_wait(&full[s], (n / NST) & 1);
        PM_SSTAMP(1);
        const ScatterSlot &sl = slot[s];
        const int tile = sl.tile;
        if (tile < 0) break;
        const int total = sl.total, n0 = sl.n0;
        const int lo = sl.lo, hi = sl.hi, pool = sl.pool;
        int t[3], t0[3], ext[3];
        tile_coords(g, tile, t, t0, ext);

        // flat index -> record: the first RCAP of the range are staged in shared memory, the rest come from global
        auto fetch = [&](int i) -> uint4 {
            if (i - lo < RCAP) return recbuf[s][i - lo];
            int r = 0;
            while (i >= sl.run_prefix[r + 1]) r++;
            return rec[sl.run_start[r] + i];
        };
        auto values = [&](uint4 q, float v[C]) {
#pragma unroll
            for (int c = 0; c < C; c++) v[c] = val[(size_t)q.w * C + c];
        };
        int *tile_acc = &acc[b][0][0];

        float scale;
        if (!HAS_VAL) {
            // unit mass: deposits are >= 0 -> UNSIGNED accumulation with scale = (2^32 - headroom) / total.  total is an
            // integer, so the scale is the same in every run: the density mesh stays bit-reproducible.  No point can
            // overflow: sum of weights at a point <= total, and each of the <= total deposits rounds by <= 0.5.
            const float room = fmaxf(4294967296.f * 0.99999f - (float)total, 1.f);
            scale = room / fmaxf((float)total, 1.f);
            if (PM_DBG(g.kshift)) scale = ldexpf(scale, -g.kshift);
            for (int i = lo + tid; i < hi; i += NCT) {
                const uint4 q = fetch(i);
                if (i < n0) {
                    Corners<true> cn(g, t0, ext, q, fr, fmask);
                    cn.each([&](int a, float w, bool) { red_shared(tile_acc + a, (int)__float2uint_rn(w * scale), true, true); });
                } else {
                    Corners<false> cn(g, t0, ext, q, fr, fmask);
                    cn.each([&](int a, float w, bool ok) { red_shared(tile_acc + a, (int)__float2uint_rn(w * scale), ok, false); });
                }
            }
        } else {
            // values: signed fixed point with a power-of-two scale from a bound on |sum| at any point of the tile.
            // The bound comes from a first pass that deposits w * max_c|v_c| (unsigned, coarse scale from
            // total * max|v|); its maximum over the tile, plus the rounding slack, bounds every component's sum.
            // Integer atomics and a float max only: the result does not depend on the order of the records.
            const int ia = tid, ib = tid + NCT;
            uint4 qa = make_uint4(0, 0, 0, 0), qb = qa;
            float va[C], vb[C];
#pragma unroll
            for (int c = 0; c < C; c++) va[c] = vb[c] = 0.f;
            if (pre_ok) {
                qa = pqa; qb = pqb;
#pragma unroll
                for (int c = 0; c < C; c++) { va[c] = pva[c]; vb[c] = pvb[c]; }
            } else {
                if (ia < total) { qa = fetch(ia); values(qa, va); }
                if (ib < total) { qb = fetch(ib); values(qb, vb); }
            }
            float ma = 0.f, mb = 0.f;
#pragma unroll
            for (int c = 0; c < C; c++) { ma = fmaxf(ma, fabsf(va[c])); mb = fmaxf(mb, fabsf(vb[c])); }
            float vmax = fmaxf(ma, mb);
            for (int i = ib + NCT; i < total; i += NCT) {
                float v[C];
                values(fetch(i), v);
#pragma unroll
                for (int c = 0; c < C; c++) vmax = fmaxf(vmax, fabsf(v[c]));
            }
            vmax = consumer_max(vmax, redf);
            scale = 1.f;
            if (total > 0 && vmax > 0.f && vmax < 3e38f) {
              float bound;
              if (total <= SFAST) {
                // Light tile (the normal case: 256 records on average): no point's sum can exceed sum_i max_c |v_i,c| (weights
                // are <= 1).  That sum is formed in INTEGER units of vmax 2^-20, each term rounded up, so it does not depend on
                // the order of the records either, and it replaces the bound pass below (8 atomics per record, a scan of the
                // tile, two barriers).  For heavy tiles it would be far too loose at the sparse points of the tile.
                const float inv = 1048576.f / vmax;
                unsigned qs = 0u;
                if (ia < total) qs += (unsigned)(ma * inv) + 2u;
                if (ib < total) qs += (unsigned)(mb * inv) + 2u;
                for (int i = ib + NCT; i < total; i += NCT) {
                    float v[C], m = 0.f;
                    values(fetch(i), v);
#pragma unroll
                    for (int c = 0; c < C; c++) m = fmaxf(m, fabsf(v[c]));
                    qs += (unsigned)(m * inv) + 2u;
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) qs += __shfl_xor_sync(0xffffffffu, qs, o);
                if (lane == 0) redu[warp] = qs;
                consumer_sync();
                qs = 0u;
#pragma unroll
                for (int k2 = 0; k2 < NCW; k2++) qs += redu[k2];
                consumer_sync();
                bound = ((float)qs * 1.0000002f) * (vmax * (1.f / 1048576.f)) * 1.001f;
              } else {
                const float sA = __uint_as_float((unsigned)(127 + min(31 - exp_above(fmaxf((float)total * vmax, 1e-30f)), 96)) << 23);
                auto pass_a = [&](int i, uint4 q, float m) {
                    const float ms = m * sA;
                    if (i < n0) {
                        Corners<true> cn(g, t0, ext, q, fr, fmask);
                        cn.each([&](int a, float w, bool) { red_shared(tile_acc + a, (int)__float2uint_rn(w * ms), true, true); });
                    } else {
                        Corners<false> cn(g, t0, ext, q, fr, fmask);
                        cn.each([&](int a, float w, bool ok) { red_shared(tile_acc + a, (int)__float2uint_rn(w * ms), ok, false); });
                    }
                };
                if (ia < total) pass_a(ia, qa, ma);
                if (ib < total) pass_a(ib, qb, mb);
                for (int i = ib + NCT; i < total; i += NCT) {
                    const uint4 q = fetch(i);
                    float v[C], m = 0.f;
                    values(q, v);
#pragma unroll
                    for (int c = 0; c < C; c++) m = fmaxf(m, fabsf(v[c]));
                    pass_a(i, q, m);
                }
                consumer_sync();
                unsigned um = 0u;
                for (int i = tid; i < TILE_PTS; i += NCT) {
                    um = max(um, (unsigned)tile_acc[i]);
                    tile_acc[i] = 0;
                }
                const float M = consumer_max((float)um * 1.0000002f, redf);  // (float) may round down: one ulp up
                bound = (M + 0.5f * (float)total + 1.f) / sA * 1.001f;
              }
                const int k = min(30 - exp_above(fmaxf(bound, 1e-37f)), 96) - PM_DBG(g.kshift);
                scale = __uint_as_float((unsigned)(127 + k) << 23);
                auto pass_b = [&](int i, uint4 q, const float v[C]) {
                    float vs[C];
#pragma unroll
                    for (int c = 0; c < C; c++) vs[c] = v[c] * scale;
                    if (i < n0) {
                        Corners<true> cn(g, t0, ext, q, fr, fmask);
                        cn.each([&](int a, float w, bool) {
#pragma unroll
                            for (int c = 0; c < C; c++) red_shared(tile_acc + c * TILE_PTS + a, __float2int_rn(w * vs[c]), true, true);
                        });
                    } else {
                        Corners<false> cn(g, t0, ext, q, fr, fmask);
                        cn.each([&](int a, float w, bool ok) {
#pragma unroll
                            for (int c = 0; c < C; c++) red_shared(tile_acc + c * TILE_PTS + a, __float2int_rn(w * vs[c]), ok, false);
                        });
                    }
                };
                if (ia < total) pass_b(ia, qa, va);
                if (ib < total) pass_b(ib, qb, vb);
                for (int i = ib + NCT; i < total; i += NCT) {
                    const uint4 q = fetch(i);
                    float v[C];
                    values(q, v);
                    pass_b(i, q, v);
                }
            }
        }
        if (HAS_VAL) {
            // if the producer has the next tile staged already, request its first two rounds of values now: their
            // round trip then overlaps the conversion and the store of this tile
            const int s1 = (n + 1) % NST;
            pre_ok = mbar_test(&full[s1], ((n + 1) / NST) & 1) && slot[s1].tile >= 0 && slot[s1].pool < 0;
            if (pre_ok) {
                const int total1 = slot[s1].total;
#pragma unroll
                for (int c = 0; c < C; c++) pva[c] = pvb[c] = 0.f;
                pqa = pqb = make_uint4(0, 0, 0, 0);
                if (tid < total1) {
                    pqa = recbuf[s1][tid];
#pragma unroll
                    for (int c = 0; c < C; c++) pva[c] = val[(size_t)pqa.w * C + c];
                }
                if (tid + NCT < total1) {
                    pqb = recbuf[s1][tid + NCT];
#pragma unroll
                    for (int c = 0; c < C; c++) pvb[c] = val[(size_t)pqb.w * C + c];
                }
            }
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

        PM_SSTAMP(2);
        if (PM_DBG(g.dbg & 8) && blockIdx.x == 0 && n < 40 && tid == 0) g.dbgbuf[n * 12 + 11] = sl.total;
        if (tid == 0) tma_store_wait_read();  // the previous tile's store has read the other buffer out
        PM_SSTAMP(3);
        consumer_sync();                      // all deposits of this tile are in; the other buffer is free
        PM_SSTAMP(4);
        if (lane == 0) mbar_arrive(&empty[s]);
        bool do_store = true;
        if (!HAS_VAL && C == 1 && pool >= 0) {
            // chunk of a heavy tile: add the accumulators into the tile's global accumulator (integers: the result does
            // not depend on who adds first and equals what one CTA alone would have accumulated); the chunk that finds
            // all others done takes the sums back, converts and stores them and leaves the accumulator zeroed
            unsigned *gp = g.spool + (size_t)pool * TILE_PTS;
            for (int i = tid; i < TILE_PTS; i += NCT) {
                const unsigned v = (unsigned)tile_acc[i];
                if (v) atomicAdd(gp + i, v);
            }
            __threadfence();
            consumer_sync();
            if (tid == 0) heavy_last = atomicAdd(&g.spool_ctl[16 + pool], 1) == (total + SCHUNK - 1) / SCHUNK - 1;
            consumer_sync();
            do_store = heavy_last != 0;
            if (do_store) {
                __threadfence();
                for (int i = tid; i < TILE_PTS; i += NCT) {
                    tile_acc[i] = (int)__ldcg(gp + i);
                    gp[i] = 0u;
                }
                if (tid == 0) g.spool_ctl[16 + pool] = 0;
            }
            consumer_sync();
        }
        {
            // int -> float in place (same bytes), and the other buffer is zeroed for the next tile
            int4 *a4 = reinterpret_cast<int4 *>(tile_acc);
            int4 *o4 = reinterpret_cast<int4 *>(&acc[b ^ 1][0][0]);
            for (int i = tid; i < C * TILE_PTS / 4; i += NCT) {
                const int4 a = a4[i];
                float4 f;
                if (HAS_VAL) {
                    f = make_float4((float)a.x * inv_scale, (float)a.y * inv_scale, (float)a.z * inv_scale, (float)a.w * inv_scale);
                } else if (mq == 0) {
                    f = make_float4((float)(unsigned)a.x * inv_scale, (float)(unsigned)a.y * inv_scale,
                                    (float)(unsigned)a.z * inv_scale, (float)(unsigned)a.w * inv_scale);
                } else if ((a.x | a.y | a.z | a.w) >= 0 && mq < (1ll << 30)) {
                    // all four below 2^31 (every point but the densest): the exact difference fits in 32 bits
                    const int m32 = (int)mq;
                    f = make_float4((float)(a.x - m32) * inv_scale - mrest, (float)(a.y - m32) * inv_scale - mrest,
                                    (float)(a.z - m32) * inv_scale - mrest, (float)(a.w - m32) * inv_scale - mrest);
                } else {
                    f = make_float4((float)((long long)(unsigned)a.x - mq) * inv_scale - mrest, (float)((long long)(unsigned)a.y - mq) * inv_scale - mrest,
                                    (float)((long long)(unsigned)a.z - mq) * inv_scale - mrest, (float)((long long)(unsigned)a.w - mq) * inv_scale - mrest);
                }
                reinterpret_cast<float4 *>(a4)[i] = f;
                o4[i] = make_int4(0, 0, 0, 0);
            }
        }
        fence_proxy_async_smem();
        PM_SSTAMP(5);
        consumer_sync();
        PM_SSTAMP(6);
        if (!do_store) {
            // another chunk of this tile stores it
        } else if (g.use_tma) {
            if (tid == 0) {
#pragma unroll
                for (int c = 0; c < C; c++) tma_store_4d(&tmap, tile_acc + c * TILE_PTS, t0[2], t0[1], t0[0], g.c0 + c);
                tma_store_commit();
            }
        } else {
            // plain path: one warp per z-row
            const float *facc = reinterpret_cast<const float *>(tile_acc);
            for (int row = warp; row < TX * TY; row += NCW) {
                const int lx = row / TY, ly = row % TY;
                if (lx < ext[0] && ly < ext[1] && lane < ext[2]) {
                    const size_t o = ((size_t)(t0[0] + lx) * g.N[1] + (t0[1] + ly)) * g.zs + (t0[2] + lane);
#pragma unroll
                    for (int c = 0; c < C; c++) mesh[(size_t)c * g.ms + o] = facc[c * TILE_PTS + row * TZ + lane];
                }
            }
            consumer_sync();  // the rows are out before anyone zeroes this buffer at the next tile
        }
    }
    if (tid == 0) tma_store_wait_all();
}

// --------------------------------------------------------------------------------------------------
// gathers
// --------------------------------------------------------------------------------------------------
// Measured on B200 (profiles/): TMA tensor loads of these narrow halo boxes (144-byte rows) sustain only about
// one row per 12 cycles per SM, and a single producer warp issuing 16-byte async copies is issue-bound; 256
// threads issuing the 16-byte copies themselves (9 per thread and tile) are not.  So the gather is a classic
// two-stage cp.async pipeline: every thread first starts the copies of the NEXT tile's halo, then interpolates
// for the particles of the current one.
enum GatherMode { G_VALUE = 0, G_GRAD = 1, G_FUSED = 2 };
constexpr int GT = 256;                                    // threads of a gather CTA
constexpr int GCH = HZP / 4;                               // 16-byte pieces per halo row (9)
constexpr int GRG = GT / GCH;                              // halo rows covered per pass of the CTA (28)

struct GatherSlot {
    int tile;  // -1: no more tiles
    int beg, end;
    int t0[3], ext[3];  // first mesh point and extent of the tile (computed once, by the drawing thread)
};

// halo stages per CTA (GST - 1 tiles in flight while one is computed).  Measured at 256^3: a single 47 KB stage for the
// four-mesh fused gather (three CTAs per SM instead of two) is slower (230 vs 221 us), three stages are slower too.
#define PM_GST(C) ((C) == 4 ? PM_GST4 : 2)
#ifndef PM_GST4
#define PM_GST4 2
#endif
template <int C>
constexpr size_t gather_smem_bytes() { return (size_t)PM_GST(C) * C * HALO_STRIDE * sizeof(float); }

__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// starts the copies of one tile's halo (C meshes) into `halo`; every thread of the CTA takes part
template <int C>
__device__ __forceinline__ void halo_issue(const CicGeom &g, const float *__restrict__ mesh, const GatherSlot &sl, float *halo)
{
    const int t0[3] = {sl.t0[0], sl.t0[1], sl.t0[2]}, ext[3] = {sl.ext[0], sl.ext[1], sl.ext[2]};
    const bool rows_ok = g.use_tma && (g.N[2] & 3) == 0;  // 16-byte aligned rows
    if (rows_ok) {
        // rows (lx, ly), lx <= ext[0], ly <= ext[1], wrapped periodically; along z either HZP contiguous floats or,
        // at the upper edge, the floats up to the edge plus 4 from z = 0.  thread -> (row of a group of GRG rows,
        // 16-byte piece); (lx, ly) are carried along, so the loop has no division.
        const bool zwrap = t0[2] + HZP > g.N[2];
        const int cpr_main = (zwrap ? g.N[2] - t0[2] : HZP) / 4;
        const int cpr = cpr_main + (zwrap ? 1 : 0);
        const int ny = ext[1] + 1, nrow = (ext[0] + 1) * ny;
        const int rg = threadIdx.x / GCH, ch = threadIdx.x - rg * GCH;
        if (rg < GRG && ch < cpr) {
            const int zoff = ch < cpr_main ? t0[2] + ch * 4 : 0;
            // full tiles (ny == HY): compile-time divisors
            int lx = ny == HY ? rg / HY : rg / ny, ly = rg - lx * ny;
            const int dlx = ny == HY ? GRG / HY : GRG / ny, dly = GRG - dlx * ny;
            for (int r = rg; r < nrow; r += GRG) {
                int gx = t0[0] + lx, gy = t0[1] + ly;
                if (gx >= g.N[0]) gx -= g.N[0];
                if (gy >= g.N[1]) gy -= g.N[1];
                const float *src = mesh + ((size_t)gx * g.N[1] + gy) * g.zs + zoff;
                float *dst = halo + (lx * HY + ly) * HZP + ch * 4;
#pragma unroll
                for (int c = 0; c < C; c++) cp_async16(dst + c * HALO_STRIDE, src + (size_t)c * g.ms);
                lx += dlx;
                ly += dly;
                if (ly >= ny) { ly -= ny; lx++; }
            }
        }
    } else {
        // meshes whose layout 16-byte copies cannot address: plain loads
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
        for (int r = w; r < C * HX * HY; r += GT / 32) {
            const int c = r / (HX * HY), r2 = r % (HX * HY);
            const int lx = r2 / HY, ly = r2 % HY;
            if (lx <= ext[0] && ly <= ext[1]) {
                int gx = t0[0] + lx, gy = t0[1] + ly;
                if (gx >= g.N[0]) gx -= g.N[0];
                if (gy >= g.N[1]) gy -= g.N[1];
                const float *src = mesh + (size_t)c * g.ms + ((size_t)gx * g.N[1] + gy) * g.zs;
                float *dst = halo + c * HALO_STRIDE + (lx * HY + ly) * HZP;
                for (int lz = lane; lz <= ext[2]; lz += 32) {
                    int gz = t0[2] + lz;
                    if (gz >= g.N[2]) gz -= g.N[2];
                    dst[lz] = src[gz];
                }
            }
        }
    }
}

// per-particle inputs that are fetched one tile ahead
template <int C, int MODE, bool HAS_COT, bool KICK>
struct ParticleIn {
    float cv[C];
    long long p[3], x[3];
    float xi[3];
    __device__ __forceinline__ void load(size_t j, const float *cot, const KickArgs &ka)
    {
        if (MODE == G_GRAD) {
#pragma unroll
            for (int c = 0; c < C; c++) cv[c] = HAS_COT ? cot[j * C + c] : 1.f;
        }
        if (MODE == G_FUSED) {
            cv[0] = 1.f;
#pragma unroll
            for (int c = 1; c < C; c++) cv[c] = cot[j * 3 + (c - 1)];
        }
        if (KICK) {
#pragma unroll
            for (int d = 0; d < 3; d++) {
                p[d] = ka.p[3 * j + d];
                if (ka.Ds != 0.0) x[d] = ka.x[3 * j + d];
                if (MODE == G_FUSED) xi[d] = ka.xi[3 * j + d];
            }
        }
    }
};

// KICK: the interpolated acc (and alpha) of a particle is applied on the spot -- p += rn(acc Ka) [+= rn(acc Kb)],
// x += rn(p D), and for the adjoint xi -= alpha K, pi -= xi D (eq. 16 L172 / eq. 49, same arithmetic and
// order as kick_drift_kernel) -- and the particle's new sort key is added to the histogram of the next sort, so
// a step needs no separate kick/drift and histogram passes and acc/alpha never travel through HBM.
template <int C, int MODE, bool HAS_COT, bool KICK>
__global__ void __launch_bounds__(GT) gather_kernel(CicGeom g, const uint4 *__restrict__ rec, const int *__restrict__ offsets,
                                                    const float *__restrict__ mesh, const float *cot, float cot_scale,
                                                    float *__restrict__ out, float *__restrict__ out2, PosGeom pg, KickArgs ka)
{
    constexpr int GST = PM_GST(C);
    constexpr int PUB = GST < 2 ? 2 : GST;  // tiles are published PUB iterations ahead (the record prefetch looks one ahead)
    extern __shared__ __align__(128) unsigned char dsm[];
    __shared__ GatherSlot slot[8];  // ring of drawn tiles: iteration n computes slot[n & 7] and starts the copies of slot[(n + GST - 1) & 7]
    auto halo_of = [&](int s) { return reinterpret_cast<float *>(dsm) + (size_t)s * C * HALO_STRIDE; };
    const int tid = threadIdx.x;
    typedef ParticleIn<C, MODE, HAS_COT, KICK> PIn;

    // thread 0 draws tiles from the global counter and publishes them two iterations ahead.  The chain
    // atomic -> offsets -> slot is software-pipelined: every iteration consumes what the previous one requested
    // (the tile index of the atomic, the offsets of the tile drawn before), so no round trip is exposed.
    pdl_enter();
    // The tiles are drawn by the LAST thread: its warp has particles only in tiles with more than GT - 32 of them, so the
    // round trips of the draw rarely sit on the critical path to the barrier (warp 0 always has the most particles).
    constexpr int DRAWER = GT - 1;
    // The pipeline registers come in two sets used by alternate iterations (the loop body is instantiated twice): a
    // freshly requested value is then never copied at the loop's back edge, which would wait for its round trip.
    struct DrawSet { int tile, beg, end; };
    DrawSet S0 = {0, 0, 0}, S1 = {0, 0, 0};  // drawing thread only: tile whose offsets are in flight
    int a0 = 0, a1 = 0;                      // drawing thread only: tile index of the atomic in flight
    auto draw_request = [&](DrawSet &fill, const int &a_use, int &a_new) {
        fill.tile = a_use;
        if (fill.tile < g.ntiles) {
            fill.beg = offsets[fill.tile * NCLS];
            fill.end = offsets[fill.tile * NCLS + NCLS];
        }
        a_new = atomicAdd(&g.sched[0], 1);
    };
    // Publishing a drawn tile.  A tile with more than GCHUNK particles is split: the first chunk is published, the others
    // go to a global queue from which any CTA takes them once the tile counter is exhausted (a dense clump would
    // otherwise keep one CTA busy long after all others have finished); protocol: see wq_reserve / wq_pop above.
    bool draw_done = false;  // drawing thread only
    auto publish_range = [&](GatherSlot &dst, int tile, int beg, int end) {
        dst.tile = tile;
        dst.beg = beg;
        dst.end = end;
        int tt[3], tt0[3], text[3];
        tile_coords(g, tile, tt, tt0, text);
#pragma unroll
        for (int k = 0; k < 3; k++) { dst.t0[k] = tt0[k]; dst.ext[k] = text[k]; }
    };
    auto draw_publish = [&](GatherSlot &dst, const DrawSet &d) {
        if (d.tile < g.ntiles) {
            int end = d.end;
            if (end - d.beg > GCHUNK) {
                const int k = (end - d.beg + GCHUNK - 1) / GCHUNK - 1;
                const int base = wq_reserve(g, k);
                if (base >= 0) {
                    for (int i = 0; i < k; i++) wq_write(g, base + i, d.tile, d.beg + GCHUNK * (i + 1), min(d.end, d.beg + GCHUNK * (i + 2)), -1);
                    __threadfence();
                    for (int i = 0; i < k; i++) wq_tag(g, base + i);
                    __threadfence();  // the tail update and the items are visible before this tile counts as published
                    end = d.beg + GCHUNK;
                }
            }
            publish_range(dst, d.tile, d.beg, end);
            atomicAdd(&g.wq[2], 1);  // one more tile whose chunks (if any) are in the queue (fenced above when it had any)
            return;
        }
        // the tile counter is exhausted: take a chunk from the queue, or finish (and stay finished: the CTA stops at the
        // first slot marked -1, so nothing may be taken from the queue after that)
        if (draw_done) { dst.tile = -1; return; }
        int qt, qlo, qhi, qpool;
        if (wq_pop(g, qt, qlo, qhi, qpool)) {
            publish_range(dst, qt, qlo, qhi);
        } else {
            draw_done = true;
            dst.tile = -1;
        }
    };
    if (tid == DRAWER) {
        // prologue (latencies exposed once): after it S0 holds the tile to publish at iteration 0 and a0 the next index
        int a = atomicAdd(&g.sched[0], 1), b = 0;
        draw_request(S0, a, b);
        for (int k = 0; k < PUB; k++) {
            draw_publish(slot[k], S0);
            a = b;
            draw_request(S0, a, b);
        }
        a0 = b;
    }
    __syncthreads();
    for (int k = 0; k < GST - 1; k++) {
        if (slot[k].tile >= 0 && slot[k].beg < slot[k].end) halo_issue<C>(g, mesh, slot[k], halo_of(k));
        cp_async_commit();
    }
    // first round of the first tile: record and per-particle inputs
    uint4 q = make_uint4(0, 0, 0, 0);
    PIn pin;
    if (slot[0].tile >= 0 && slot[0].beg + tid < slot[0].end) {
        q = rec[slot[0].beg + tid];
        pin.load(q.w, cot, ka);
    }

    const float fr = 1.f / (float)(1u << g.fbits);
    const unsigned fmask = (1u << g.fbits) - 1u;
    auto body = [&](const int n, DrawSet &Spub, DrawSet &Sfill, int &a_use, int &a_new) -> bool {
        const GatherSlot cur = slot[n & 7];
        if (cur.tile < 0) return false;
#define PM_STAMP(k) do { if (PM_DBG(g.dbg & 8) && blockIdx.x == 0 && n < 40 && (tid == 0 || tid == GT - 1)) g.dbgbuf[((tid ? 1 : 0) * 40 + n) * 12 + (k)] = clock64(); } while (0)
        PM_STAMP(0);
        if (PM_DBG(g.dbg & 8) && blockIdx.x == 0 && n < 40 && tid == 0) g.dbgbuf[n * 12 + 11] = cur.end - cur.beg;
        // the halo of the tile GST - 1 iterations ahead starts to fly now (its stage was released by the barrier that
        // ended iteration n - 1)
        {
            const GatherSlot far = slot[(n + GST - 1) & 7];
            if (far.tile >= 0 && far.beg < far.end && !PM_DBG(g.dbg & 2)) halo_issue<C>(g, mesh, far, halo_of((n + GST - 1) % GST));
        }
        cp_async_commit();
        PM_STAMP(1);
        const GatherSlot nxt = slot[(n + 1) & 7];
        uint4 q_nx = make_uint4(0, 0, 0, 0);
        const bool has_nx = nxt.tile >= 0 && nxt.beg + tid < nxt.end;
        if (has_nx) q_nx = rec[nxt.beg + tid];
        // a second round of the current tile (more than GT particles): its record is requested now, its per-particle
        // inputs right after the barrier, so that neither round trip is exposed between the rounds
        const int cnt = PM_DBG(g.dbg & 1) ? 0 : cur.end - cur.beg;
        uint4 q2 = make_uint4(0, 0, 0, 0);
        if (tid + GT < cnt) q2 = rec[cur.beg + tid + GT];
        cp_async_wait<GST - 1>();  // this thread's copies of the current tile have landed ...
        PM_STAMP(2);
        __syncthreads();     // ... and everybody else's
        PM_STAMP(3);
        PIn pin2;
        if (tid + GT < cnt) pin2.load(q2.w, cot, ka);

        const int t0[3] = {cur.t0[0], cur.t0[1], cur.t0[2]};
        const float *halo = halo_of(n % GST);
        for (int i = tid; i < cnt; i += GT) {
            if (i == tid + GT) {
                q = q2;
                pin = pin2;
            } else if (i != tid) {
                q = rec[cur.beg + i];
                pin.load(q.w, cot, ka);
            }
            const size_t j = q.w;
            const unsigned X[3] = {q.x, q.y, q.z};
            int l[3];
            float w[3][2];
#pragma unroll
            for (int d = 0; d < 3; d++) {
                l[d] = (int)(X[d] >> g.fbits) - t0[d];
                const float td = (float)(X[d] & fmask) * fr;
                w[d][0] = 1.f - td;
                w[d][1] = td;
            }
            const int base = (l[0] * HY + l[1]) * HZP + l[2];
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
                            if (MODE != G_VALUE) m += pin.cv[c] * f;
                        }
                        if (MODE != G_VALUE) {
                            gr[0] += dWx * m;
                            gr[1] += dWy * m;
                            gr[2] += dWz * m;
                        }
                    }
            if (KICK) {
                const float *a3 = MODE == G_FUSED ? &val[C - 3] : &val[0];
                unsigned int Xn[3];
#pragma unroll
                for (int d = 0; d < 3; d++) {
                    const size_t i3 = 3 * j + d;
                    long long pv = pin.p[d];
                    if (ka.Ka != 0.0) pv += __double2ll_rn((double)a3[d] * ka.Ka);
                    if (ka.Kb != 0.0) pv += __double2ll_rn((double)a3[d] * ka.Kb);
                    ka.p[i3] = pv;
                    if (MODE == G_FUSED) {
                        float v = pin.xi[d];
                        if (ka.Ka != 0.0) v = fmaf(-gr[d], ka.Kaf, v);
                        if (ka.Kb != 0.0) v = fmaf(-gr[d], ka.Kbf, v);
                        ka.xi[i3] = v;
                        if (ka.Ds != 0.0) ka.pi[i3] = fmaf(-v, ka.Df, pin.cv[C - 3 + d]);
                    }
                    if (ka.Ds != 0.0) {
                        const long long xv = pin.x[d] + __double2ll_rn((double)pv * ka.Ds);
                        ka.x[i3] = xv;
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
                if (PM_DBG(g.dbg & 4) && val[0] != 12345.f) continue;
#pragma unroll
                for (int c = 0; c < C; c++) out[j * C + c] = val[c];
            } else if (MODE == G_GRAD) {
#pragma unroll
                for (int e = 0; e < 3; e++) out[j * 3 + e] = gr[e] * cot_scale;
            } else {
#pragma unroll
                for (int e = 0; e < 3; e++) {
                    out[j * 3 + e] = val[C - 3 + e];
                    out2[j * 3 + e] = gr[e];
                }
            }
        }
        PM_STAMP(4);
        // the next tile's first record has arrived by now: its per-particle inputs are requested before the barrier
        q = q_nx;
        if (has_nx) pin.load(q.w, cot, ka);
        PM_STAMP(7);
        if (tid == DRAWER) {
            draw_publish(slot[(n + PUB) & 7], Spub);
            PM_STAMP(8);
            draw_request(Sfill, a_use, a_new);
        }
        PM_STAMP(5);
        __syncthreads();  // stage n % GST may be overwritten; slot[(n + PUB) & 7] is published
        PM_STAMP(6);
        return true;
    };
    for (int n = 0;; n += 2) {
        if (!body(n, S0, S1, a0, a1)) break;
        if (!body(n + 1, S1, S0, a1, a0)) break;
    }
    cp_async_wait<0>();
    if (tid == DRAWER) sched_finish(g.sched, g.wq);
}

// --------------------------------------------------------------------------------------------------
// host: launches
// --------------------------------------------------------------------------------------------------
// persistent grid: as many CTAs per SM as the stage buffers and 1536 threads allow, never more CTAs than tiles
static int persistent_grid(pm_ctx *c, size_t smem_bytes, int threads)
{
    int per_sm = (int)((size_t)(227 * 1024) / (smem_bytes + 2048));
    const int cap = 1536 / threads;  // 6 gather CTAs (256 threads) or 5 scatter CTAs (288) at most
    if (per_sm > cap) per_sm = cap;
    if (per_sm < 1) per_sm = 1;
    long long n = (long long)c->num_sms * per_sm;
    if (n > c->g.ntiles) n = c->g.ntiles;
    return (int)n;
}

template <class K>
static cudaError_t allow_smem(K kernel, size_t bytes)
{
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

#define PM_CIC_LAUNCH(ctx, name, kernel, threads, smem, ...)                                          \
    do {                                                                                     \
        static unsigned long long attr_mask_ = 0;                                            \
        if (smem_attr_needed(ctx, &attr_mask_)) PM_CUDA(ctx, allow_smem(kernel, smem));      \
        PM_CUDA(ctx, launch_pdl(kernel, dim3(persistent_grid(ctx, smem, threads)), dim3(threads), smem, (ctx)->stream, __VA_ARGS__)); \
        PM_LAUNCH_CHECK(ctx, name);                                                          \
    } while (0)

int scatter_sorted(pm_ctx *c, const float *val, int C, float *mesh, int zs, long long ms, double mean)
{
    CUtensorMap map;
    CicGeom g = make_cic_geom(c, mesh, C, zs, ms, true, &map);
    g.mean = (C == 1 && !val) ? mean : 0.0;
    double np = (double)c->cur_np, ng = (double)c->g.ng;
    if (C == 1 && !val) {
        Timer t(c, TC_SCATTER1, 12.0 * np + 4.0 * ng);
        PM_CIC_LAUNCH(c, "scatter_kernel<1>", (scatter_kernel<1, false>), NTHREADS, scatter_smem_bytes<1>(), map, g, c->rec, c->offsets, nullptr, mesh);
        t.stop();
    } else if (C == 1) {
        Timer t(c, TC_SCATTER1, 16.0 * np + 4.0 * ng);
        PM_CIC_LAUNCH(c, "scatter_kernel<1,val>", (scatter_kernel<1, true>), NTHREADS, scatter_smem_bytes<1>(), map, g, c->rec, c->offsets, val, mesh);
        t.stop();
    } else if (C == 3 && val) {
        Timer t(c, TC_SCATTER3, 24.0 * np + 12.0 * ng);
        PM_CIC_LAUNCH(c, "scatter_kernel<3,val>", (scatter_kernel<3, true>), NTHREADS, scatter_smem_bytes<3>(), map, g, c->rec, c->offsets, val, mesh);
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
    PosGeom pg = make_pos_geom(c->g);
    KickArgs none;
    memset(&none, 0, sizeof none);
    if (ka && C != 3) return fail(c, PM_EINVAL, "gather", "internal: kick needs C = 3");
    if (C == 1) {
        Timer t(c, TC_GATHER3, 16.0 * np + 4.0 * ng);
        PM_CIC_LAUNCH(c, "gather_kernel<1>", (gather_kernel<1, G_VALUE, false, false>), GT, gather_smem_bytes<1>(), g, c->rec, c->offsets, mesh, nullptr, 1.f, out, nullptr, pg, none);
        t.stop();
    } else if (C == 3 && !ka) {
        Timer t(c, TC_GATHER3, 24.0 * np + 12.0 * ng);
        PM_CIC_LAUNCH(c, "gather_kernel<3>", (gather_kernel<3, G_VALUE, false, false>), GT, gather_smem_bytes<3>(), g, c->rec, c->offsets, mesh, nullptr, 1.f, out, nullptr, pg, none);
        t.stop();
    } else if (C == 3) {
        Timer t(c, TC_GATHER_KICK, (12.0 + kick_bytes(ka, false)) * np + 12.0 * ng);
        PM_CIC_LAUNCH(c, "gather_kernel<3,kick>", (gather_kernel<3, G_VALUE, false, true>), GT, gather_smem_bytes<3>(), g, c->rec, c->offsets, mesh, nullptr, 1.f, out, nullptr, pg, *ka);
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
    PosGeom pg = make_pos_geom(c->g);
    KickArgs none;
    memset(&none, 0, sizeof none);
    if (C != 1 && C != 3) return fail(c, PM_EINVAL, "gather_grad", "C must be 1 or 3");
    Timer t(c, TC_GATHER_GRAD, (24.0 + (cot ? 4.0 * C : 0.0)) * np + 4.0 * C * ng);
    if (C == 1 && !cot)
        PM_CIC_LAUNCH(c, "gather_kernel<1,grad>", (gather_kernel<1, G_GRAD, false, false>), GT, gather_smem_bytes<1>(), g, c->rec, c->offsets, mesh, nullptr, cot_scale, out, nullptr, pg, none);
    else if (C == 1)
        PM_CIC_LAUNCH(c, "gather_kernel<1,grad,cot>", (gather_kernel<1, G_GRAD, true, false>), GT, gather_smem_bytes<1>(), g, c->rec, c->offsets, mesh, cot, cot_scale, out, nullptr, pg, none);
    else if (!cot)
        PM_CIC_LAUNCH(c, "gather_kernel<3,grad>", (gather_kernel<3, G_GRAD, false, false>), GT, gather_smem_bytes<3>(), g, c->rec, c->offsets, mesh, nullptr, cot_scale, out, nullptr, pg, none);
    else
        PM_CIC_LAUNCH(c, "gather_kernel<3,grad,cot>", (gather_kernel<3, G_GRAD, true, false>), GT, gather_smem_bytes<3>(), g, c->rec, c->offsets, mesh, cot, cot_scale, out, nullptr, pg, none);
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
    if (!ka) {
        KickArgs none;
        memset(&none, 0, sizeof none);
        Timer t(c, TC_GATHER_FUSED, 48.0 * np + 16.0 * ng);
        PM_CIC_LAUNCH(c, "gather_kernel<fused>", (gather_kernel<4, G_FUSED, true, false>), GT, gather_smem_bytes<4>(), g, c->rec, c->offsets, mesh4, pi, 1.f, acc, alpha, pg, none);
        t.stop();
    } else {
        Timer t(c, TC_GATHER_FUSED, (24.0 + kick_bytes(ka, true)) * np + 16.0 * ng);
        PM_CIC_LAUNCH(c, "gather_kernel<fused,kick>", (gather_kernel<4, G_FUSED, true, true>), GT, gather_smem_bytes<4>(), g, c->rec, c->offsets, mesh4, pi, 1.f, acc, alpha, pg, *ka);
        t.stop();
    }
    return PM_OK;
}

}  // namespace pm
