// pm_fft.cu -- own 3-D FFT passes with the k-space operators fused into the x pass (power-of-two meshes).
//
// PAPER.md L127-131 (eq. 11): the force costs "4 (1 forward and 3 inverse) FFTs"; with a library FFT that is
// 4 x 3 passes over the mesh plus the Green's-function kernel.  Here the transform along x, the multiplication
// by  i kt_d G(k)  (eq. 11; pm_kspace.cu states the operators) and the three inverse transforms along x are ONE
// kernel: a CTA holds a tile of x-columns in shared memory, transforms it, and writes the three force components
// already transformed back along x.  A force evaluation then moves
//     z R2C (1r + 1w), y (1r + 1w), x fused (1r + 3w), 3 x y^-1 (3r + 3w), 3 x z^-1 C2R (3r + 3w) = 20 mesh transfers
// instead of 28 with cuFFT (4 transforms x 3 passes x 2 + the 1r + 3w k-space kernel); the adjoint operator
// (3 meshes in, 1 out; transpose of eq. 11) is fused the same way.
//
// The 1-D transforms are Stockham-free in-place decimation-in-frequency stages of radix 16/8/4/2 on a shared-memory
// tile [position][column]: a thread loads R elements of one column into registers, runs an R-point DFT there,
// applies the stage twiddles (fp64-built table) and stores.  Forward stages leave the spectrum in digit-reversed
// order along x and y; the inverse runs the inverse stages in reverse order, so no reordering pass exists:
// only the per-axis k tables (kt, k^2, deconvolution) are stored in that permuted order.  z is kept in natural
// order (the real <-> half-complex pre/post-processing pairs k with N/2 - k inside the tile anyway).
// Conventions as cuFFT: forward e^{-ikg} unnormalised, inverse unnormalised (1/N_g is folded into G, R13).
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <type_traits>

#include "pm_internal.cuh"

namespace pm {

// ---- R-point DFT in registers ----------------------------------------------------------------------------
// complex add / subtract as ONE packed fp32x2 instruction (FADD2 on sm_100a; same rounding as two scalar adds)
__device__ __forceinline__ float2 cadd(float2 a, float2 b)
{
    unsigned long long ra = *reinterpret_cast<unsigned long long *>(&a), rb = *reinterpret_cast<unsigned long long *>(&b), rd;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
    return *reinterpret_cast<float2 *>(&rd);
}
__device__ __forceinline__ float2 csub(float2 a, float2 b)
{
    unsigned long long ra = *reinterpret_cast<unsigned long long *>(&a), rb = *reinterpret_cast<unsigned long long *>(&b), rd;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
    return *reinterpret_cast<float2 *>(&rd);
}
__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) { return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }  // a * conj(b)

// d * exp(-+ 2 pi i idx / 16); idx is a compile-time constant after unrolling
template <bool INV>
__device__ __forceinline__ float2 mul_w16(float2 d, int idx)
{
    const float c1 = 0.92387953251128674f, s1 = 0.38268343236508977f, h = 0.70710678118654752f;
    float c, s;
    switch (idx) {
        case 0: return d;
        case 1: c = c1; s = s1; break;
        case 2: c = h; s = h; break;
        case 3: c = s1; s = c1; break;
        case 4: return INV ? make_float2(-d.y, d.x) : make_float2(d.y, -d.x);
        case 5: c = -s1; s = c1; break;
        case 6: c = -h; s = h; break;
        default: c = -c1; s = s1; break;
    }
    // forward: (c - i s); inverse: (c + i s)
    return INV ? make_float2(d.x * c - d.y * s, d.y * c + d.x * s) : make_float2(d.x * c + d.y * s, d.y * c - d.x * s);
}

__host__ __device__ constexpr int bitrev(int i, int R)
{
    int r = 0;
    for (int b = 1; b < R; b <<= 1) { r = (r << 1) | (i & 1); i >>= 1; }
    return r;
}

// in place; natural order in, v[i] = X[bitrev(i)] out
template <int R, bool INV>
__device__ __forceinline__ void reg_dft(float2 (&v)[R])
{
#pragma unroll
    for (int len = R; len >= 2; len >>= 1) {
        const int half = len >> 1;
#pragma unroll
        for (int b = 0; b < R; b += len) {
#pragma unroll
            for (int j = 0; j < half; j++) {
                const float2 a = v[b + j], c = v[b + j + half];
                v[b + j] = cadd(a, c);
                v[b + j + half] = mul_w16<INV>(csub(a, c), j * (16 / len));
            }
        }
    }
}

constexpr int FFT_T = 256;  // threads per CTA of every FFT kernel

// radix of the stage that works on spans of length L (a power of two): 16 where possible, but 8 when that would leave a
// radix-2 stage at the end (L = 32, 512, ...: 32 = 8 x 4, 512 = 8 x 16 x 4); the host mirror uses the same function
__host__ __device__ constexpr int stage_radix(int L)
{
    int lg = 0;
    for (int v = L; v > 1; v >>= 1) lg++;
    return L >= 16 ? (lg % 4 == 1 ? 8 : 16) : L;
}

// ---- bank-conflict-free rows of 8 columns ------------------------------------------------------------------
// A tile row of 8 float2 columns (64 bytes) covers half of the 32 banks: even rows one half, odd rows the other.  The
// stages whose butterflies sit 4 rows apart (the last radix-4 stage; the stage of span 64 of the 512 / 1024 plans) then
// find all rows of a warp request in the same half (ncu: 25-32 % of the shared-memory wavefronts of the y and x passes
// at 512 were bank conflicts).  Rows are therefore stored at row ^ bit 2 of the row: consecutive rows still alternate
// halves, and so do rows 4 apart.  Tiles of 16 columns (128-byte rows) and the padded z tiles need none of this.
template <bool SWZ>
__device__ __forceinline__ int trow(int pos) { return SWZ ? pos ^ ((pos >> 2) & 1) : pos; }

// ---- one transform along the tile's position axis, everything but the data known at compile time -----------
// tile [N][PITCH] (float2), columns [0, ncol) of 1 << CS; tw = exp(-2 pi i k / N), k < N (shared memory).
// Stage of span L, radix R = stage_radix(L): butterfly (blk, j) takes positions blk L + j + m L/R, m < R.
struct NoOut {
    __device__ __forceinline__ void operator()(int, int, float2) const {}
};
// OUT = NoOut: the stage works in place on the tile.  Any other OUT receives the results instead -- out(position, column,
// value) -- so that the LAST stage of a transform can hand them straight to global memory (no store to the tile, no
// barrier, no copy-out pass).
struct NoIn {
    __device__ __forceinline__ float2 operator()(int, int) const { return make_float2(0.f, 0.f); }
};
// IN = NoIn: the stage reads the tile.  Any other IN supplies the inputs instead -- in(position, column) -- so that the
// FIRST stage of a transform can take them from where they already are (the z pass: the row-major staging area).
template <int N, int L, bool INV, int PITCH, int CS, class OUT, class IN = NoIn>
__device__ __forceinline__ void fft_stage_impl(float2 *tile, int ncol, const float2 *tw, const OUT &out, const IN &in = IN())
{
    constexpr bool FROM_TILE = std::is_same<IN, NoIn>::value;
    constexpr int R = stage_radix(L);
    constexpr int Lr = L / R, twstep = N / L;
    constexpr int nwork = (N / R) << CS;
    constexpr bool SWZ = CS == 3 && PITCH == 8;      // rows of 8 unpadded columns: see trow()
    constexpr bool SAME = !SWZ || Lr % 8 == 0;        // every element of a butterfly gets the same row swizzle
    constexpr bool TO_TILE = std::is_same<OUT, NoOut>::value;
#pragma unroll 1
    for (int wk = threadIdx.x; wk < nwork; wk += FFT_T) {
        const int col = wk & ((1 << CS) - 1);
        if (col >= ncol) continue;
        const int bf = wk >> CS;
        const int blk = bf / Lr, j = bf - blk * Lr;
        const int base = blk * L + j;
        float2 *p = tile + (SAME ? trow<SWZ>(base) : base) * PITCH + col;
        float2 v[R];
#pragma unroll
        for (int m = 0; m < R; m++)
            v[m] = !FROM_TILE ? in(base + m * Lr, col) : (SAME ? p[m * Lr * PITCH] : tile[trow<SWZ>(base + m * Lr) * PITCH + col]);
        if (INV && Lr > 1) {
#pragma unroll
            for (int q = 1; q < R; q++) v[q] = cmulc(v[q], tw[j * q * twstep]);
        }
        reg_dft<R, INV>(v);
#pragma unroll
        for (int i = 0; i < R; i++) {
            const int q = bitrev(i, R);
            float2 o = v[i];
            if (!INV && Lr > 1 && q != 0) o = cmul(o, tw[j * q * twstep]);
            if (!TO_TILE) out(base + q * Lr, col, o);
            else if (SAME) p[q * Lr * PITCH] = o;
            else tile[trow<SWZ>(base + q * Lr) * PITCH + col] = o;
        }
    }
}
template <int N, int L, bool INV, int PITCH, int CS>
__device__ __forceinline__ void fft_stage(float2 *tile, int ncol, const float2 *tw)
{
    fft_stage_impl<N, L, INV, PITCH, CS, NoOut>(tile, ncol, tw, NoOut());
}

template <int N, int L, bool INV, int PITCH, int CS>
struct AxisFFT {
    static constexpr int R = stage_radix(L);
    static __device__ __forceinline__ void run(float2 *tile, int ncol, const float2 *tw)
    {
        if (!INV) {
            fft_stage<N, L, false, PITCH, CS>(tile, ncol, tw);
            __syncthreads();
            AxisFFT<N, L / R, INV, PITCH, CS>::run(tile, ncol, tw);
        } else {
            AxisFFT<N, L / R, INV, PITCH, CS>::run(tile, ncol, tw);
            fft_stage<N, L, true, PITCH, CS>(tile, ncol, tw);
            __syncthreads();
        }
    }
};
template <int N, bool INV, int PITCH, int CS>
struct AxisFFT<N, 1, INV, PITCH, CS> {
    static __device__ __forceinline__ void run(float2 *, int, const float2 *) {}
};

// host mirror of the stage sequence (for the position <-> frequency tables)
struct AxisPlan {
    int N;
    int nst;
    int radix[4];
    int span[4];
};

// ---- device-side description of the mesh in k-space layout --------------------------------------------------
struct FftGeom {
    int N[3];
    int zsc;             // complex elements per z-row in memory (zs / 2); columns [0, zsc) are moved, Nz/2 + 1 are meaningful
    long long cstride;   // complex elements per mesh
    const float2 *twx, *twy, *twz;   // exp(-2 pi i k / N) for N = Nx, Ny, Nz/2
    const float2 *twzr;  // exp(-2 pi i k / Nz), k = 0 .. Nz/2: real <-> half-complex post-processing
    const int *posz;     // position of frequency k after the forward stages of the Nz/2-point transform
    const double *ktab;  // [3 axes][3: kt, k^2, dec][tabn] in MEMORY order (x, y digit-reversed, z natural)
    int tabn;
    double c0;           // 3/2 Om / (nbar N_g)
};


__device__ __forceinline__ void fft_cp_async16(void *dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"((unsigned long long)src) : "memory");
}
__device__ __forceinline__ void fft_cp_async_wait_all() { asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory"); }

// global -> tile [N][1 << CS]: element (pos, col) from base[pos * stride + col]; 16-byte async copies (column pairs;
// ncol is even: 16, 8 or the 2 columns of the last tile)
template <int N, int CS>
__device__ __forceinline__ void tile_load(float2 *tile, const float2 *base, long long stride, int ncol)
{
    constexpr int HB = 1 << (CS - 1);  // column pairs per position
    const int cp = threadIdx.x & (HB - 1);
    if (2 * cp < ncol) {
#pragma unroll 4
        for (int pos = threadIdx.x >> (CS - 1); pos < N; pos += FFT_T >> (CS - 1))
            fft_cp_async16(tile + (trow<CS == 3>(pos) << CS) + 2 * cp, base + (size_t)pos * stride + 2 * cp);
    }
}
template <int N, int CS>
__device__ __forceinline__ void tile_store(const float2 *tile, float2 *base, long long stride, int ncol)
{
    constexpr int HB = 1 << (CS - 1);
    const int cp = threadIdx.x & (HB - 1);
    if (2 * cp < ncol) {
#pragma unroll 4
        for (int pos = threadIdx.x >> (CS - 1); pos < N; pos += FFT_T >> (CS - 1))
            *reinterpret_cast<float4 *>(base + (size_t)pos * stride + 2 * cp) = *reinterpret_cast<const float4 *>(tile + (trow<CS == 3>(pos) << CS) + 2 * cp);
    }
}
__device__ __forceinline__ void load_tw(float2 *dst, const float2 *src, int n)
{
    for (int i = threadIdx.x; i < n; i += FFT_T) dst[i] = src[i];
}

// ---- y pass: in-place transform along y of nb meshes ---------------------------------------------------------
// grid = (column tiles along z, Nx, nb); dynamic shared memory: tile [Ny][1 << CS] + Ny twiddles
__host__ __device__ constexpr int last_span(int N)
{
    int L = N;
    while (stage_radix(L) != L) L /= stage_radix(L);
    return L;
}

// the stages with span > LSTOP only (forward: descending spans, inverse: ascending); every stage is followed by a barrier
template <int N, int L, bool INV, int PITCH, int CS, int LSTOP>
struct AxisFFTPartial {
    static constexpr int R = stage_radix(L);
    static __device__ __forceinline__ void run(float2 *tile, int ncol, const float2 *tw)
    {
        if (!INV) {
            fft_stage<N, L, false, PITCH, CS>(tile, ncol, tw);
            __syncthreads();
            AxisFFTPartial<N, L / R, INV, PITCH, CS, LSTOP>::run(tile, ncol, tw);
        } else {
            AxisFFTPartial<N, L / R, INV, PITCH, CS, LSTOP>::run(tile, ncol, tw);
            fft_stage<N, L, true, PITCH, CS>(tile, ncol, tw);
            __syncthreads();
        }
    }
};
template <int N, int LS, bool INV, int PITCH, int CS>
struct AxisFFTPartial<N, LS, INV, PITCH, CS, LS> {
    static __device__ __forceinline__ void run(float2 *, int, const float2 *) {}
};

// result (position, column) -> base[position * stride + column]
struct StoreOut {
    float2 *base;
    long long stride;
    __device__ __forceinline__ void operator()(int pos, int col, float2 v) const { base[(size_t)pos * stride + col] = v; }
};

template <int NY, int CS, bool INV>
__global__ void __launch_bounds__(FFT_T) fft_y_kernel(FftGeom g, float2 *data)
{
    extern __shared__ __align__(16) unsigned char fsm[];
    pdl_trigger();  // the constant tables are loaded before pdl_wait(), the data after it
    float2 *tile = reinterpret_cast<float2 *>(fsm);
    float2 *tw = tile + (NY << CS);
    constexpr int B = 1 << CS;
    const int col0 = blockIdx.x * B, ncol = min(B, g.zsc - col0);
    float2 *base = data + (size_t)blockIdx.z * g.cstride + (size_t)blockIdx.y * NY * g.zsc + col0;
    load_tw(tw, g.twy, NY);
    pdl_wait();
    tile_load<NY, CS>(tile, base, g.zsc, ncol);
    fft_cp_async_wait_all();
    __syncthreads();
    // the last stage writes its results straight to global memory (the CTA has read all of its columns by now)
    const StoreOut out = {base, g.zsc};
    if (!INV) {
        constexpr int RL = last_span(NY);
        AxisFFTPartial<NY, NY, false, B, CS, RL>::run(tile, ncol, tw);
        fft_stage_impl<NY, RL, false, B, CS>(tile, ncol, tw, out);
    } else {
        AxisFFTPartial<NY, NY / stage_radix(NY), true, B, CS, 1>::run(tile, ncol, tw);
        fft_stage_impl<NY, NY, true, B, CS>(tile, ncol, tw, out);
    }
}

// G(k) = c0 dec / k^2 of one mode, fp64 rounded to fp32 once; G(0) = 0 (R9).  The x-dependent table entries come from
// shared memory, the (y, z)-dependent parts are per-thread constants; the division is a reciprocal seed refined by one
// Newton step in fp64 (relative error ~1e-14, far below the final rounding to fp32).
struct GreenCol {
    double k2yz, decyz, c0;
};
__device__ __forceinline__ GreenCol green_col(const FftGeom &g, int iy, int iz)
{
    const double *ty = g.ktab + 3 * g.tabn, *tz = g.ktab + 6 * g.tabn;
    GreenCol c;
    c.k2yz = ty[g.tabn + iy] + tz[g.tabn + iz];
    c.decyz = ty[2 * g.tabn + iy] * tz[2 * g.tabn + iz];
    c.c0 = g.c0;
    return c;
}
__device__ __forceinline__ float mode_green(const GreenCol &c, double k2x, double decx)
{
    const double k2 = k2x + c.k2yz;
    if (!(k2 > 0.0)) return 0.f;
    double r = (double)__frcp_rn((float)k2);
    r = r * (2.0 - k2 * r);
    return (float)(c.c0 * (decx * c.decyz) * r);
}

// ---- the fused x kernels: transform along x, k-space operator, back-transform, ONE shared-memory tile ---------------
// The last forward stage (span RL = its radix, butterflies over RL neighbouring positions) and the first inverse stage
// work on the same groups of positions, so a thread keeps the outputs of its last-stage butterflies in REGISTERS, applies
// the operator there and feeds them straight into the first inverse stage(s): the spectrum never goes back to shared
// memory, and the two back-transforms of the force kernel (f_x, and the common part of f_y, f_z) run one after the other
// through the same tile.  Half the shared memory of a two-tile design: 8 columns (64-byte pieces) at Nx = 1024 with two
// CTAs per SM, four CTAs per SM at 512.
template <int NX, int CS>
struct XPlan {
    static constexpr int B = 1 << CS;
    static constexpr int RL = last_span(NX);               // span and radix of the last forward / first inverse stage
    static constexpr int NWORK = (NX / RL) << CS;          // its butterflies per tile
    static constexpr int IT = (NWORK + FFT_T - 1) / FFT_T; // butterflies per thread: IT * RL spectrum elements in registers
    // butterfly `it` of this thread: column and first position; false = none (short tile or column beyond ncol)
    static __device__ __forceinline__ bool item(int it, int ncol, int &col, int &pos0)
    {
        const int wk = threadIdx.x + it * FFT_T;
        col = wk & (B - 1);
        pos0 = (wk >> CS) * RL;
        return wk < NWORK && col < ncol;
    }
    // last forward stage: X[pos0 + m] of the column, m < RL, in natural order
    static __device__ __forceinline__ void last_fwd(const float2 *tile, int col, int pos0, float2 (&x)[RL])
    {
        float2 v[RL];
#pragma unroll
        for (int m = 0; m < RL; m++) v[m] = tile[(trow<CS == 3>(pos0 + m) << CS) + col];
        reg_dft<RL, false>(v);
#pragma unroll
        for (int m = 0; m < RL; m++) x[m] = v[bitrev(m, RL)];
    }
    // first inverse stage: takes the RL spectrum elements, leaves its outputs in the tile for the remaining stages
    // (when the whole transform is this one stage, NX == RL, the outputs are final and go to `out` instead)
    template <class OUT>
    static __device__ __forceinline__ void first_inv(float2 *tile, int col, int pos0, float2 (&v)[RL], const OUT &out)
    {
        reg_dft<RL, true>(v);
#pragma unroll
        for (int i = 0; i < RL; i++) {
            if (NX == RL) out(pos0 + bitrev(i, RL), col, v[i]);
            else tile[(trow<CS == 3>(pos0 + bitrev(i, RL)) << CS) + col] = v[i];
        }
    }
    // the inverse stages after the first one; the last of them hands its results to `out`
    template <class OUT>
    static __device__ __forceinline__ void inv_rest(float2 *tile, int ncol, const float2 *tw, const OUT &out)
    {
        if (NX != RL) {
            __syncthreads();
            AxisFFTPartial<NX, NX / stage_radix(NX), true, B, CS, (NX != RL ? RL : 1)>::run(tile, ncol, tw);
            fft_stage_impl<NX, NX, true, B, CS>(tile, ncol, tw, out);
        }
    }
};

#define PM_X_MINBLOCKS(NX, CS) ((NX) >= 1024 ? 2 : ((NX) >= 512 ? ((CS) == 4 ? 2 : 3) : 2))

// T(position, column) -> f_y = i kt_y T and f_z = i kt_z T (kt_z of the thread's own column: a thread only ever sees one)
struct StoreYZ {
    float2 *fy;
    long long stride, cstride;
    float kty, ktz;
    __device__ __forceinline__ void operator()(int pos, int col, float2 t) const
    {
        float2 *dst = fy + (size_t)pos * stride + col;
        dst[0] = make_float2(-kty * t.y, kty * t.x);
        dst[cstride] = make_float2(-ktz * t.y, ktz * t.x);
    }
};

// ---- x pass fused with the force operator: rho(k) -> f_d(k) = i kt_d G rho(k), d = 1..3, back-transformed along x ----
// grid = (column tiles along z, Ny); shared: one tile + Nx twiddles + the x-dependent k tables
template <int NX, int CS>
__global__ void __launch_bounds__(FFT_T, PM_X_MINBLOCKS(NX, CS)) fft_x_force_kernel(FftGeom g, const float2 *rho, float2 *f)
{
    typedef XPlan<NX, CS> P;
    constexpr int B = P::B, RL = P::RL, IT = P::IT;
    extern __shared__ __align__(16) unsigned char fsm[];
    pdl_trigger();  // the constant tables are loaded before pdl_wait(), the data after it
    float2 *tile = reinterpret_cast<float2 *>(fsm);
    float2 *tw = tile + (NX << CS);
    double *k2x = reinterpret_cast<double *>(tw + NX), *decx = k2x + NX;
    float *ktx = reinterpret_cast<float *>(decx + NX);
    const int col0 = blockIdx.x * B, ncol = min(B, g.zsc - col0);
    const int iy = blockIdx.y;
    const long long stride = (long long)g.N[1] * g.zsc;
    const size_t off = (size_t)iy * g.zsc + col0;
    load_tw(tw, g.twx, NX);
    for (int i = threadIdx.x; i < NX; i += FFT_T) {
        ktx[i] = (float)g.ktab[i];
        k2x[i] = g.ktab[g.tabn + i];
        decx[i] = g.ktab[2 * g.tabn + i];
    }
    pdl_wait();
    tile_load<NX, CS>(tile, rho + off, stride, ncol);
    fft_cp_async_wait_all();
    __syncthreads();
    AxisFFTPartial<NX, NX, false, B, CS, RL>::run(tile, ncol, tw);
    // last forward stage and Green's function (fp64, rounded once) in registers: h = G rho(k)
    float2 h[IT][RL];
    const float kty = (float)g.ktab[3 * g.tabn + iy];
    {
        const int colt = threadIdx.x & (B - 1);  // the column of all butterflies of this thread (FFT_T is a multiple of B)
        const GreenCol gc = green_col(g, iy, min(col0 + colt, g.N[2] / 2));
#pragma unroll
        for (int it = 0; it < IT; it++) {
            int col, pos0;
            if (!P::item(it, ncol, col, pos0)) continue;
            P::last_fwd(tile, col, pos0, h[it]);
#pragma unroll
            for (int m = 0; m < RL; m++) {
                const float G = mode_green(gc, k2x[pos0 + m], decx[pos0 + m]);
                h[it][m] = make_float2(G * h[it][m].x, G * h[it][m].y);
            }
        }
    }
    const StoreOut out_x = {f + off, stride};
    const StoreYZ out_yz = {f + g.cstride + off, stride, g.cstride, kty, (float)g.ktab[6 * g.tabn + min(col0 + (int)(threadIdx.x & (B - 1)), g.N[2] / 2)]};
    // f_x: back-transform of i kt_x h (a thread rewrites only the tile elements it has just read: no barrier before)
#pragma unroll
    for (int it = 0; it < IT; it++) {
        int col, pos0;
        if (!P::item(it, ncol, col, pos0)) continue;
        float2 v[RL];
#pragma unroll
        for (int m = 0; m < RL; m++) {
            const float c = ktx[pos0 + m];
            v[m] = make_float2(-c * h[it][m].y, c * h[it][m].x);
        }
        P::first_inv(tile, col, pos0, v, out_x);
    }
    P::inv_rest(tile, ncol, tw, out_x);   // the last stage stores f_x
    __syncthreads();
    // kt_y and kt_z do not depend on x, so ONE back-transform T of h serves f_y = i kt_y T and f_z = i kt_z T
#pragma unroll
    for (int it = 0; it < IT; it++) {
        int col, pos0;
        if (!P::item(it, ncol, col, pos0)) continue;
        P::first_inv(tile, col, pos0, h[it], out_yz);
    }
    P::inv_rest(tile, ncol, tw, out_yz);  // the last stage stores f_y and f_z
}

// ---- x pass fused with the adjoint operator: psi(k) = -i G sum_d kt_d Pi_d(k), back-transformed along x ----------
template <int NX, int CS>
__global__ void __launch_bounds__(FFT_T, PM_X_MINBLOCKS(NX, CS)) fft_x_adjoint_kernel(FftGeom g, const float2 *Pi, float2 *psi)
{
    typedef XPlan<NX, CS> P;
    constexpr int B = P::B, RL = P::RL, IT = P::IT;
    extern __shared__ __align__(16) unsigned char fsm[];
    pdl_trigger();  // the constant tables are loaded before pdl_wait(), the data after it
    float2 *tile = reinterpret_cast<float2 *>(fsm);
    float2 *tw = tile + (NX << CS);
    double *k2x = reinterpret_cast<double *>(tw + NX), *decx = k2x + NX;
    float *ktx = reinterpret_cast<float *>(decx + NX);
    const int col0 = blockIdx.x * B, ncol = min(B, g.zsc - col0);
    const int iy = blockIdx.y;
    const long long stride = (long long)g.N[1] * g.zsc;
    const size_t off = (size_t)iy * g.zsc + col0;
    const float kty = (float)g.ktab[3 * g.tabn + iy];
    load_tw(tw, g.twx, NX);
    for (int i = threadIdx.x; i < NX; i += FFT_T) {
        ktx[i] = (float)g.ktab[i];
        k2x[i] = g.ktab[g.tabn + i];
        decx[i] = g.ktab[2 * g.tabn + i];
    }
    pdl_wait();
    // Pi_x: transform along x, spectrum kept in registers
    tile_load<NX, CS>(tile, Pi + off, stride, ncol);
    fft_cp_async_wait_all();
    __syncthreads();
    AxisFFTPartial<NX, NX, false, B, CS, RL>::run(tile, ncol, tw);
    float2 hx[IT][RL];
#pragma unroll
    for (int it = 0; it < IT; it++) {
        int col, pos0;
        if (!P::item(it, ncol, col, pos0)) continue;
        P::last_fwd(tile, col, pos0, hx[it]);
    }
    __syncthreads();  // the tile is refilled by other threads
    // kt_y and kt_z do not depend on x: kt_y Pi_y + kt_z Pi_z is formed BEFORE the transform along x, so two forward
    // transforms (Pi_x and that sum) instead of three
    {
        constexpr int HB = 1 << (CS - 1);
        const int cp = threadIdx.x & (HB - 1);
        if (2 * cp < ncol) {
            const float kz0 = (float)g.ktab[6 * g.tabn + min(col0 + 2 * cp, g.N[2] / 2)];
            const float kz1 = (float)g.ktab[6 * g.tabn + min(col0 + 2 * cp + 1, g.N[2] / 2)];
            const float2 *py = Pi + g.cstride + off + 2 * cp, *pz = py + g.cstride;
#pragma unroll 4
            for (int pos = threadIdx.x >> (CS - 1); pos < NX; pos += FFT_T >> (CS - 1)) {
                const float4 a = __ldg(reinterpret_cast<const float4 *>(py + (size_t)pos * stride));
                const float4 b = __ldg(reinterpret_cast<const float4 *>(pz + (size_t)pos * stride));
                *reinterpret_cast<float4 *>(tile + (trow<CS == 3>(pos) << CS) + 2 * cp) =
                    make_float4(kty * a.x + kz0 * b.x, kty * a.y + kz0 * b.y, kty * a.z + kz1 * b.z, kty * a.w + kz1 * b.w);
            }
        }
    }
    __syncthreads();
    AxisFFTPartial<NX, NX, false, B, CS, RL>::run(tile, ncol, tw);
    const StoreOut out_psi = {psi + off, stride};
    {
        const int colt = threadIdx.x & (B - 1);
        const GreenCol gc = green_col(g, iy, min(col0 + colt, g.N[2] / 2));
#pragma unroll
        for (int it = 0; it < IT; it++) {
            int col, pos0;
            if (!P::item(it, ncol, col, pos0)) continue;
            float2 a[RL];
            P::last_fwd(tile, col, pos0, a);
#pragma unroll
            for (int m = 0; m < RL; m++) {
                const float c = ktx[pos0 + m];
                const float G = mode_green(gc, k2x[pos0 + m], decx[pos0 + m]);
                const float2 v = hx[it][m];
                // times -i G: (re, im) -> (G im, -G re)
                a[m] = make_float2(G * (c * v.y + a[m].y), -G * (c * v.x + a[m].x));
            }
            P::first_inv(tile, col, pos0, a, out_psi);
        }
    }
    P::inv_rest(tile, ncol, tw, out_psi);  // the last stage stores psi
}

// result (position, row) of the z pass into the row-major staging area [row][pitch]
struct StoreOutRow {
    float2 *base;
    int pitch;
    __device__ __forceinline__ void operator()(int pos, int row, float2 v) const { base[row * pitch + pos] = v; }
};
// input (position, row) of the z pass from the row-major staging area [row][pitch]
struct StageIn {
    const float2 *base;
    int pitch;
    __device__ __forceinline__ float2 operator()(int pos, int row) const { return base[row * pitch + pos]; }
};

// ---- z pass, real -> half-complex, in place on ZROWS consecutive z-rows per CTA ---------------------------------
// row = [zs floats] -> [zsc complex]; x_n real, n < Nz = 2M: z_n = x_2n + i x_2n+1, Z = FFT_M(z),
// E_k = (Z_k + conj Z_{M-k}) / 2, O_k = (Z_k - conj Z_{M-k}) / (2i), X_k = E_k + w^k O_k, w = e^{-2 pi i / Nz}, k = 0..M
// shared: tile [M][ZP] + out [M + 1][ZP] + M twiddles + (M + 1) post twiddles + M positions
template <int M, int ZRS>
__global__ void __launch_bounds__(FFT_T) fft_z_r2c_kernel(FftGeom g, float *data, long long nrows)
{
    constexpr int ZROWS = 1 << ZRS, ZP = ZROWS + 1;  // z-rows per CTA; padded pitch of the transposing buffer
    constexpr int TP = ZRS == 3 ? 8 : ZP;            // tile pitch: 8 rows are kept unpadded and swizzled instead (trow)
#define ZT(pos) (trow<ZRS == 3>(pos) * TP)
    extern __shared__ __align__(16) unsigned char fsm[];
    pdl_trigger();  // the constant tables are loaded before pdl_wait(), the data after it
    float2 *tile = reinterpret_cast<float2 *>(fsm);
    float2 *outb = tile + M * TP;
    float2 *tw = outb + max((M + 1) * ZP, ZROWS * g.zsc);
    float2 *twr = tw + M;
    int *posz = reinterpret_cast<int *>(twr + (M + 1));
    const int zs = 2 * g.zsc;
    const long long row0 = (long long)blockIdx.x * ZROWS;
    const int nr = (int)min((long long)ZROWS, nrows - row0);
    float *rows = data + (size_t)row0 * zs;
    // the nr rows are contiguous in memory: 16-byte async copies into a row-major staging area (which shares its
    // shared memory with outb), then the transposing fill of the tile
    float *stage = reinterpret_cast<float *>(outb);
    load_tw(tw, g.twz, M);
    load_tw(twr, g.twzr, M + 1);
    for (int i = threadIdx.x; i < M; i += FFT_T) posz[i] = g.posz[i];
    pdl_wait();
    {
        const int nchunk = nr * (zs / 4);
        for (int i = threadIdx.x; i < nchunk; i += FFT_T) fft_cp_async16(stage + 4 * i, rows + 4 * (size_t)i);
    }
    fft_cp_async_wait_all();
    __syncthreads();
    // z_n = x_2n + i x_2n+1 is element n of the staged row: the first stage reads it there (no transposing fill pass)
    {
        const StageIn sin = {reinterpret_cast<const float2 *>(stage), M + 2};
        fft_stage_impl<M, M, false, TP, ZRS, NoOut, StageIn>(tile, nr, tw, NoOut(), sin);
        __syncthreads();
        AxisFFTPartial<M, M / stage_radix(M), false, TP, ZRS, 1>::run(tile, nr, tw);
    }

    {
        const int r = threadIdx.x & (ZROWS - 1);
        if (r < nr) {
#pragma unroll 4
            // one thread per PAIR (k, M - k): X_k = E + w^k O and X_{M-k} = conj(E - w^k O) from one read of Z_k, Z_{M-k}
            // and one twiddle (half the shared-memory reads of a loop over all k)
            for (int k = threadIdx.x >> ZRS; k <= M / 2; k += FFT_T >> ZRS) {
                const float2 a = tile[ZT(posz[k]) + r];
                if (k == 0) {
                    outb[r] = make_float2(a.x + a.y, 0.f);               // X_0
                    outb[M * ZP + r] = make_float2(a.x - a.y, 0.f);      // X_M (Nyquist)
                } else {
                    const float2 b = tile[ZT(posz[M - k]) + r];
                    const float2 E = make_float2(0.5f * (a.x + b.x), 0.5f * (a.y - b.y));
                    const float2 O = make_float2(0.5f * (a.y + b.y), -0.5f * (a.x - b.x));  // (a - conj b) / (2i)
                    const float2 t = cmul(twr[k], O);
                    outb[k * ZP + r] = cadd(E, t);
                    const float2 d = csub(E, t);
                    if (2 * k != M) outb[(M - k) * ZP + r] = make_float2(d.x, -d.y);
                }
            }
        }
    }
    __syncthreads();
    float2 *crow = reinterpret_cast<float2 *>(rows);
    for (int r = threadIdx.x / 64; r < nr; r += FFT_T / 64)
        for (int k = threadIdx.x & 63; k < M + 2; k += 64) crow[r * (M + 2) + k] = k <= M ? outb[k * ZP + r] : make_float2(0.f, 0.f);  // zsc = M + 2
}

// ---- z pass, half-complex -> real (unnormalised: Nz times the inverse), in place ------------------------------
// E_k = X_k + conj X_{M-k}, O_k = (X_k - conj X_{M-k}) conj(w^k), Z_k = E_k + i O_k (twice the textbook Z: the
// M-point inverse then yields Nz * x), z = IFFT_M(Z), x_2n = Re z_n, x_2n+1 = Im z_n
template <int M, int ZRS>
__global__ void __launch_bounds__(FFT_T) fft_z_c2r_kernel(FftGeom g, float *data, long long nrows)
{
    constexpr int ZROWS = 1 << ZRS, ZP = ZROWS + 1;  // z-rows per CTA; padded pitch of the transposing buffer
    constexpr int TP = ZRS == 3 ? 8 : ZP;            // tile pitch: 8 rows are kept unpadded and swizzled instead (trow)
#define ZT(pos) (trow<ZRS == 3>(pos) * TP)
    extern __shared__ __align__(16) unsigned char fsm[];
    pdl_trigger();  // the constant tables are loaded before pdl_wait(), the data after it
    float2 *tile = reinterpret_cast<float2 *>(fsm);
    float2 *inb = tile + M * TP;
    float2 *tw = inb + max((M + 1) * ZP, ZROWS * g.zsc);
    float2 *twr = tw + M;
    int *posz = reinterpret_cast<int *>(twr + (M + 1));
    const int zs = 2 * g.zsc;
    const long long row0 = (long long)blockIdx.x * ZROWS;
    const int nr = (int)min((long long)ZROWS, nrows - row0);
    float *rows = data + (size_t)row0 * zs;
    load_tw(tw, g.twz, M);
    load_tw(twr, g.twzr, M + 1);
    for (int i = threadIdx.x; i < M; i += FFT_T) posz[i] = g.posz[i];
    pdl_wait();
    {   // the nr rows are contiguous in memory: 16-byte async copies, row-major [row][zsc]
        const int nchunk = nr * (zs / 4);
        for (int i = threadIdx.x; i < nchunk; i += FFT_T) fft_cp_async16(reinterpret_cast<float *>(inb) + 4 * i, rows + 4 * (size_t)i);
    }
    fft_cp_async_wait_all();
    __syncthreads();
    {
        const int r = threadIdx.x & (ZROWS - 1);
        if (r < nr) {
#pragma unroll 4
            // one thread per PAIR (k, M - k): Z_k = E + i O and Z_{M-k} = conj(E - i O) from one read of X_k, X_{M-k}
            for (int k = threadIdx.x >> ZRS; k <= M / 2; k += FFT_T >> ZRS) {
                const float2 a = inb[r * (M + 2) + k], b = inb[r * (M + 2) + M - k];
                const float2 E = make_float2(a.x + b.x, a.y - b.y);
                const float2 O = cmulc(make_float2(a.x - b.x, a.y + b.y), twr[k]);
                tile[ZT(posz[k]) + r] = make_float2(E.x - O.y, E.y + O.x);  // E + i O
                if (k != 0 && 2 * k != M) tile[ZT(posz[M - k]) + r] = make_float2(E.x + O.y, O.x - E.y);
            }
        }
    }
    __syncthreads();
    if (ZRS == 3) {
        // 8 unpadded rows: reading the tile along n for the row-wise store would put every lane on two banks.  The last
        // stage hands its results to the (free again) row-major staging area instead, and the rows leave from there.
        AxisFFTPartial<M, M / stage_radix(M), true, TP, ZRS, 1>::run(tile, nr, tw);
        float2 *stage2 = inb;
        const StoreOutRow so = {stage2, M + 2};
        fft_stage_impl<M, M, true, TP, ZRS>(tile, nr, tw, so);
        __syncthreads();
        float2 *rows2 = reinterpret_cast<float2 *>(rows);
        for (int idx = threadIdx.x; idx < nr * (M / 2); idx += FFT_T) {
            const int r = idx / (M / 2), c = idx - r * (M / 2);
            *reinterpret_cast<float4 *>(rows2 + (size_t)r * (M + 2) + 2 * c) = *reinterpret_cast<const float4 *>(stage2 + r * (M + 2) + 2 * c);
        }
        return;
    }
    AxisFFT<M, M, true, TP, ZRS>::run(tile, nr, tw);
    if (M <= FFT_T) {
        constexpr int RPP = FFT_T / M > 0 ? FFT_T / M : 1;
        const int n = threadIdx.x % M, r0 = threadIdx.x / M;
#pragma unroll 4
        for (int r = r0; r < nr; r += RPP) *reinterpret_cast<float2 *>(rows + r * (2 * M + 4) + 2 * n) = tile[ZT(n) + r];  // zs = 2 M + 4
    } else {
        for (int r = 0; r < nr; r++)
            for (int n = threadIdx.x; n < M; n += FFT_T) *reinterpret_cast<float2 *>(rows + (size_t)r * zs + 2 * n) = tile[ZT(n) + r];
    }
}
#undef ZT

// ---- host ------------------------------------------------------------------------------------------------------
static bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

static AxisPlan make_axis_plan(int N)
{
    AxisPlan p;
    p.N = N;
    p.nst = 0;
    int n = N;
    while (n > 1) {
        int r = stage_radix(n);
        p.radix[p.nst] = r;
        p.span[p.nst] = n;
        p.nst++;
        n /= r;
    }
    return p;
}

// frequency held at memory position pos after the forward stages of the plan
static int freq_of_pos(const AxisPlan &p, int pos)
{
    int k = 0, mul = 1, L = p.N;
    for (int s = 0; s < p.nst; s++) {
        int Lr = L / p.radix[s];
        int q = pos / Lr;
        k += q * mul;
        mul *= p.radix[s];
        pos -= q * Lr;
        L = Lr;
    }
    return k;
}

bool fft_own_supported(const Geometry &g)
{
    const char *e = getenv("PM_FFT");
    if (e && strcmp(e, "cufft") == 0) return false;
    // powers of two from 16 to 1024 per axis (at 1024^3 the own passes take 9.2 s of a configs[3] run, cuFFT 10.6 s)
    for (int d = 0; d < 3; d++)
        if (!is_pow2(g.N[d]) || g.N[d] < 16 || g.N[d] > 1024) return false;
    return true;
}

size_t fft_own_table_bytes(const Geometry &g)
{
    return sizeof(float2) * (size_t)(g.N[0] + g.N[1] + g.N[2] + 16) + sizeof(int) * (size_t)g.N[2] + 1024;
}

// memory order of an axis in k-space: the frequency index (0..N-1, cuFFT order) stored at each position
void fft_own_axis_order(const pm_ctx *c, int axis, std::vector<int> &freq)
{
    const int N = c->g.N[axis];
    freq.resize(N);
    if (!c->own_fft || axis == 2) {
        for (int i = 0; i < N; i++) freq[i] = i;
    } else {
        AxisPlan p = make_axis_plan(N);
        for (int i = 0; i < N; i++) freq[i] = freq_of_pos(p, i);
    }
}

// host-only view of the same table for the ABI (include/pm.h: pm_host_fft_order)
int fft_own_order_host(int n, int *out)
{
    if (!out || !is_pow2(n) || n < 8 || n > 1024) return PM_EINVAL;
    AxisPlan p = make_axis_plan(n);
    for (int i = 0; i < n; i++) out[i] = freq_of_pos(p, i);
    return PM_OK;
}

static FftGeom *geom_of(pm_ctx *c) { return reinterpret_cast<FftGeom *>(c->fft_geom); }

int fft_own_init(pm_ctx *c)
{
    static_assert(sizeof(FftGeom) <= sizeof(c->fft_geom), "fft_geom storage too small");
    const Geometry &g = c->g;
    c->own_fft = fft_own_supported(g);
    if (!c->own_fft) return PM_OK;
    FftGeom *fg = geom_of(c);
    const int M = g.N[2] / 2;
    for (int d = 0; d < 3; d++) fg->N[d] = g.N[d];
    fg->zsc = g.zs / 2;
    fg->cstride = g.mesh_stride / 2;
    const AxisPlan pz = make_axis_plan(M);
    const double PI = 3.14159265358979323846264338327950288;
    std::vector<float2> h;
    auto push_tw = [&](int N, int count) {
        size_t o = h.size();
        for (int k = 0; k < count; k++) {
            double a = -2.0 * PI * (double)k / (double)N;
            h.push_back(make_float2((float)std::cos(a), (float)std::sin(a)));
        }
        return o;
    };
    size_t ox = push_tw(g.N[0], g.N[0]), oy = push_tw(g.N[1], g.N[1]), oz = push_tw(M, M), ozr = push_tw(g.N[2], M + 1);
    std::vector<int> posz(M);
    for (int pos = 0; pos < M; pos++) posz[freq_of_pos(pz, pos)] = pos;
    float2 *dtab = reinterpret_cast<float2 *>(c->fft_tab);
    int *dpos = reinterpret_cast<int *>(dtab + ((h.size() + 15) / 16) * 16);
    PM_CUDA(c, cudaMemcpy(dtab, h.data(), sizeof(float2) * h.size(), cudaMemcpyHostToDevice));
    PM_CUDA(c, cudaMemcpy(dpos, posz.data(), sizeof(int) * posz.size(), cudaMemcpyHostToDevice));
    fg->twx = dtab + ox;
    fg->twy = dtab + oy;
    fg->twz = dtab + oz;
    fg->twzr = dtab + ozr;
    fg->posz = dpos;
    fg->ktab = c->ktab;
    fg->tabn = c->ktabn;
    fg->c0 = 0.0;
    return PM_OK;
}

#define PM_FFT_LAUNCH(ctx, name, kernel, grid, smem, ...)                                  \
    do {                                                                                   \
        /* every instantiation is launched with ONE shared-memory size per mesh axis length, the largest it ever needs */ \
        static unsigned long long attr_mask_ = 0;                                          \
        static size_t attr_bytes_ = 0;                                                     \
        if ((smem) > attr_bytes_) { attr_mask_ = 0; attr_bytes_ = (smem); }                \
        if (smem_attr_needed(ctx, &attr_mask_))                                            \
            PM_CUDA(ctx, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)attr_bytes_)); \
        PM_CUDA(ctx, launch_pdl(kernel, dim3(grid), dim3(FFT_T), smem, (ctx)->stream, __VA_ARGS__)); \
        PM_LAUNCH_CHECK(ctx, name);                                                        \
    } while (0)

// N is a template parameter of every kernel: dispatch over the supported powers of two
#define PM_FFT_SWITCH_X(n, CASE)        \
    switch (n) {                        \
        case 16: CASE(16, 4); break;    \
        case 32: CASE(32, 4); break;    \
        case 64: CASE(64, 4); break;    \
        case 128: CASE(128, 4); break;  \
        case 256: CASE(256, 4); break;  \
        case 512: CASE(512, 4); break;  \
        case 1024: CASE(1024, 3); break; \
        default: return fail(c, PM_EINVAL, "own FFT", "unsupported axis length"); \
    }
#define PM_FFT_SWITCH(n, CASE)          \
    switch (n) {                        \
        case 8: CASE(8, 4); break;      \
        case 16: CASE(16, 4); break;    \
        case 32: CASE(32, 4); break;    \
        case 64: CASE(64, 4); break;    \
        case 128: CASE(128, 4); break;  \
        case 256: CASE(256, 4); break;  \
        case 512: CASE(512, 4); break;  \
        case 1024: CASE(1024, 3); break; \
        default: return fail(c, PM_EINVAL, "own FFT", "unsupported axis length"); \
    }

static int fft_z(pm_ctx *c, float *mesh, int nb, bool inverse)
{
    const Geometry &g = c->g;
    FftGeom fg = *geom_of(c);
    const int M = g.N[2] / 2;
    long long nrows = (long long)nb * g.N[0] * g.N[1];
    // 16 rows per CTA, 8 for the longest rows (2 CTAs per SM at Nz = 1024); 8 rows at Nz = 512 were measured slower (0.48 -> 0.53 ms)
    const int ZRS = M >= 512 ? 3 : 4, ZROWS = 1 << ZRS, ZP = ZROWS + 1;
    unsigned grid = (unsigned)((nrows + ZROWS - 1) / ZROWS);
    size_t second = (size_t)(M + 1) * ZP;                       // outb / inb: transposed [M + 1][ZP] or row-major staging
    if (second < (size_t)ZROWS * (g.zs / 2)) second = (size_t)ZROWS * (g.zs / 2);
    const int TP = ZRS == 3 ? 8 : ZP;                           // tile pitch (8 unpadded, swizzled rows: see trow)
    size_t smem = sizeof(float2) * ((size_t)M * TP + second + M + (M + 1)) + sizeof(int) * (size_t)M;
    Timer t(c, inverse ? TC_FFT_Z_C2R : TC_FFT_Z_R2C, 8.0 * (double)g.ng * nb);
#define Z_CASE(NN, CS_)                                                                                     \
    if (inverse) PM_FFT_LAUNCH(c, "fft_z_c2r_kernel", (fft_z_c2r_kernel<NN, CS_>), grid, smem, fg, mesh, nrows);  \
    else PM_FFT_LAUNCH(c, "fft_z_r2c_kernel", (fft_z_r2c_kernel<NN, CS_>), grid, smem, fg, mesh, nrows)
    switch (M) {
        case 8: Z_CASE(8, 4); break;
        case 16: Z_CASE(16, 4); break;
        case 32: Z_CASE(32, 4); break;
        case 64: Z_CASE(64, 4); break;
        case 128: Z_CASE(128, 4); break;
        case 256: Z_CASE(256, 4); break;
        case 512: Z_CASE(512, 3); break;
        default: return fail(c, PM_EINVAL, "own FFT", "unsupported Nz");
    }
#undef Z_CASE
    t.stop();
    return PM_OK;
}

static int fft_y(pm_ctx *c, float *mesh, int nb, bool inverse)
{
    const Geometry &g = c->g;
    FftGeom fg = *geom_of(c);
    // 16 columns (128-byte pieces) up to 512 points: 0.445 -> 0.394 ms per launch at 512^3 against 8 columns; at 1024 a
    // 16-column tile is 128 KB (one CTA per SM) and loses (3.9 -> 5.1 ms): 8 columns there
    const int cs = g.N[1] <= 512 ? 4 : 3, B = 1 << cs;
    dim3 grid((unsigned)((fg.zsc + B - 1) / B), (unsigned)g.N[0], (unsigned)nb);
    size_t smem = sizeof(float2) * ((size_t)g.N[1] + (size_t)g.N[1] * B);
    Timer t(c, TC_FFT_Y, 16.0 * (double)g.nk * nb);
#define Y_CASE(NN, CS_)                                                                                                   \
    if (inverse) PM_FFT_LAUNCH(c, "fft_y_kernel<inv>", (fft_y_kernel<NN, CS_, true>), grid, smem, fg, (float2 *)mesh);   \
    else PM_FFT_LAUNCH(c, "fft_y_kernel<fwd>", (fft_y_kernel<NN, CS_, false>), grid, smem, fg, (float2 *)mesh)
    PM_FFT_SWITCH(g.N[1], Y_CASE)
#undef Y_CASE
    t.stop();
    return PM_OK;
}

static int fft_x_fused(pm_ctx *c, const float *in, float *out, double nbar, bool adjoint)
{
    const Geometry &g = c->g;
    FftGeom fg = *geom_of(c);
    fg.c0 = 1.5 * c->prm.omega_m / (nbar * (double)g.ng);
    // one tile of Nx x B: 16 columns (128-byte pieces) up to 512 points (0.76 -> 0.71 ms at 512^3 against 8 columns, two CTAs
    // per SM at 128 registers), 8 columns at 1024
    const int cs = g.N[0] <= 512 ? 4 : 3, B = 1 << cs;
    dim3 grid((unsigned)((fg.zsc + B - 1) / B), (unsigned)g.N[1]);
    size_t smem = sizeof(float2) * ((size_t)g.N[0] + (size_t)g.N[0] * B) + (2 * sizeof(double) + sizeof(float)) * (size_t)g.N[0];
    Timer t(c, adjoint ? TC_KSPACE_ADJ : TC_KSPACE_FORCE, 32.0 * (double)g.nk);
#define X_CASE(NN, CS_)                                                                                                                   \
    if (adjoint) PM_FFT_LAUNCH(c, "fft_x_adjoint_kernel", (fft_x_adjoint_kernel<NN, CS_>), grid, smem, fg, (const float2 *)in, (float2 *)out); \
    else PM_FFT_LAUNCH(c, "fft_x_force_kernel", (fft_x_force_kernel<NN, CS_>), grid, smem, fg, (const float2 *)in, (float2 *)out)
    PM_FFT_SWITCH_X(g.N[0], X_CASE)
#undef X_CASE
    t.stop();
    return PM_OK;
}

// rho (1 mesh, real, padded) -> f_d (3 meshes, real, padded): eq. 11 with the spectral gradient (L127-131).
// part 1 = z, y forward and the fused x kernel (rho is dead afterwards), part 2 = the inverse y and z passes; 0 = both
int fft_own_force(pm_ctx *c, float *rho, float *f3, double nbar, int part)
{
    if (part != 2) {
        PM_TRY(fft_z(c, rho, 1, false));
        PM_TRY(fft_y(c, rho, 1, false));
        PM_TRY(fft_x_fused(c, rho, f3, nbar, false));
    }
    if (part != 1) {
        PM_TRY(fft_y(c, f3, 3, true));
        PM_TRY(fft_z(c, f3, 3, true));
    }
    return PM_OK;
}

// Pi_d (3 meshes) -> psi (1 mesh): the transpose of the force operator.
// part 1 = z, y forward on the three meshes, part 2 = the fused x kernel (writes psi) and the inverse y, z; 0 = both
int fft_own_adjoint(pm_ctx *c, float *Pi3, float *psi, double nbar, int part)
{
    if (part != 2) {
        PM_TRY(fft_z(c, Pi3, 3, false));
        PM_TRY(fft_y(c, Pi3, 3, false));
    }
    if (part != 1) {
        PM_TRY(fft_x_fused(c, Pi3, psi, nbar, true));
        PM_TRY(fft_y(c, psi, 1, true));
        PM_TRY(fft_z(c, psi, 1, true));
    }
    return PM_OK;
}

}  // namespace pm
