// pm_debug_prec.cu -- PROBE BUILD ONLY (-DPM_DEBUG, libpm_debug.so; an empty translation unit in libpm.so).
//
// Per-stage precision A/B of the hot path (DESIGN.md section 7 "Precision A/B"): every stage of F(x), of the force VJP
// and of the objective can be swapped for a plain fp64 variant -- naive kernels, fp64 atomics, cuFFT D2Z / Z2D, positions
// taken from the int64 state without the 2^-fbits quantisation of the sort records -- so that the contribution of each
// stage's fp32 rounding to the final-position and gradient differences against the oracle can be measured one by one.
// PM_DBG_PREC (bit mask, read at pm_init):
//    1  S   unit-mass scatter in fp64              8  S3  scatter of pi in fp64
//    2  T   transforms + eq. 11 in fp64           16  T'  transforms + transposed operator in fp64
//    4  G   force gather in fp64                  32  G'  weight-gradient (fused) gather in fp64
//   64  O   objective: scatter, residual, J, xi_n in fp64
//  128  A   adjoint variables xi, pi, alpha held and updated in fp64
//  256  (no stage swapped) run the step-by-step product kernels through this driver (must equal libpm.so bit for bit)
// Not bit-reversible when S, S3 or O are on (fp64 atomics are unordered): the reverse pass then differs from the forward
// one at the 1e-16 level, irrelevant for the A/B.
#ifdef PM_DEBUG
#include <cstdio>
#include <cstdlib>

#include "pm_pos.cuh"

namespace pm {

enum { DP_S = 1, DP_T = 2, DP_G = 4, DP_S3 = 8, DP_TA = 16, DP_GA = 32, DP_O = 64, DP_A = 128, DP_DRIVER = 256 };

struct DbgPrec {
    int flags;
    double *dm[7];            // fp64 meshes, padded in-place D2Z layout [Nx][Ny][Nz + 2]
    cufftHandle d2z, z2d;
    double *ktab;             // [3 axes][3: kt, k2, dec][tabn] in NATURAL frequency order
    int tabn;
    double *dxi, *dpi, *dalpha;   // DP_A
    double *dJ;
    float *scratch3;          // [np][3] floats: acc output of the product's fused gather when it must not clobber c->acc
    bool f64_force_valid;     // dm[1..3] hold the force meshes of the current positions
};

static DbgPrec *g_dbg = nullptr;   // one ctx at a time in the probe build
static pm_ctx *g_dbg_ctx = nullptr;

int dbg_prec_flags(pm_ctx *c) { return (g_dbg && g_dbg_ctx == c) ? g_dbg->flags : 0; }

#define DBG_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return fail(c, PM_ECUDA, #call, cudaGetErrorString(e_)); } while (0)
#define DBG_FFT(call) do { cufftResult r_ = (call); if (r_ != CUFFT_SUCCESS) { char b_[32]; snprintf(b_, sizeof b_, "cufftResult %d", (int)r_); return fail(c, PM_ECUFFT, #call, b_); } } while (0)

static inline int nblk(long long n) { long long b = (n + 255) / 256; return (int)(b > 148 * 32 ? 148 * 32 : (b < 1 ? 1 : b)); }

int dbg_prec_init(pm_ctx *c)
{
    const char *e = getenv("PM_DBG_PREC");
    if (!e) return PM_OK;
    const int flags = atoi(e);
    if (!flags) return PM_OK;
    const Geometry &g = c->g;
    DbgPrec *d = new DbgPrec();
    d->flags = flags;
    const size_t dstride = (size_t)g.N[0] * g.N[1] * (g.N[2] + 2);
    for (int k = 0; k < 7; k++) DBG_CUDA(cudaMalloc(&d->dm[k], sizeof(double) * dstride));
    DBG_FFT(cufftPlan3d(&d->d2z, g.N[0], g.N[1], g.N[2], CUFFT_D2Z));
    DBG_FFT(cufftPlan3d(&d->z2d, g.N[0], g.N[1], g.N[2], CUFFT_Z2D));
    DBG_FFT(cufftSetStream(d->d2z, c->stream));
    DBG_FFT(cufftSetStream(d->z2d, c->stream));
    int tn = c->ktabn;
    d->tabn = tn;
    std::vector<double> h((size_t)9 * tn, 0.0);
    const double PI = 3.14159265358979323846264338327950288;
    for (int ax = 0; ax < 3; ax++) {
        const int N = g.N[ax];
        for (int i = 0; i < N; i++) {
            const int m = i < (N + 1) / 2 ? i : i - N;
            const double k = 2.0 * PI * (double)m / (double)N;
            const bool nyq = (N % 2 == 0) && (m == -N / 2);
            double dec = 1.0;
            if (c->prm.deconvolve && m != 0) {
                const double hh = 0.5 * k, sc = sin(hh) / hh;
                dec = 1.0 / (sc * sc * sc * sc);
            }
            h[(size_t)(3 * ax + 0) * tn + i] = nyq ? 0.0 : k;
            h[(size_t)(3 * ax + 1) * tn + i] = k * k;
            h[(size_t)(3 * ax + 2) * tn + i] = dec;
        }
    }
    DBG_CUDA(cudaMalloc(&d->ktab, sizeof(double) * h.size()));
    DBG_CUDA(cudaMemcpy(d->ktab, h.data(), sizeof(double) * h.size(), cudaMemcpyHostToDevice));
    const size_t n3 = 3 * (size_t)g.np;
    DBG_CUDA(cudaMalloc(&d->dxi, sizeof(double) * n3));
    DBG_CUDA(cudaMalloc(&d->dpi, sizeof(double) * n3));
    DBG_CUDA(cudaMalloc(&d->dalpha, sizeof(double) * n3));
    DBG_CUDA(cudaMalloc(&d->dJ, sizeof(double)));
    DBG_CUDA(cudaMalloc(&d->scratch3, sizeof(float) * n3));
    d->f64_force_valid = false;
    g_dbg = d;
    g_dbg_ctx = c;
    fprintf(stderr, "[libpm_debug] PM_DBG_PREC=%d\n", flags);
    return PM_OK;
}

void dbg_prec_destroy(pm_ctx *c)
{
    if (!g_dbg || g_dbg_ctx != c) return;
    for (int k = 0; k < 7; k++) cudaFree(g_dbg->dm[k]);
    cufftDestroy(g_dbg->d2z);
    cufftDestroy(g_dbg->z2d);
    cudaFree(g_dbg->ktab);
    cudaFree(g_dbg->dxi);
    cudaFree(g_dbg->dpi);
    cudaFree(g_dbg->dalpha);
    cudaFree(g_dbg->dJ);
    cudaFree(g_dbg->scratch3);
    delete g_dbg;
    g_dbg = nullptr;
    g_dbg_ctx = nullptr;
}

// ---- exact CIC geometry from the int64 state -------------------------------------------------------------------------
struct Cic64 {
    int i0[3], i1[3];
    double w[3][2];
};
__device__ __forceinline__ Cic64 cic64(const long long *__restrict__ x, long long j, int Nx, int Ny, int Nz)
{
    const int N[3] = {Nx, Ny, Nz};
    Cic64 r;
#pragma unroll
    for (int d = 0; d < 3; d++) {
        const long long v = x[3 * j + d];
        long long cell = v >> XBITS;                       // floor
        const double t = (double)(unsigned long long)(v & 0xffffffffll) * (1.0 / 4294967296.0);
        long long m = cell % N[d];
        if (m < 0) m += N[d];
        r.i0[d] = (int)m;
        r.i1[d] = (int)(m + 1 == N[d] ? 0 : m + 1);
        r.w[d][0] = 1.0 - t;
        r.w[d][1] = t;
    }
    return r;
}
#define CIC64_IDX(r, bx, by, bz, Ny, zs) (((size_t)((bx) ? r.i1[0] : r.i0[0]) * (Ny) + ((by) ? r.i1[1] : r.i0[1])) * (zs) + ((bz) ? r.i1[2] : r.i0[2]))

template <class V>
__global__ void k_scatter64(long long np, const long long *__restrict__ x, const V *__restrict__ val, int C, int Nx, int Ny, int Nz,
                            double *__restrict__ m0, double *__restrict__ m1, double *__restrict__ m2)
{
    const int zs = Nz + 2;
    double *mm[3] = {m0, m1, m2};
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < np; j += (long long)gridDim.x * blockDim.x) {
        const Cic64 r = cic64(x, j, Nx, Ny, Nz);
        double v[3] = {1.0, 0.0, 0.0};
        if (val) for (int c = 0; c < C; c++) v[c] = (double)val[(size_t)j * C + c];
#pragma unroll
        for (int bx = 0; bx < 2; bx++)
#pragma unroll
            for (int by = 0; by < 2; by++)
#pragma unroll
                for (int bz = 0; bz < 2; bz++) {
                    const double W = r.w[0][bx] * r.w[1][by] * r.w[2][bz];
                    const size_t o = CIC64_IDX(r, bx, by, bz, Ny, zs);
                    for (int c = 0; c < C; c++) atomicAdd(mm[c] + o, W * v[c]);
                }
    }
}

// acc_d = sum_g W f_d(g)
__global__ void k_gather64(long long np, const long long *__restrict__ x, int Nx, int Ny, int Nz, const double *__restrict__ f0,
                           const double *__restrict__ f1, const double *__restrict__ f2, float *__restrict__ acc)
{
    const int zs = Nz + 2;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < np; j += (long long)gridDim.x * blockDim.x) {
        const Cic64 r = cic64(x, j, Nx, Ny, Nz);
        double a[3] = {0, 0, 0};
#pragma unroll
        for (int bx = 0; bx < 2; bx++)
#pragma unroll
            for (int by = 0; by < 2; by++)
#pragma unroll
                for (int bz = 0; bz < 2; bz++) {
                    const double W = r.w[0][bx] * r.w[1][by] * r.w[2][bz];
                    const size_t o = CIC64_IDX(r, bx, by, bz, Ny, zs);
                    a[0] += W * f0[o];
                    a[1] += W * f1[o];
                    a[2] += W * f2[o];
                }
        for (int d = 0; d < 3; d++) acc[3 * j + d] = (float)a[d];
    }
}

// out_e = scale * sum_g d_eW(g, x_j) [ psi(g) + sum_d cot_d f_d(g) ]   (f == NULL: the scalar mesh only)
template <class V>
__global__ void k_gradgather64(long long np, const long long *__restrict__ x, int Nx, int Ny, int Nz, const double *__restrict__ psi,
                               const double *__restrict__ f0, const double *__restrict__ f1, const double *__restrict__ f2,
                               const V *__restrict__ cot, double scale, float *__restrict__ outf, double *__restrict__ outd)
{
    const int zs = Nz + 2;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < np; j += (long long)gridDim.x * blockDim.x) {
        const Cic64 r = cic64(x, j, Nx, Ny, Nz);
        double cv[3] = {0, 0, 0};
        if (f0) for (int d = 0; d < 3; d++) cv[d] = (double)cot[3 * j + d];
        double gr[3] = {0, 0, 0};
#pragma unroll
        for (int bx = 0; bx < 2; bx++)
#pragma unroll
            for (int by = 0; by < 2; by++)
#pragma unroll
                for (int bz = 0; bz < 2; bz++) {
                    const size_t o = CIC64_IDX(r, bx, by, bz, Ny, zs);
                    double m = psi[o];
                    if (f0) m += cv[0] * f0[o] + cv[1] * f1[o] + cv[2] * f2[o];
                    gr[0] += (bx ? 1.0 : -1.0) * r.w[1][by] * r.w[2][bz] * m;
                    gr[1] += (by ? 1.0 : -1.0) * r.w[0][bx] * r.w[2][bz] * m;
                    gr[2] += (bz ? 1.0 : -1.0) * r.w[0][bx] * r.w[1][by] * m;
                }
        for (int e = 0; e < 3; e++) {
            if (outf) outf[3 * j + e] = (float)(gr[e] * scale);
            if (outd) outd[3 * j + e] = gr[e] * scale;
        }
    }
}

// ---- k-space in fp64, natural order (cuFFT layout: [Nx][Ny][Nz/2 + 1] complex) ----------------------------------------
__global__ void k_kspace_force64(int Nx, int Ny, int Nz, const double *__restrict__ tab, int tn, double c0, const double2 *__restrict__ rho,
                                 double2 *__restrict__ f0, double2 *__restrict__ f1, double2 *__restrict__ f2)
{
    const int nzc = Nz / 2 + 1;
    const long long nk = (long long)Nx * Ny * nzc;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nk; i += (long long)gridDim.x * blockDim.x) {
        const int iz = (int)(i % nzc);
        const long long row = i / nzc;
        const int iy = (int)(row % Ny), ix = (int)(row / Ny);
        const double k2 = tab[tn + ix] + tab[3 * tn + tn + iy] + tab[6 * tn + tn + iz];
        const double dec = tab[2 * tn + ix] * tab[3 * tn + 2 * tn + iy] * tab[6 * tn + 2 * tn + iz];
        const double G = (ix | iy | iz) == 0 ? 0.0 : c0 * dec / k2;
        const double2 r = rho[i];
        const double kt[3] = {tab[ix], tab[3 * tn + iy], tab[6 * tn + iz]};
        double2 *f[3] = {f0, f1, f2};
        for (int d = 0; d < 3; d++) {
            const double c = kt[d] * G;
            f[d][i] = make_double2(-c * r.y, c * r.x);
        }
    }
}

__global__ void k_kspace_adj64(int Nx, int Ny, int Nz, const double *__restrict__ tab, int tn, double c0, const double2 *__restrict__ P0,
                               const double2 *__restrict__ P1, const double2 *__restrict__ P2, double2 *__restrict__ psi)
{
    const int nzc = Nz / 2 + 1;
    const long long nk = (long long)Nx * Ny * nzc;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nk; i += (long long)gridDim.x * blockDim.x) {
        const int iz = (int)(i % nzc);
        const long long row = i / nzc;
        const int iy = (int)(row % Ny), ix = (int)(row / Ny);
        const double k2 = tab[tn + ix] + tab[3 * tn + tn + iy] + tab[6 * tn + tn + iz];
        const double dec = tab[2 * tn + ix] * tab[3 * tn + 2 * tn + iy] * tab[6 * tn + 2 * tn + iz];
        const double G = (ix | iy | iz) == 0 ? 0.0 : c0 * dec / k2;
        const double kt[3] = {tab[ix], tab[3 * tn + iy], tab[6 * tn + iz]};
        const double2 *P[3] = {P0, P1, P2};
        double re = 0, im = 0;
        for (int d = 0; d < 3; d++) {
            const double2 v = P[d][i];
            re += kt[d] * G * v.x;
            im += kt[d] * G * v.y;
        }
        psi[i] = make_double2(im, -re);
    }
}

// ---- conversions between the padded fp32 meshes [..][zs] and the padded fp64 meshes [..][Nz + 2] --------------------
__global__ void k_f2d(long long nrow, int Nz, int zs, const float *__restrict__ src, double *__restrict__ dst)
{
    const long long n = nrow * Nz;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const long long row = i / Nz;
        const int iz = (int)(i % Nz);
        dst[(size_t)row * (Nz + 2) + iz] = (double)src[(size_t)row * zs + iz];
    }
}
__global__ void k_d2f(long long nrow, int Nz, int zs, const double *__restrict__ src, double sub, float *__restrict__ dst)
{
    const long long n = nrow * Nz;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const long long row = i / Nz;
        const int iz = (int)(i % Nz);
        dst[(size_t)row * zs + iz] = (float)(src[(size_t)row * (Nz + 2) + iz] - sub);
    }
}
__global__ void k_f2d_vec(long long n, const float *__restrict__ s, double *__restrict__ d)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) d[i] = (double)s[i];
}
__global__ void k_d2f_vec(long long n, const double *__restrict__ s, float *__restrict__ d)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) d[i] = (float)s[i];
}
// xi -= alpha K ; pi -= xi D  in fp64 (eq. 49)
__global__ void k_adj_update64(long long n, double K, double D, double *__restrict__ xi, double *__restrict__ pi, const double *__restrict__ alpha)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        double v = xi[i];
        if (K != 0.0) { v -= alpha[i] * K; xi[i] = v; }
        if (D != 0.0) pi[i] -= v * D;
    }
}
// r = rho/nbar - 1 - target in place (fp64 mesh), J += 1/2 sum r^2
__global__ void k_objective64(long long nrow, int Nz, double inv_nbar, double *__restrict__ m, const float *__restrict__ target, double *__restrict__ J)
{
    const long long n = nrow * Nz;
    double part = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const long long row = i / Nz;
        const int iz = (int)(i % Nz);
        const size_t o = (size_t)row * (Nz + 2) + iz;
        const double r = m[o] * inv_nbar - 1.0 - (double)target[i];
        m[o] = r;
        part += 0.5 * r * r;
    }
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(J, part);
}

// ---- drivers ---------------------------------------------------------------------------------------------------------
static size_t dstride(const Geometry &g) { return (size_t)g.N[0] * g.N[1] * (g.N[2] + 2); }
static long long nrows(const Geometry &g) { return (long long)g.N[0] * g.N[1]; }

// declared in pm_api.cu (same library): the product's stages
int dbg_product_transforms_force(pm_ctx *c, double nbar);     // c->mesh[0] (rho - nbar) -> c->mesh[1..3]
int dbg_product_transforms_adjoint(pm_ctx *c, double nbar);   // c->mesh[4..6] -> c->mesh[0]

// acc = F(x) of the current (sorted) state into c->acc
int dbg_force(pm_ctx *c)
{
    DbgPrec *d = g_dbg;
    const Geometry &g = c->g;
    const int F = d->flags;
    const double nbar = (double)g.np / (double)g.ng;
    const int Nx = g.N[0], Ny = g.N[1], Nz = g.N[2];
    cudaStream_t st = c->stream;
    // S
    if (F & DP_S) {
        DBG_CUDA(cudaMemsetAsync(d->dm[0], 0, sizeof(double) * dstride(g), st));
        k_scatter64<float><<<nblk(g.np), 256, 0, st>>>(g.np, c->x, (const float *)nullptr, 1, Nx, Ny, Nz, d->dm[0], nullptr, nullptr);
        if (!(F & DP_T)) k_d2f<<<nblk(g.ng), 256, 0, st>>>(nrows(g), Nz, g.zs, d->dm[0], nbar, c->mesh[0]);
    } else {
        PM_TRY(scatter_sorted(c, nullptr, 1, c->mesh[0], g.zs, g.mesh_stride, nbar));
        if (F & DP_T) k_f2d<<<nblk(g.ng), 256, 0, st>>>(nrows(g), Nz, g.zs, c->mesh[0], d->dm[0]);
    }
    // T
    if (F & DP_T) {
        DBG_FFT(cufftExecD2Z(d->d2z, d->dm[0], (cufftDoubleComplex *)d->dm[0]));
        const double c0 = 1.5 * c->prm.omega_m / (nbar * (double)g.ng);
        k_kspace_force64<<<nblk(g.nk), 256, 0, st>>>(Nx, Ny, Nz, d->ktab, d->tabn, c0, (const double2 *)d->dm[0], (double2 *)d->dm[1],
                                                      (double2 *)d->dm[2], (double2 *)d->dm[3]);
        for (int k = 1; k <= 3; k++) DBG_FFT(cufftExecZ2D(d->z2d, (cufftDoubleComplex *)d->dm[k], d->dm[k]));
        d->f64_force_valid = true;
        // the product's gathers (G off, or the fused gather of the VJP with G' off) read the fp32 meshes
        for (int k = 1; k <= 3; k++) k_d2f<<<nblk(g.ng), 256, 0, st>>>(nrows(g), Nz, g.zs, d->dm[k], 0.0, c->mesh[k]);
    } else {
        PM_TRY(dbg_product_transforms_force(c, nbar));
        d->f64_force_valid = false;
        if (F & (DP_G | DP_GA)) {
            for (int k = 1; k <= 3; k++) k_f2d<<<nblk(g.ng), 256, 0, st>>>(nrows(g), Nz, g.zs, c->mesh[k], d->dm[k]);
            d->f64_force_valid = true;
        }
    }
    // G
    if (F & DP_G) k_gather64<<<nblk(g.np), 256, 0, st>>>(g.np, c->x, Nx, Ny, Nz, d->dm[1], d->dm[2], d->dm[3], c->acc);
    else PM_TRY(gather_sorted(c, c->mesh[1], 3, g.zs, g.mesh_stride, c->acc));
    PM_LAUNCH_CHECK(c, "dbg_force");
    return PM_OK;
}

// alpha = pi . dF/dx for the current state; force meshes as left by dbg_force.  Writes c->alpha (and dalpha with DP_A).
int dbg_vjp(pm_ctx *c)
{
    DbgPrec *d = g_dbg;
    const Geometry &g = c->g;
    const int F = d->flags;
    const double nbar = (double)g.np / (double)g.ng;
    const int Nx = g.N[0], Ny = g.N[1], Nz = g.N[2];
    cudaStream_t st = c->stream;
    const long long n3 = 3 * g.np;
    if (F & DP_A) k_d2f_vec<<<nblk(n3), 256, 0, st>>>(n3, d->dpi, c->pi);   // the product kernels read fp32 pi
    // S3
    if (F & DP_S3) {
        for (int k = 4; k <= 6; k++) DBG_CUDA(cudaMemsetAsync(d->dm[k], 0, sizeof(double) * dstride(g), st));
        if (F & DP_A) k_scatter64<double><<<nblk(g.np), 256, 0, st>>>(g.np, c->x, d->dpi, 3, Nx, Ny, Nz, d->dm[4], d->dm[5], d->dm[6]);
        else k_scatter64<float><<<nblk(g.np), 256, 0, st>>>(g.np, c->x, c->pi, 3, Nx, Ny, Nz, d->dm[4], d->dm[5], d->dm[6]);
        if (!(F & DP_TA)) for (int k = 4; k <= 6; k++) k_d2f<<<nblk(g.ng), 256, 0, st>>>(nrows(g), Nz, g.zs, d->dm[k], 0.0, c->mesh[k]);
    } else {
        PM_TRY(scatter_sorted(c, c->pi, 3, c->mesh[4], g.zs, g.mesh_stride));
        if (F & DP_TA) for (int k = 4; k <= 6; k++) k_f2d<<<nblk(g.ng), 256, 0, st>>>(nrows(g), Nz, g.zs, c->mesh[k], d->dm[k]);
    }
    // T'
    if (F & DP_TA) {
        for (int k = 4; k <= 6; k++) DBG_FFT(cufftExecD2Z(d->d2z, d->dm[k], (cufftDoubleComplex *)d->dm[k]));
        const double c0 = 1.5 * c->prm.omega_m / (nbar * (double)g.ng);
        k_kspace_adj64<<<nblk(g.nk), 256, 0, st>>>(Nx, Ny, Nz, d->ktab, d->tabn, c0, (const double2 *)d->dm[4], (const double2 *)d->dm[5],
                                                    (const double2 *)d->dm[6], (double2 *)d->dm[0]);
        DBG_FFT(cufftExecZ2D(d->z2d, (cufftDoubleComplex *)d->dm[0], d->dm[0]));
        if (!(F & DP_GA)) k_d2f<<<nblk(g.ng), 256, 0, st>>>(nrows(g), Nz, g.zs, d->dm[0], 0.0, c->mesh[0]);
    } else {
        PM_TRY(dbg_product_transforms_adjoint(c, nbar));
        if (F & DP_GA) k_f2d<<<nblk(g.ng), 256, 0, st>>>(nrows(g), Nz, g.zs, c->mesh[0], d->dm[0]);
    }
    // G'
    if (F & DP_GA) {
        if (!d->f64_force_valid) return fail(c, PM_ESTATE, "dbg_vjp", "fp64 force meshes missing");
        if (F & DP_A)
            k_gradgather64<double><<<nblk(g.np), 256, 0, st>>>(g.np, c->x, Nx, Ny, Nz, d->dm[0], d->dm[1], d->dm[2], d->dm[3], d->dpi, 1.0, c->alpha, d->dalpha);
        else
            k_gradgather64<float><<<nblk(g.np), 256, 0, st>>>(g.np, c->x, Nx, Ny, Nz, d->dm[0], d->dm[1], d->dm[2], d->dm[3], c->pi, 1.0, c->alpha, nullptr);
    } else {
        // the product's fused gather also writes acc: into a scratch array, c->acc keeps what dbg_force produced
        PM_TRY(gather_fused_sorted(c, c->mesh[0], g.zs, g.mesh_stride, c->pi, d->scratch3, c->alpha));
        if (F & DP_A) k_f2d_vec<<<nblk(n3), 256, 0, st>>>(n3, c->alpha, d->dalpha);
    }
    PM_LAUNCH_CHECK(c, "dbg_vjp");
    return PM_OK;
}

int dbg_objective(pm_ctx *c, const float *target)
{
    DbgPrec *d = g_dbg;
    const Geometry &g = c->g;
    const int F = d->flags;
    const double nbar = (double)g.np / (double)g.ng;
    const int Nx = g.N[0], Ny = g.N[1], Nz = g.N[2];
    cudaStream_t st = c->stream;
    const long long n3 = 3 * g.np;
    if (F & DP_O) {
        DBG_CUDA(cudaMemsetAsync(d->dm[0], 0, sizeof(double) * dstride(g), st));
        DBG_CUDA(cudaMemsetAsync(d->dJ, 0, sizeof(double), st));
        k_scatter64<float><<<nblk(g.np), 256, 0, st>>>(g.np, c->x, (const float *)nullptr, 1, Nx, Ny, Nz, d->dm[0], nullptr, nullptr);
        k_objective64<<<nblk(g.ng), 256, 0, st>>>(nrows(g), Nz, 1.0 / nbar, d->dm[0], target, d->dJ);
        DBG_CUDA(cudaMemcpyAsync(c->scal, d->dJ, sizeof(double), cudaMemcpyDeviceToDevice, st));
        k_gradgather64<float><<<nblk(g.np), 256, 0, st>>>(g.np, c->x, Nx, Ny, Nz, d->dm[0], nullptr, nullptr, nullptr, (const float *)nullptr,
                                                          1.0 / nbar, c->xi, (F & DP_A) ? d->dxi : nullptr);
    } else {
        PM_TRY(scatter_sorted(c, nullptr, 1, c->mesh[0], g.zs, g.mesh_stride));
        PM_TRY(objective_residual(c, c->mesh[0], target, nbar));
        PM_TRY(gather_grad_sorted(c, c->mesh[0], 1, g.zs, g.mesh_stride, nullptr, (float)(1.0 / nbar), c->xi));
        if (F & DP_A) k_f2d_vec<<<nblk(n3), 256, 0, st>>>(n3, c->xi, d->dxi);
    }
    PM_TRY(fill_zero(c, c->pi, sizeof(float) * (size_t)n3));
    PM_TRY(fill_zero(c, c->alpha, sizeof(float) * (size_t)n3));
    if (F & DP_A) {
        DBG_CUDA(cudaMemsetAsync(d->dpi, 0, sizeof(double) * (size_t)n3, st));
        DBG_CUDA(cudaMemsetAsync(d->dalpha, 0, sizeof(double) * (size_t)n3, st));
    }
    PM_LAUNCH_CHECK(c, "dbg_objective");
    return PM_OK;
}

// xi -= alpha K; pi -= xi D on the fp64 copies (DP_A); the fp32 copies follow at the end of the run
int dbg_adj_update(pm_ctx *c, double K, double D)
{
    DbgPrec *d = g_dbg;
    const long long n3 = 3 * c->g.np;
    k_adj_update64<<<nblk(n3), 256, 0, c->stream>>>(n3, K, D, d->dxi, d->dpi, d->dalpha);
    PM_LAUNCH_CHECK(c, "dbg_adj_update");
    return PM_OK;
}

int dbg_adj_finish(pm_ctx *c)
{
    DbgPrec *d = g_dbg;
    if (!(d->flags & DP_A)) return PM_OK;
    const long long n3 = 3 * c->g.np;
    k_d2f_vec<<<nblk(n3), 256, 0, c->stream>>>(n3, d->dxi, c->xi);
    k_d2f_vec<<<nblk(n3), 256, 0, c->stream>>>(n3, d->dpi, c->pi);
    PM_LAUNCH_CHECK(c, "dbg_adj_finish");
    return PM_OK;
}

}  // namespace pm
#endif  // PM_DEBUG
