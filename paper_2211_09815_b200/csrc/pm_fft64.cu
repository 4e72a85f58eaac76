// pm_fft64.cu -- the 3-D transforms and the k-space operators of eq. 11 in DOUBLE precision (pm_params.flags bit 0,
// PM_FLAG_FP64_TRANSFORMS).
//
// where the reverse-time integration / the gradient needs it, "more precise floating-point numbers" are
// the paper's first remedy (its Tables 1-2 carry fp64 rows, L430-472).  The per-stage precision A/B of DESIGN.md
// section 7 shows that of all fp32 stages of F(x) only the transforms matter for the gradient at configs[1]: an fp32 FFT
// at its theoretical rounding error (~3e-7 of the mesh rms) moves the forward trajectory by 7e-6 cell and the gradient by
// 1.7e-3, the same transforms in fp64 by 1.7e-6 cell and 1.5e-4.  This mode therefore keeps every particle and mesh array
// of the path in fp32 (scatter, gathers, kick/drift unchanged) and runs only
//     rho (fp32) -> fp64 -> D2Z -> f_d(k) = i kt_d G rho(k) (fp64) -> 3 x Z2D -> fp32 force meshes       (eq. 11)
//     Pi_d (fp32) -> fp64 -> 3 x D2Z -> psi(k) = -i G sum_d kt_d Pi_d(k) -> Z2D -> fp32                    (its transpose)
// through cuFFT's double-precision plans (cuFFT is allowed for the 3-D transforms) and the two fp64 kernels below.
// Four fp64 meshes and the plans' work area are carved from the caller's workspace (pm_workspace_bytes grows).
#include <cstdio>

#include "pm_internal.cuh"

namespace pm {

#define PM_FFT64(ctx, call)                                                    \
    do {                                                                       \
        cufftResult r_ = (call);                                               \
        if (r_ != CUFFT_SUCCESS) {                                             \
            char b_[32];                                                       \
            snprintf(b_, sizeof b_, "cufftResult %d", (int)r_);                \
            return pm::fail(ctx, PM_ECUFFT, #call, b_);                        \
        }                                                                      \
    } while (0)

static inline int grid_for(long long n)
{
    long long b = (n + 255) / 256;
    return (int)(b > 148 * 16 ? 148 * 16 : (b < 1 ? 1 : b));
}

// padded fp32 mesh [rows][zs] <-> padded fp64 mesh [rows][Nz + 2] (real part of the in-place D2Z layout)
__global__ void f32_to_f64_kernel(long long nrow, int Nz, int zs, const float *__restrict__ src, double *__restrict__ dst)
{
    const long long n = nrow * Nz;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const long long row = i / Nz;
        const int iz = (int)(i - row * Nz);
        dst[(size_t)row * (Nz + 2) + iz] = (double)src[(size_t)row * zs + iz];
    }
}
__global__ void f64_to_f32_kernel(long long nrow, int Nz, int zs, const double *__restrict__ src, float *__restrict__ dst)
{
    const long long n = nrow * Nz;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const long long row = i / Nz;
        const int iz = (int)(i - row * Nz);
        dst[(size_t)row * zs + iz] = (float)src[(size_t)row * (Nz + 2) + iz];
    }
}

// G(k) = c0 dec / k^2, G(0) = 0 (R9); tab = [3 axes][kt, k^2, dec][tn] in natural frequency order (the cuFFT layout)
struct Mode64 {
    double G, kt[3];
};
__device__ __forceinline__ Mode64 mode64(const double *__restrict__ tab, int tn, double c0, int ix, int iy, int iz)
{
    Mode64 m;
    const double k2 = tab[tn + ix] + tab[3 * tn + tn + iy] + tab[6 * tn + tn + iz];
    const double dec = tab[2 * tn + ix] * tab[3 * tn + 2 * tn + iy] * tab[6 * tn + 2 * tn + iz];
    m.G = (ix | iy | iz) == 0 ? 0.0 : c0 * dec / k2;
    m.kt[0] = tab[ix];
    m.kt[1] = tab[3 * tn + iy];
    m.kt[2] = tab[6 * tn + iz];
    return m;
}

// f_d(k) = i kt_d G rho(k)   (eq. 11 with the spectral gradient, L127-131; kt = 0 on the Nyquist planes, R10)
__global__ void kspace_force64_kernel(int Nx, int Ny, int Nz, const double *__restrict__ tab, int tn, double c0,
                                      const double2 *__restrict__ rho, double2 *__restrict__ f0, double2 *__restrict__ f1,
                                      double2 *__restrict__ f2)
{
    const int nzc = Nz / 2 + 1;
    const long long nk = (long long)Nx * Ny * nzc;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nk; i += (long long)gridDim.x * blockDim.x) {
        const int iz = (int)(i % nzc);
        const long long row = i / nzc;
        const int iy = (int)(row % Ny), ix = (int)(row / Ny);
        const Mode64 m = mode64(tab, tn, c0, ix, iy, iz);
        const double2 r = rho[i];
        const double cx = m.kt[0] * m.G, cy = m.kt[1] * m.G, cz = m.kt[2] * m.G;
        f0[i] = make_double2(-cx * r.y, cx * r.x);
        f1[i] = make_double2(-cy * r.y, cy * r.x);
        f2[i] = make_double2(-cz * r.y, cz * r.x);
    }
}

// psi(k) = -i G sum_d kt_d Pi_d(k)   (the transpose of the operator above)
__global__ void kspace_adjoint64_kernel(int Nx, int Ny, int Nz, const double *__restrict__ tab, int tn, double c0,
                                        const double2 *__restrict__ P0, const double2 *__restrict__ P1,
                                        const double2 *__restrict__ P2, double2 *__restrict__ psi)
{
    const int nzc = Nz / 2 + 1;
    const long long nk = (long long)Nx * Ny * nzc;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nk; i += (long long)gridDim.x * blockDim.x) {
        const int iz = (int)(i % nzc);
        const long long row = i / nzc;
        const int iy = (int)(row % Ny), ix = (int)(row / Ny);
        const Mode64 m = mode64(tab, tn, c0, ix, iy, iz);
        const double2 a = P0[i], b = P1[i], d = P2[i];
        const double re = m.G * (m.kt[0] * a.x + m.kt[1] * b.x + m.kt[2] * d.x);
        const double im = m.G * (m.kt[0] * a.y + m.kt[1] * b.y + m.kt[2] * d.y);
        psi[i] = make_double2(im, -re);
    }
}

size_t fft64_mesh_doubles(const Geometry &g) { return (size_t)g.N[0] * g.N[1] * (g.N[2] + 2); }
// cuFFT's double-precision plans ask for about one complex mesh of work area; two are reserved (checked in fft64_init)
size_t fft64_work_bytes(const Geometry &g) { return 2 * sizeof(double) * fft64_mesh_doubles(g) + (32u << 20); }

int fft64_init(pm_ctx *c)
{
    const Geometry &g = c->g;
    size_t ws = 0, need = 0;
    PM_FFT64(c, cufftCreate(&c->plan_d2z));
    PM_FFT64(c, cufftCreate(&c->plan_z2d));
    c->plans64_ok = true;
    PM_FFT64(c, cufftSetAutoAllocation(c->plan_d2z, 0));
    PM_FFT64(c, cufftSetAutoAllocation(c->plan_z2d, 0));
    PM_FFT64(c, cufftMakePlan3d(c->plan_d2z, g.N[0], g.N[1], g.N[2], CUFFT_D2Z, &ws));
    need = ws;
    PM_FFT64(c, cufftMakePlan3d(c->plan_z2d, g.N[0], g.N[1], g.N[2], CUFFT_Z2D, &ws));
    if (ws > need) need = ws;
    if (need > c->fft64_work_bytes) {
        char b[128];
        snprintf(b, sizeof b, "cuFFT fp64 work area %zu > reserved %zu", need, c->fft64_work_bytes);
        return fail(c, PM_EWORKSPACE, "fft64_init", b);
    }
    PM_FFT64(c, cufftSetWorkArea(c->plan_d2z, c->fft64_work));
    PM_FFT64(c, cufftSetWorkArea(c->plan_z2d, c->fft64_work));
    PM_FFT64(c, cufftSetStream(c->plan_d2z, c->stream));
    PM_FFT64(c, cufftSetStream(c->plan_z2d, c->stream));
    return PM_OK;
}

void fft64_destroy(pm_ctx *c)
{
    if (c->plans64_ok) {
        cufftDestroy(c->plan_d2z);
        cufftDestroy(c->plan_z2d);
        c->plans64_ok = false;
    }
}

static int to64(pm_ctx *c, const float *src, double *dst)
{
    const Geometry &g = c->g;
    Timer t(c, TC_CONVERT, 12.0 * (double)g.ng);
    f32_to_f64_kernel<<<grid_for(g.ng), 256, 0, c->stream>>>((long long)g.N[0] * g.N[1], g.N[2], g.zs, src, dst);
    PM_LAUNCH_CHECK(c, "f32_to_f64_kernel");
    t.stop();
    return PM_OK;
}
static int to32(pm_ctx *c, const double *src, float *dst)
{
    const Geometry &g = c->g;
    Timer t(c, TC_CONVERT, 12.0 * (double)g.ng);
    f64_to_f32_kernel<<<grid_for(g.ng), 256, 0, c->stream>>>((long long)g.N[0] * g.N[1], g.N[2], g.zs, src, dst);
    PM_LAUNCH_CHECK(c, "f64_to_f32_kernel");
    t.stop();
    return PM_OK;
}
static int d2z(pm_ctx *c, double *m)
{
    Timer t(c, TC_FFT_R2C, 16.0 * (double)c->g.ng);
    PM_FFT64(c, cufftExecD2Z(c->plan_d2z, m, (cufftDoubleComplex *)m));
    t.stop();
    return PM_OK;
}
static int z2d(pm_ctx *c, double *m)
{
    Timer t(c, TC_FFT_C2R, 16.0 * (double)c->g.ng);
    PM_FFT64(c, cufftExecZ2D(c->plan_z2d, (cufftDoubleComplex *)m, m));
    t.stop();
    return PM_OK;
}

// rho (fp32 internal mesh) -> the three force meshes f3[0..2] (fp32 internal meshes)
int fft64_force(pm_ctx *c, const float *rho, float *f3, double nbar)
{
    const Geometry &g = c->g;
    const double c0 = 1.5 * c->prm.omega_m / (nbar * (double)g.ng);
    PM_TRY(to64(c, rho, c->dmesh[0]));
    PM_TRY(d2z(c, c->dmesh[0]));
    {
        Timer t(c, TC_KSPACE_FORCE, 64.0 * (double)g.nk);
        kspace_force64_kernel<<<grid_for(g.nk), 256, 0, c->stream>>>(g.N[0], g.N[1], g.N[2], c->ktab, c->ktabn, c0, (const double2 *)c->dmesh[0],
                                                                      (double2 *)c->dmesh[1], (double2 *)c->dmesh[2], (double2 *)c->dmesh[3]);
        PM_LAUNCH_CHECK(c, "kspace_force64_kernel");
        t.stop();
    }
    for (int d = 0; d < 3; d++) {
        PM_TRY(z2d(c, c->dmesh[1 + d]));
        PM_TRY(to32(c, c->dmesh[1 + d], f3 + (size_t)d * g.mesh_stride));
    }
    return PM_OK;
}

// Pi3[0..2] (fp32 internal meshes) -> psi (fp32 internal mesh)
int fft64_adjoint(pm_ctx *c, const float *Pi3, float *psi, double nbar)
{
    const Geometry &g = c->g;
    const double c0 = 1.5 * c->prm.omega_m / (nbar * (double)g.ng);
    for (int d = 0; d < 3; d++) {
        PM_TRY(to64(c, Pi3 + (size_t)d * g.mesh_stride, c->dmesh[1 + d]));
        PM_TRY(d2z(c, c->dmesh[1 + d]));
    }
    {
        Timer t(c, TC_KSPACE_ADJ, 64.0 * (double)g.nk);
        kspace_adjoint64_kernel<<<grid_for(g.nk), 256, 0, c->stream>>>(g.N[0], g.N[1], g.N[2], c->ktab, c->ktabn, c0, (const double2 *)c->dmesh[1],
                                                                        (const double2 *)c->dmesh[2], (const double2 *)c->dmesh[3], (double2 *)c->dmesh[0]);
        PM_LAUNCH_CHECK(c, "kspace_adjoint64_kernel");
        t.stop();
    }
    PM_TRY(z2d(c, c->dmesh[0]));
    return to32(c, c->dmesh[0], psi);
}

}  // namespace pm
