// pm_kspace.cu -- fused k-space kernels: Poisson Green's function x spectral gradient, and its transpose.
//
// PAPER.md eq. 9, 11 (L117-131), H0 = 1, cell units:  -k^2 varphi(k) = 3/2 Om delta(k);  the force is
// -i k varphi(k), "4 (1 forward and 3 inverse) FFTs in total" (L131).  With delta = rho/nbar - 1 (L79;
// the "-1" only touches k = 0, which is zeroed) and cuFFT's unnormalised transforms:
//     f_d(k)  = +i kt_d * G(k) * rho(k),         G(k) = 3/2 Om * dec(k) / (k^2 nbar N_g),  G(0) = 0
//     psi(k)  = -i G(k) * sum_d kt_d * Pi_d(k)   (transpose: kernel conjugated, components summed)
// kt_d = k_d except 0 on the Nyquist plane (R10); k^2 uses the full k also there; dec = 1 or the CIC
// deconvolution prod_d sinc(k_d/2)^-4 (R12).  Per-axis tables (kt, k^2, dec) are built on the host in fp64.
#include "pm_internal.cuh"

namespace pm {

struct KGeom {
    int N[3];
    int nzc;            // Nz/2 + 1 modes per z-row
    int zsc;            // complex elements per (padded) z-row in memory: zs / 2
    long long nk;       // complex elements per mesh
    long long cstride;  // complex elements between components (padded mesh stride / 2)
    const double *tab;  // [3 axes][3: kt, k2, dec][tabn], fp64: G(k) kt_d is rounded to fp32 ONCE, so the same
    int tabn;           //   (coherent) relative error is not applied to a mode at every step
    double c0;          // 3/2 Om / (nbar N_g)
};

// idx enumerates the Nx*Ny*(Nz/2+1) modes; returns the element offset of that mode in the padded mesh
__device__ __forceinline__ size_t k_factors(const KGeom &g, long long idx, double kt[3], double *G)
{
    int iz = (int)(idx % g.nzc);
    long long row = idx / g.nzc;
    int iy = (int)(row % g.N[1]);
    int ix = (int)(row / g.N[1]);
    const double *tx = g.tab, *ty = g.tab + 3 * g.tabn, *tz = g.tab + 6 * g.tabn;
    kt[0] = tx[ix];
    kt[1] = ty[iy];
    kt[2] = tz[iz];
    double k2 = tx[g.tabn + ix] + ty[g.tabn + iy] + tz[g.tabn + iz];
    double dec = tx[2 * g.tabn + ix] * ty[2 * g.tabn + iy] * tz[2 * g.tabn + iz];
    // reciprocal seed + one Newton step in fp64 (relative error ~1e-14) instead of an fp64 division
    double r = (double)__frcp_rn((float)k2);
    r = r * (2.0 - k2 * r);
    *G = (ix | iy | iz) == 0 ? 0.0 : g.c0 * dec * r;
    return (size_t)row * g.zsc + iz;
}

__global__ void __launch_bounds__(256) kspace_force_kernel(KGeom g, const float2 *__restrict__ rho_k, float2 *__restrict__ f_k)
{
    long long stride = (long long)gridDim.x * blockDim.x;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < g.nk; idx += stride) {
        double kt[3], G;
        size_t o = k_factors(g, idx, kt, &G);
        float2 r = rho_k[o];
#pragma unroll
        for (int d = 0; d < 3; d++) {
            float c = (float)(kt[d] * G);  // times +i: (re, im) -> (-c im, c re)
            f_k[(size_t)d * g.cstride + o] = make_float2(-c * r.y, c * r.x);
        }
    }
}

__global__ void __launch_bounds__(256) kspace_adjoint_kernel(KGeom g, const float2 *__restrict__ Pi_k, float2 *__restrict__ psi_k)
{
    long long stride = (long long)gridDim.x * blockDim.x;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < g.nk; idx += stride) {
        double kt[3], G;
        size_t o = k_factors(g, idx, kt, &G);
        float re = 0.f, im = 0.f;
#pragma unroll
        for (int d = 0; d < 3; d++) {
            float2 v = Pi_k[(size_t)d * g.cstride + o];
            float c = (float)(kt[d] * G);  // the same fp32 factors as the force kernel: exact transpose
            re += c * v.x;
            im += c * v.y;
        }
        // times -i: (re, im) -> (im, -re)
        psi_k[o] = make_float2(im, -re);
    }
}

static KGeom make_kgeom(pm_ctx *c, double nbar)
{
    KGeom k;
    for (int d = 0; d < 3; d++) k.N[d] = c->g.N[d];
    k.nzc = c->g.N[2] / 2 + 1;
    k.zsc = c->g.zs / 2;
    k.nk = c->g.nk;
    k.cstride = c->g.mesh_stride / 2;
    k.tab = c->ktab;
    k.tabn = c->ktabn;
    k.c0 = 1.5 * c->prm.omega_m / (nbar * (double)c->g.ng);
    return k;
}

int kspace_force(pm_ctx *c, const float2 *rho_k, float2 *f_k, double nbar)
{
    KGeom k = make_kgeom(c, nbar);
    int blocks = (int)((k.nk + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    Timer t(c, TC_KSPACE_FORCE, 32.0 * (double)k.nk);
    kspace_force_kernel<<<blocks, 256, 0, c->stream>>>(k, rho_k, f_k);
    PM_LAUNCH_CHECK(c, "kspace_force_kernel");
    t.stop();
    return PM_OK;
}

int kspace_adjoint(pm_ctx *c, const float2 *Pi_k, float2 *psi_k, double nbar)
{
    KGeom k = make_kgeom(c, nbar);
    int blocks = (int)((k.nk + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    Timer t(c, TC_KSPACE_ADJ, 32.0 * (double)k.nk);
    kspace_adjoint_kernel<<<blocks, 256, 0, c->stream>>>(k, Pi_k, psi_k);
    PM_LAUNCH_CHECK(c, "kspace_adjoint_kernel");
    t.stop();
    return PM_OK;
}

}  // namespace pm
