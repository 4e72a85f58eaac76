// pm_ic.cu -- initial conditions from white noise by Lagrangian perturbation theory on the device, and the VJP that
// turns the adjoint run's (xi_0, pi_0) into dJ/d(omega).
//
// PAPER.md eq. 2 (L59-63): s = D1 s1 + D2 s2, p = a^2 H (D1' s1 + D2' s2); eq. 3-4 (L69-77): s_m = -grad phi_m,
// lap phi_1 = delta_1, lap phi_2 = sum_{a<b} (phi_1,aa phi_1,bb - phi_1,ab^2); eq. 6 (L87): delta_1(k) = sqrt(V P) omega(k)
// with omega(k) the transform of a real white-noise field on the particle lattice (L89); eq. 51 second line (L406):
// dJ/d omega = xi_0 . dx_0/d omega + pi_0 . dp_0/d omega (the paper leaves this VJP to AD, L408; here it is the transpose
// of the steps below, taken backwards).  Readings (R29): P(k) = k^ns exp(-(rc k)^2) with the volume factor
// inside amp (the configs' recipe is ns = -1.5, rc = 2); k_d = 2 pi m_d / N_d per mesh cell for lattice mode m_d; odd
// multipliers (i k_d, k_a k_b with a != b) vanish on the lattice's Nyquist planes, even ones (k^2, k_a^2) do not (R10).
//
// Everything here lives on the PARTICLE LATTICE (Lx x Ly x Lz, an eighth of the mesh in the configs): fields sit in the
// padded in-place R2C layout [Lx][Ly][2 (Lz/2 + 1)] inside the ctx's mesh buffers (free outside a run), transforms are
// cuFFT plans on the lattice (allowed for the 3-D transforms), the multipliers are evaluated in fp64 per mode.
// 14 transforms forward, 25 for the VJP at second order -- a few per cent of one forward + adjoint run.
#include <cmath>
#include <cstdio>

#include "pm_internal.cuh"

namespace pm {

#define PM_ICFFT(ctx, call)                                                    \
    do {                                                                       \
        cufftResult r_ = (call);                                               \
        if (r_ != CUFFT_SUCCESS) {                                             \
            char b_[32];                                                       \
            snprintf(b_, sizeof b_, "cufftResult %d", (int)r_);                \
            return pm::fail(ctx, PM_ECUFFT, #call, b_);                        \
        }                                                                      \
    } while (0)

struct IcGeom {
    int L[3], N[3];
    int lzc;        // complex elements per z-row: Lz/2 + 1
    long long nk;   // Lx Ly lzc
    long long np;
    double amp, ns, rc;
};

static inline int ic_grid(long long n)
{
    long long b = (n + 255) / 256;
    return (int)(b > 148 * 16 ? 148 * 16 : (b < 1 ? 1 : b));
}

struct IcMode {
    double k[3], kt[3], k2;
};
__device__ __forceinline__ IcMode ic_mode(const IcGeom &g, long long i)
{
    IcMode m;
    const int iz = (int)(i % g.lzc);
    const long long r = i / g.lzc;
    const int idx[3] = {(int)(r / g.L[1]), (int)(r % g.L[1]), iz};
    m.k2 = 0.0;
#pragma unroll
    for (int d = 0; d < 3; d++) {
        const int L = g.L[d];
        const int mm = idx[d] < (L + 1) / 2 ? idx[d] : idx[d] - L;   // z: idx <= Lz/2, so +Lz/2 stands for the Nyquist plane
        const double k = 6.283185307179586476925286766559 * (double)mm / (double)g.N[d];
        const bool nyq = (L % 2 == 0) && (idx[d] == L / 2);
        m.k[d] = k;
        m.kt[d] = nyq ? 0.0 : k;
        m.k2 += k * k;
    }
    return m;
}
// amp sqrt(P(k)), P = k^ns exp(-(rc k)^2); 0 at k = 0
__device__ __forceinline__ double ic_transfer(const IcGeom &g, double k2)
{
    return k2 > 0.0 ? g.amp * sqrt(pow(k2, 0.5 * g.ns) * exp(-g.rc * g.rc * k2)) : 0.0;
}
// k_a k_b / k^2 for ab = xx yy zz xy xz yz
__device__ __forceinline__ double ic_hess(const IcMode &m, int ab)
{
    if (!(m.k2 > 0.0)) return 0.0;
    switch (ab) {
        case 0: return m.k[0] * m.k[0] / m.k2;
        case 1: return m.k[1] * m.k[1] / m.k2;
        case 2: return m.k[2] * m.k[2] / m.k2;
        case 3: return m.kt[0] * m.kt[1] / m.k2;
        case 4: return m.kt[0] * m.kt[2] / m.k2;
        default: return m.kt[1] * m.kt[2] / m.k2;
    }
}

// omega(k) -> delta_1(k) in place (eq. 6)
__global__ void ic_delta1_kernel(IcGeom g, float2 *w)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.nk; i += (long long)gridDim.x * blockDim.x) {
        const float t = (float)ic_transfer(g, ic_mode(g, i).k2);
        const float2 v = w[i];
        w[i] = make_float2(t * v.x, t * v.y);
    }
}
// dst = scale * (i kt_d / k^2) src : the spectrum of -d/dq_d of the potential sourced by src (eq. 3-4)
__global__ void ic_grad_kernel(IcGeom g, const float2 *__restrict__ src, int d, double scale, float2 *__restrict__ dst)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.nk; i += (long long)gridDim.x * blockDim.x) {
        const IcMode m = ic_mode(g, i);
        const float c = m.k2 > 0.0 ? (float)(scale * m.kt[d] / m.k2) : 0.f;
        const float2 v = src[i];
        dst[i] = make_float2(-c * v.y, c * v.x);
    }
}
// dst = scale * (k_a k_b / k^2) src : the spectrum of phi_1,ab (eq. 4)
__global__ void ic_hess_kernel(IcGeom g, const float2 *__restrict__ src, int ab, double scale, float2 *__restrict__ dst)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.nk; i += (long long)gridDim.x * blockDim.x) {
        const float c = (float)(scale * ic_hess(ic_mode(g, i), ab));
        const float2 v = src[i];
        dst[i] = make_float2(c * v.x, c * v.y);
    }
}
// transposes, accumulated: acc += (-i kt_d / k^2) src   /   acc += (k_a k_b / k^2) src
__global__ void ic_gradT_acc_kernel(IcGeom g, const float2 *__restrict__ src, int d, float2 *__restrict__ acc)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.nk; i += (long long)gridDim.x * blockDim.x) {
        const IcMode m = ic_mode(g, i);
        const float c = m.k2 > 0.0 ? (float)(m.kt[d] / m.k2) : 0.f;
        const float2 v = src[i];
        float2 a = acc[i];
        a.x += c * v.y;
        a.y -= c * v.x;
        acc[i] = a;
    }
}
__global__ void ic_hess_acc_kernel(IcGeom g, const float2 *__restrict__ src, int ab, float2 *__restrict__ acc)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.nk; i += (long long)gridDim.x * blockDim.x) {
        const float c = (float)ic_hess(ic_mode(g, i), ab);
        const float2 v = src[i];
        float2 a = acc[i];
        a.x += c * v.x;
        a.y += c * v.y;
        acc[i] = a;
    }
}
// w *= scale * amp sqrt(P)  (the transpose of eq. 6: real and even, its own transpose) or, with transfer == 0, w *= scale
__global__ void ic_scale_kernel(IcGeom g, float2 *w, double scale, int transfer)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.nk; i += (long long)gridDim.x * blockDim.x) {
        const float t = (float)(scale * (transfer ? ic_transfer(g, ic_mode(g, i).k2) : 1.0));
        const float2 v = w[i];
        w[i] = make_float2(t * v.x, t * v.y);
    }
}

// ---- real space, padded rows of 2 lzc floats -----------------------------------------------------------------------
#define IC_REAL_LOOP(g, j, o)                                                                                                 \
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x, o; j < (g).np; j += (long long)gridDim.x * blockDim.x) \
        if (o = (j / (g).L[2]) * (2 * (g).lzc) + (j % (g).L[2]), true)

// field <- cx * x[:, d] + cp * p[:, d]   (x == NULL: the scalar array p[j])
__global__ void ic_pack_kernel(IcGeom g, const float *__restrict__ x, const float *__restrict__ p, int d, double cx, double cp,
                               float *__restrict__ field)
{
    IC_REAL_LOOP(g, j, o) field[o] = x ? (float)(cx * (double)x[3 * j + d] + cp * (double)p[3 * j + d]) : p[j];
}
// s0[:, d] (+)= cs * field, p0[:, d] (+)= cp * field   (eq. 2)
__global__ void ic_accum_kernel(IcGeom g, const float *__restrict__ field, int d, double cs, double cp, int first,
                                float *__restrict__ s0, float *__restrict__ p0)
{
    IC_REAL_LOOP(g, j, o)
    {
        const double v = (double)field[o];
        s0[3 * j + d] = (float)((first ? 0.0 : (double)s0[3 * j + d]) + cs * v);
        p0[3 * j + d] = (float)((first ? 0.0 : (double)p0[3 * j + d]) + cp * v);
    }
}
// S = sum_{a<b} (phi_aa phi_bb - phi_ab^2) into f[0]   (eq. 4); f = xx yy zz xy xz yz
__global__ void ic_source_kernel(IcGeom g, float *f0, const float *f1, const float *f2, const float *f3, const float *f4, const float *f5)
{
    IC_REAL_LOOP(g, j, o)
    {
        const float xx = f0[o], yy = f1[o], zz = f2[o], xy = f3[o], xz = f4[o], yz = f5[o];
        f0[o] = xx * yy + xx * zz + yy * zz - xy * xy - xz * xz - yz * yz;
    }
}
// cotangents of the diagonal second derivatives, in place: xx <- Sbar (yy + zz), ...
__global__ void ic_phibar_diag_kernel(IcGeom g, float *fxx, float *fyy, float *fzz, const float *sbar)
{
    IC_REAL_LOOP(g, j, o)
    {
        const float xx = fxx[o], yy = fyy[o], zz = fzz[o], s = sbar[o];
        fxx[o] = s * (yy + zz);
        fyy[o] = s * (xx + zz);
        fzz[o] = s * (xx + yy);
    }
}
__global__ void ic_phibar_off_kernel(IcGeom g, float *fab, const float *sbar)
{
    IC_REAL_LOOP(g, j, o) fab[o] = -2.f * sbar[o] * fab[o];
}
__global__ void ic_unpad_kernel(IcGeom g, const float *__restrict__ field, float *__restrict__ out)
{
    IC_REAL_LOOP(g, j, o) out[j] = field[o];
}

// D2, D2' = dD2/dlna by integrating eq. A1 (both lines, in D, L520) with the initial conditions A3 (L528) from a = 1e-6:
// RK4 in ln a.  (The oracle integrates the G form A5/A6 instead: two formulations, one answer.)
static void growth2_host(double om, double a, double out[2])
{
    auto rhs = [&](double lna, const double y[4], double dy[4]) {
        const double aa = std::exp(lna);
        const double E2 = om / (aa * aa * aa) + 1.0 - om;
        const double oma = om / (aa * aa * aa) / E2, hh = -1.5 * oma;
        dy[0] = y[1];
        dy[1] = -(2.0 + hh) * y[1] + 1.5 * oma * y[0];
        dy[2] = y[3];
        dy[3] = -(2.0 + hh) * y[3] + 1.5 * oma * y[2] + 1.5 * oma * y[0] * y[0];
    };
    const double ai = 1e-6, l0 = std::log(ai), l1 = std::log(a);
    long n = (long)std::ceil((l1 - l0) / 1e-3);
    if (n < 1) n = 1;
    const double h = (l1 - l0) / (double)n;
    double y[4] = {ai, ai, 3.0 / 7.0 * ai * ai, 6.0 / 7.0 * ai * ai};
    for (long i = 0; i < n; i++) {
        const double t = l0 + h * (double)i;
        double k1[4], k2[4], k3[4], k4[4], yt[4];
        rhs(t, y, k1);
        for (int c = 0; c < 4; c++) yt[c] = y[c] + 0.5 * h * k1[c];
        rhs(t + 0.5 * h, yt, k2);
        for (int c = 0; c < 4; c++) yt[c] = y[c] + 0.5 * h * k2[c];
        rhs(t + 0.5 * h, yt, k3);
        for (int c = 0; c < 4; c++) yt[c] = y[c] + h * k3[c];
        rhs(t + h, yt, k4);
        for (int c = 0; c < 4; c++) y[c] += h / 6.0 * (k1[c] + 2.0 * k2[c] + 2.0 * k3[c] + k4[c]);
    }
    out[0] = y[2];
    out[1] = y[3];
}

// {D1, D2, a^2 E D1', a^2 E D2'}: the four time factors of eq. 2
void ic_factors_host(double om, double a0, double out[4])
{
    double g1[4], g2[2];
    growth_host(om, a0, g1);
    growth2_host(om, a0, g2);
    const double a2E = a0 * a0 * std::sqrt(om / (a0 * a0 * a0) + 1.0 - om);
    out[0] = g1[0];
    out[1] = g2[0];
    out[2] = g1[2];          // G_D = a^2 E D1'
    out[3] = a2E * g2[1];
}

struct IcRun {
    pm_ctx *c;
    IcGeom g;
    size_t fstride;   // floats per lattice field
    float *F[7];
    cudaStream_t st;
};

static int ic_setup(pm_ctx *c, double amp, double ns, double rc, int order, IcRun *r)
{
    const Geometry &g = c->g;
    if (order != 1 && order != 2) return fail(c, PM_EINVAL, "pm_ic", "order must be 1 or 2");
    if (c->a.empty()) return fail(c, PM_ESTATE, "pm_ic", "the ctx has no scale factors (a_0 is needed)");
    if (!(amp >= 0.0) || !std::isfinite(ns) || !(rc >= 0.0)) return fail(c, PM_EINVAL, "pm_ic", "amp, ns, rc");
    IcGeom &q = r->g;
    for (int d = 0; d < 3; d++) { q.L[d] = g.L[d]; q.N[d] = g.N[d]; }
    q.lzc = g.L[2] / 2 + 1;
    q.nk = (long long)g.L[0] * g.L[1] * q.lzc;
    q.np = g.np;
    q.amp = amp; q.ns = ns; q.rc = rc;
    r->c = c;
    r->st = c->stream;
    r->fstride = ((size_t)q.nk * 2 + 63) / 64 * 64;
    if (r->fstride * 7 > (size_t)g.mesh_stride * 7) return fail(c, PM_EWORKSPACE, "pm_ic", "lattice fields do not fit the mesh buffers (lattice larger than the mesh)");
    for (int k = 0; k < 7; k++) r->F[k] = c->mesh[0] + (size_t)k * r->fstride;
    if (!c->plans_ic_ok) {
        long long n[3] = {g.L[0], g.L[1], g.L[2]};
        long long rembed[3] = {g.L[0], g.L[1], 2 * q.lzc}, cembed[3] = {g.L[0], g.L[1], q.lzc};
        size_t ws = 0, need = 0;
        PM_ICFFT(c, cufftCreate(&c->plan_ic_r2c));
        PM_ICFFT(c, cufftCreate(&c->plan_ic_c2r));
        c->plans_ic_ok = true;
        PM_ICFFT(c, cufftSetAutoAllocation(c->plan_ic_r2c, 0));
        PM_ICFFT(c, cufftSetAutoAllocation(c->plan_ic_c2r, 0));
        PM_ICFFT(c, cufftMakePlanMany64(c->plan_ic_r2c, 3, n, rembed, 1, (long long)r->fstride, cembed, 1, (long long)r->fstride / 2, CUFFT_R2C, 1, &ws));
        need = ws;
        PM_ICFFT(c, cufftMakePlanMany64(c->plan_ic_c2r, 3, n, cembed, 1, (long long)r->fstride / 2, rembed, 1, (long long)r->fstride, CUFFT_C2R, 1, &ws));
        if (ws > need) need = ws;
        if (need > c->fft_work_bytes) return fail(c, PM_EWORKSPACE, "pm_ic", "cuFFT work area of the lattice plans exceeds the reserve");
        PM_ICFFT(c, cufftSetWorkArea(c->plan_ic_r2c, c->fft_work));
        PM_ICFFT(c, cufftSetWorkArea(c->plan_ic_c2r, c->fft_work));
        PM_ICFFT(c, cufftSetStream(c->plan_ic_r2c, c->stream));
        PM_ICFFT(c, cufftSetStream(c->plan_ic_c2r, c->stream));
    }
    // the mesh buffers are scratch here: whatever state / sort / adjoint bookkeeping pointed into them is void
    c->t_index = -1;
    c->have_adjoint = false;
    return PM_OK;
}

void ic_destroy(pm_ctx *c)
{
    if (c->plans_ic_ok) {
        cufftDestroy(c->plan_ic_r2c);
        cufftDestroy(c->plan_ic_c2r);
        c->plans_ic_ok = false;
    }
}

#define IC_LAUNCH(r, kernel, n, ...)                                                 \
    do {                                                                             \
        (r).c->n_own++;                                                              \
        kernel<<<ic_grid(n), 256, 0, (r).st>>>((r).g, __VA_ARGS__);                  \
        PM_LAUNCH_CHECK((r).c, #kernel);                                             \
    } while (0)
static int ic_r2c(IcRun &r, float *f)
{
    r.c->n_fft++;
    PM_ICFFT(r.c, cufftExecR2C(r.c->plan_ic_r2c, f, (cufftComplex *)f));
    return PM_OK;
}
static int ic_c2r(IcRun &r, float *f)
{
    r.c->n_fft++;
    PM_ICFFT(r.c, cufftExecC2R(r.c->plan_ic_c2r, (cufftComplex *)f, f));
    return PM_OK;
}

// F[0] <- delta_1(k) of the white noise omega
static int ic_delta1(IcRun &r, const float *dev_omega)
{
    IC_LAUNCH(r, ic_pack_kernel, r.g.np, (const float *)nullptr, dev_omega, 0, 0.0, 0.0, r.F[0]);
    PM_TRY(ic_r2c(r, r.F[0]));
    IC_LAUNCH(r, ic_delta1_kernel, r.g.nk, (float2 *)r.F[0]);
    return PM_OK;
}

int ic_forward(pm_ctx *c, const float *dev_omega, double amp, double ns, double rc, int order, float *dev_s0, float *dev_p0)
{
    IcRun r;
    PM_TRY(ic_setup(c, amp, ns, rc, order, &r));
    double f[4];
    ic_factors_host(c->prm.omega_m, c->a[0], f);
    const double inv_np = 1.0 / (double)r.g.np;
    PM_TRY(ic_delta1(r, dev_omega));
    for (int d = 0; d < 3; d++) {                                                    // s1 = -grad phi_1 (eq. 3)
        IC_LAUNCH(r, ic_grad_kernel, r.g.nk, (const float2 *)r.F[0], d, inv_np, (float2 *)r.F[1]);
        PM_TRY(ic_c2r(r, r.F[1]));
        IC_LAUNCH(r, ic_accum_kernel, r.g.np, (const float *)r.F[1], d, f[0], f[2], 1, dev_s0, dev_p0);
    }
    if (order == 2) {
        for (int ab = 0; ab < 6; ab++) {                                             // phi_1,ab
            IC_LAUNCH(r, ic_hess_kernel, r.g.nk, (const float2 *)r.F[0], ab, inv_np, (float2 *)r.F[1 + ab]);
            PM_TRY(ic_c2r(r, r.F[1 + ab]));
        }
        IC_LAUNCH(r, ic_source_kernel, r.g.np, r.F[1], (const float *)r.F[2], (const float *)r.F[3], (const float *)r.F[4],
                  (const float *)r.F[5], (const float *)r.F[6]);                     // eq. 4, second line
        PM_TRY(ic_r2c(r, r.F[1]));
        for (int d = 0; d < 3; d++) {                                                // s2 = -grad phi_2
            IC_LAUNCH(r, ic_grad_kernel, r.g.nk, (const float2 *)r.F[1], d, inv_np, (float2 *)r.F[2]);
            PM_TRY(ic_c2r(r, r.F[2]));
            IC_LAUNCH(r, ic_accum_kernel, r.g.np, (const float *)r.F[2], d, f[1], f[3], 0, dev_s0, dev_p0);
        }
    }
    return PM_OK;
}

int ic_vjp(pm_ctx *c, const float *dev_omega, double amp, double ns, double rc, int order, const float *dev_xi0,
           const float *dev_pi0, float *dev_domega)
{
    IcRun r;
    PM_TRY(ic_setup(c, amp, ns, rc, order, &r));
    double f[4];
    ic_factors_host(c->prm.omega_m, c->a[0], f);
    const double inv_np = 1.0 / (double)r.g.np;
    float *dbar = r.F[5];                                                            // delta_1bar(k)
    PM_CUDA(c, cudaMemsetAsync(dbar, 0, sizeof(float) * r.fstride, r.st));
    for (int d = 0; d < 3; d++) {                                                    // through s1: c1 = D1 xi + (a^2 E D1') pi
        IC_LAUNCH(r, ic_pack_kernel, r.g.np, dev_xi0, dev_pi0, d, f[0], f[2], r.F[1]);
        PM_TRY(ic_r2c(r, r.F[1]));
        IC_LAUNCH(r, ic_gradT_acc_kernel, r.g.nk, (const float2 *)r.F[1], d, (float2 *)dbar);
    }
    if (order == 2) {
        PM_TRY(ic_delta1(r, dev_omega));                                             // the forward pass's delta_1(k) again
        float *sbar = r.F[2];
        PM_CUDA(c, cudaMemsetAsync(sbar, 0, sizeof(float) * r.fstride, r.st));
        for (int d = 0; d < 3; d++) {                                                // through s2: c2 = D2 xi + (a^2 E D2') pi
            IC_LAUNCH(r, ic_pack_kernel, r.g.np, dev_xi0, dev_pi0, d, f[1], f[3], r.F[1]);
            PM_TRY(ic_r2c(r, r.F[1]));
            IC_LAUNCH(r, ic_gradT_acc_kernel, r.g.nk, (const float2 *)r.F[1], d, (float2 *)sbar);
        }
        IC_LAUNCH(r, ic_scale_kernel, r.g.nk, (float2 *)sbar, inv_np, 0);
        PM_TRY(ic_c2r(r, sbar));                                                     // Sbar(q)
        float *diag[3] = {r.F[1], r.F[3], r.F[4]};
        for (int a = 0; a < 3; a++) {
            IC_LAUNCH(r, ic_hess_kernel, r.g.nk, (const float2 *)r.F[0], a, inv_np, (float2 *)diag[a]);
            PM_TRY(ic_c2r(r, diag[a]));
        }
        IC_LAUNCH(r, ic_phibar_diag_kernel, r.g.np, diag[0], diag[1], diag[2], (const float *)sbar);
        for (int a = 0; a < 3; a++) {
            PM_TRY(ic_r2c(r, diag[a]));
            IC_LAUNCH(r, ic_hess_acc_kernel, r.g.nk, (const float2 *)diag[a], a, (float2 *)dbar);
        }
        for (int ab = 3; ab < 6; ab++) {
            IC_LAUNCH(r, ic_hess_kernel, r.g.nk, (const float2 *)r.F[0], ab, inv_np, (float2 *)r.F[1]);
            PM_TRY(ic_c2r(r, r.F[1]));
            IC_LAUNCH(r, ic_phibar_off_kernel, r.g.np, r.F[1], (const float *)sbar);
            PM_TRY(ic_r2c(r, r.F[1]));
            IC_LAUNCH(r, ic_hess_acc_kernel, r.g.nk, (const float2 *)r.F[1], ab, (float2 *)dbar);
        }
    }
    IC_LAUNCH(r, ic_scale_kernel, r.g.nk, (float2 *)dbar, inv_np, 1);               // transpose of eq. 6
    PM_TRY(ic_c2r(r, dbar));
    IC_LAUNCH(r, ic_unpad_kernel, r.g.np, (const float *)dbar, dev_domega);
    return PM_OK;
}

}  // namespace pm

extern "C" {

int pm_host_ic_factors(double omega_m, double a0, double out[4])
{
    if (!out || !(a0 > 0.0) || !(omega_m > 0.0) || omega_m > 1.0) return PM_EINVAL;
    pm::ic_factors_host(omega_m, a0, out);
    return PM_OK;
}

int pm_ic_fwd(pm_ctx *c, const float *dev_omega, double amp, double ns, double rc, int order, float *dev_s0, float *dev_p0)
{
    if (!c) return PM_EINVAL;
    if (!dev_omega || !dev_s0 || !dev_p0 || (((uintptr_t)dev_omega | (uintptr_t)dev_s0 | (uintptr_t)dev_p0) & 3))
        return pm::fail(c, PM_EINVAL, "pm_ic_fwd", "NULL or misaligned pointer");
    return pm::ic_forward(c, dev_omega, amp, ns, rc, order, dev_s0, dev_p0);
}

int pm_ic_vjp(pm_ctx *c, const float *dev_omega, double amp, double ns, double rc, int order, const float *dev_xi0,
              const float *dev_pi0, float *dev_domega)
{
    if (!c) return PM_EINVAL;
    if (!dev_omega || !dev_xi0 || !dev_pi0 || !dev_domega ||
        (((uintptr_t)dev_omega | (uintptr_t)dev_xi0 | (uintptr_t)dev_pi0 | (uintptr_t)dev_domega) & 3))
        return pm::fail(c, PM_EINVAL, "pm_ic_vjp", "NULL or misaligned pointer");
    return pm::ic_vjp(c, dev_omega, amp, ns, rc, order, dev_xi0, dev_pi0, dev_domega);
}

}  // extern "C"
