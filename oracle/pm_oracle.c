/*
 * pm_oracle.c -- CPU fp64 ORACLE for the adjoint particle-mesh hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or helper with the CUDA library in
 * paper_2211_09815_b200/csrc/, and neither side includes or imports the other.
 *
 * It is written from /root/reference/PAPER.md ("Differentiable Cosmological Simulation
 * with the Adjoint Method", arxiv 2211.09815) and follows the paper's algorithm step by
 * step, in the paper's order and notation, in double precision.  No blocking, fusion or
 * reordering: every routine is the plain definition with a loop around it.  The only
 * parallelism is an OpenMP "parallel for" over independent particles / FFT lines;
 * the scatter loop is serial so that the result is deterministic.
 *
 * Units (reading R1): length = one mesh cell (l = 1 in eq. 10), time = 1/H0.
 * Decoded symbols (the PDF extraction prints three things as "alpha", R2):
 *   a     scale factor,   acc = -grad(varphi) the particle acceleration (eq. 16),
 *   alpha = -pi . d grad(varphi)/dx the force VJP (eq. 49),  xi = dJ/dx,  pi = dJ/dp.
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): P1 mass conservation, P2 transpose
 * identity, P3/P4/P5 momentum conservation / lattice symmetry / translation, P6 FFT vs
 * direct DFT and numpy.fft, P7 EdS closed forms, P8 LCDM growth vs Heath integral, P9
 * Zel'dovich plane-wave growth, P10 reversibility, P11 finite-difference gradient,
 * P12 reverse-integrated adjoint == store-all backprop, P13 VJP duality, P14 J = 0 case.
 * Every function here is covered by at least one of them; nothing is "parity unpinned".
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;
static const double PI_ = 3.14159265358979323846264338327950288;

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------ */
/* 1. Growth (App. A; eq. A2, A5 first line, A6, A7, A8 with m = 1)   */
/* ------------------------------------------------------------------------------------ */

/* E^2(a) = H^2/H0^2 for flat matter + Lambda */
static double E2_of_a(double om, double a) { return om / (a * a * a) + 1.0 - om; }
/* Omega_m(a), eq. A2 (L524) */
static double Om_of_a(double om, double a) { return om / (a * a * a) / E2_of_a(om, a); }
/* H'/H = dlnH/dlna = -1.5 Omega_m(a) for flat matter + Lambda */
static double dlnH_of_a(double om, double a) { return -1.5 * Om_of_a(om, a); }

/* right-hand side of eq. A5 (first line, L537), y = (G1, G1'), ' = d/dlna */
static void growth_rhs(double om, double lna, const double y[2], double dy[2])
{
    double a = exp(lna);
    double hh = dlnH_of_a(om, a);
    dy[0] = y[1];
    dy[1] = -(4.0 + hh) * y[1] - (3.0 + hh - 1.5 * Om_of_a(om, a)) * y[0];
}

/* Integrate A5 from a_ini = 1e-6 (reading R4) with G1 = 1, G1' = 0 (A6, L541-545) by
 * fixed-step RK4 in ln a, step <= 1e-3.  out = {D1, D1', D1''} (' = d/dlna), eq. A8.  */
void orc_growth(double om, double a, double out[3])
{
    const double lna0 = log(1e-6), lna1 = log(a);
    long nstep = (long)ceil((lna1 - lna0) / 1e-3);
    if (nstep < 1) nstep = 1;
    double h = (lna1 - lna0) / (double)nstep;
    double y[2] = {1.0, 0.0};
    for (long i = 0; i < nstep; i++) {
        double t = lna0 + h * (double)i;
        double k1[2], k2[2], k3[2], k4[2], yt[2];
        growth_rhs(om, t, y, k1);
        yt[0] = y[0] + 0.5 * h * k1[0]; yt[1] = y[1] + 0.5 * h * k1[1];
        growth_rhs(om, t + 0.5 * h, yt, k2);
        yt[0] = y[0] + 0.5 * h * k2[0]; yt[1] = y[1] + 0.5 * h * k2[1];
        growth_rhs(om, t + 0.5 * h, yt, k3);
        yt[0] = y[0] + h * k3[0]; yt[1] = y[1] + h * k3[1];
        growth_rhs(om, t + h, yt, k4);
        y[0] += h / 6.0 * (k1[0] + 2.0 * k2[0] + 2.0 * k3[0] + k4[0]);
        y[1] += h / 6.0 * (k1[1] + 2.0 * k2[1] + 2.0 * k3[1] + k4[1]);
    }
    double dy[2];
    growth_rhs(om, lna1, y, dy);
    double G = y[0], Gp = y[1], Gpp = dy[1];
    out[0] = a * G;                    /* D1   = a G1                         (A8) */
    out[1] = a * (G + Gp);             /* D1'  = a (G1 + G1')                 (A8) */
    out[2] = a * (G + 2.0 * Gp + Gpp); /* D1'' = a (G1 + 2 G1' + G1'')        (A8) */
}

/* eq. A7 (L551), H0 = 1:  G_D = a^2 H D1',  G_K = a^3 H^2 [D1'' + (2 + H'/H) D1']     */
void orc_GD_GK(double om, double a, double out[2])
{
    double g[3];
    orc_growth(om, a, g);
    double E2 = E2_of_a(om, a);
    out[0] = a * a * sqrt(E2) * g[1];
    out[1] = a * a * a * E2 * (g[2] + (2.0 + dlnH_of_a(om, a)) * g[1]);
}

/* eq. 15 (L165): D(tc, ta, tb) = (D1(tb) - D1(ta)) / G_D(tc)                           */
double orc_drift_factor(double om, double ac, double aa, double ab)
{
    double gb[3], ga[3], gc[2];
    orc_growth(om, ab, gb);
    orc_growth(om, aa, ga);
    orc_GD_GK(om, ac, gc);
    return (gb[0] - ga[0]) / gc[0];
}

/* eq. 15 (L167): K(tc, ta, tb) = (G_D(tb) - G_D(ta)) / G_K(tc)                         */
double orc_kick_factor(double om, double ac, double aa, double ab)
{
    double gb[2], ga[2], gc[2];
    orc_GD_GK(om, ab, gb);
    orc_GD_GK(om, aa, ga);
    orc_GD_GK(om, ac, gc);
    return (gb[0] - ga[0]) / gc[1];
}

/* ------------------------------------------------------------------------------------ */
/* 2. FFT: the definition  X(k) = sum_g x(g) exp(sign * i k.g)  (forward    */
/*    sign = -1), unnormalised, any length (mixed radix; prime lengths by the direct sum) */
/* ------------------------------------------------------------------------------------ */

static int smallest_factor(int n)
{
    for (int p = 2; p * p <= n; p++)
        if (n % p == 0) return p;
    return n;
}

/* y[k] = sum_j x[j*s] w_n^{jk},  w_n^j = w[(j mod n) * (wn/n)],  w has wn entries       */
static void dft_rec(int n, const cplx *x, int s, cplx *y, const cplx *w, int wn)
{
    if (n == 1) { y[0] = x[0]; return; }
    int p = smallest_factor(n), m = n / p, ws = wn / n;
    if (p == n || p > 64) { /* prime length (or a factor too large for the butterfly buffers): direct sum */
        for (int k = 0; k < n; k++) {
            cplx acc = 0.0;
            for (int j = 0; j < n; j++) acc += x[(size_t)j * s] * w[(size_t)(((long)j * k) % n) * ws];
            y[k] = acc;
        }
        return;
    }
    /* Cooley-Tukey: p transforms of length m over the residues r (mod p) ...            */
    for (int r = 0; r < p; r++) dft_rec(m, x + (size_t)r * s, s * p, y + (size_t)r * m, w, wn);
    /* ... combined by  X[k + q m] = sum_r w_n^{r (k + q m)} Y_r[k]                      */
    cplx t[64], o[64];
    for (int k = 0; k < m; k++) {
        for (int r = 0; r < p; r++) t[r] = y[(size_t)r * m + k] * w[(size_t)(((long)r * k) % n) * ws];
        for (int q = 0; q < p; q++) {
            cplx acc = 0.0;
            for (int r = 0; r < p; r++) acc += t[r] * w[(size_t)(((long)r * q * m) % n) * ws];
            o[q] = acc;
        }
        for (int q = 0; q < p; q++) y[(size_t)q * m + k] = o[q];
    }
}

static cplx *twiddles(int n, int sign)
{
    cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    for (int j = 0; j < n; j++) {
        double ang = (double)sign * 2.0 * PI_ * (double)j / (double)n;
        w[j] = cos(ang) + I * sin(ang);
    }
    return w;
}

/* 1-D transform of `count` lines of length n; line l starts at base + l-dependent offset */
void orc_fft1d(int n, cplx *x, int sign)
{
    cplx *w = twiddles(n, sign);
    cplx *y = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    dft_rec(n, x, 1, y, w, n);
    memcpy(x, y, sizeof(cplx) * (size_t)n);
    free(y); free(w);
}

/* in-place 3-D transform of data[nx][ny][nz] (row-major), unnormalised                  */
void orc_fft3d(int nx, int ny, int nz, cplx *data, int sign)
{
    cplx *wx = twiddles(nx, sign), *wy = twiddles(ny, sign), *wz = twiddles(nz, sign);
    int nmax = nx > ny ? nx : ny; if (nz > nmax) nmax = nz;
#pragma omp parallel
    {
        cplx *in = (cplx *)malloc(sizeof(cplx) * (size_t)nmax);
        cplx *out = (cplx *)malloc(sizeof(cplx) * (size_t)nmax);
        /* along z (contiguous) */
#pragma omp for schedule(static)
        for (long l = 0; l < (long)nx * ny; l++) {
            cplx *p = data + (size_t)l * nz;
            dft_rec(nz, p, 1, out, wz, nz);
            memcpy(p, out, sizeof(cplx) * (size_t)nz);
        }
        /* along y (stride nz) */
#pragma omp for schedule(static)
        for (long l = 0; l < (long)nx * nz; l++) {
            long ix = l / nz, iz = l % nz;
            cplx *p = data + (size_t)ix * ny * nz + iz;
            for (int j = 0; j < ny; j++) in[j] = p[(size_t)j * nz];
            dft_rec(ny, in, 1, out, wy, ny);
            for (int j = 0; j < ny; j++) p[(size_t)j * nz] = out[j];
        }
        /* along x (stride ny*nz) */
#pragma omp for schedule(static)
        for (long l = 0; l < (long)ny * nz; l++) {
            cplx *p = data + l;
            for (int j = 0; j < nx; j++) in[j] = p[(size_t)j * ny * nz];
            dft_rec(nx, in, 1, out, wx, nx);
            for (int j = 0; j < nx; j++) p[(size_t)j * ny * nz] = out[j];
        }
        free(in); free(out);
    }
    free(wx); free(wy); free(wz);
}

/* ------------------------------------------------------------------------------------ */
/* 3. Cloud-in-cell (eq. 10, l = 1; L133 "same grid points, same       */
/*    weights").  Mesh point g sits at coordinate g (reading R6); periodic.              */
/*    Cell i_d = floor(x_d), t_d = x_d - i_d in [0,1): weight (1 - t_d) at i_d mod N_d   */
/*    and t_d at (i_d + 1) mod N_d (reading R7: floor convention, right derivative).     */
/* ------------------------------------------------------------------------------------ */

static inline long wrap(long i, long n) { long r = i % n; return r < 0 ? r + n : r; }

/* the 8 mesh points of particle x[3]: flat index, weight W, and dW/dx_e (e = 0,1,2)     */
static inline void cic8(const int N[3], const double x[3], size_t idx[8], double W[8], double dW[8][3])
{
    long i0[3]; double t[3];
    for (int d = 0; d < 3; d++) { double f = floor(x[d]); i0[d] = (long)f; t[d] = x[d] - f; }
    int c = 0;
    for (int bx = 0; bx < 2; bx++)
        for (int by = 0; by < 2; by++)
            for (int bz = 0; bz < 2; bz++, c++) {
                int b[3] = {bx, by, bz};
                double w1[3], g1[3];
                long g[3];
                for (int d = 0; d < 3; d++) {
                    w1[d] = b[d] ? t[d] : 1.0 - t[d];   /* max(1 - |g - x|, 0) at the two nearest points */
                    g1[d] = b[d] ? 1.0 : -1.0;          /* its derivative with respect to x_d            */
                    g[d] = wrap(i0[d] + b[d], N[d]);
                }
                idx[c] = ((size_t)g[0] * N[1] + g[1]) * N[2] + g[2];
                W[c] = w1[0] * w1[1] * w1[2];
                dW[c][0] = g1[0] * w1[1] * w1[2];
                dW[c][1] = w1[0] * g1[1] * w1[2];
                dW[c][2] = w1[0] * w1[1] * g1[2];
            }
}

/* scatter:  mesh_c(g) = sum_j val_{j,c} W(g, x_j);  val == NULL means unit mass, C = 1. */
/* mesh[C][Nx][Ny][Nz] is OVERWRITTEN.  Serial loop: deterministic.                      */
void orc_scatter(const int N[3], long np, const double *x, const double *val, int C, double *mesh)
{
    size_t Ng = (size_t)N[0] * N[1] * N[2];
    memset(mesh, 0, sizeof(double) * Ng * (size_t)C);
    for (long j = 0; j < np; j++) {
        size_t idx[8]; double W[8], dW[8][3];
        cic8(N, x + 3 * j, idx, W, dW);
        for (int c = 0; c < C; c++) {
            double v = val ? val[(size_t)j * C + c] : 1.0;
            for (int k = 0; k < 8; k++) mesh[(size_t)c * Ng + idx[k]] += v * W[k];
        }
    }
}

/* gather:  out_{j,c} = sum_g W(g, x_j) mesh_c(g)                                        */
void orc_gather(const int N[3], long np, const double *x, const double *mesh, int C, double *out)
{
    size_t Ng = (size_t)N[0] * N[1] * N[2];
#pragma omp parallel for schedule(static)
    for (long j = 0; j < np; j++) {
        size_t idx[8]; double W[8], dW[8][3];
        cic8(N, x + 3 * j, idx, W, dW);
        for (int c = 0; c < C; c++) {
            double acc = 0.0;
            for (int k = 0; k < 8; k++) acc += W[k] * mesh[(size_t)c * Ng + idx[k]];
            out[(size_t)j * C + c] = acc;
        }
    }
}

/* weight-gradient gather (the position VJP of both scatter and gather, L410):           */
/*   out_{j,e} = sum_c cot_{j,c} sum_g dW(g, x_j)/dx_e mesh_c(g);  cot == NULL means 1.  */
void orc_gather_grad(const int N[3], long np, const double *x, const double *mesh, int C,
                     const double *cot, double *out)
{
    size_t Ng = (size_t)N[0] * N[1] * N[2];
#pragma omp parallel for schedule(static)
    for (long j = 0; j < np; j++) {
        size_t idx[8]; double W[8], dW[8][3];
        cic8(N, x + 3 * j, idx, W, dW);
        double acc[3] = {0.0, 0.0, 0.0};
        for (int c = 0; c < C; c++) {
            double v = cot ? cot[(size_t)j * C + c] : 1.0;
            for (int k = 0; k < 8; k++)
                for (int e = 0; e < 3; e++) acc[e] += v * dW[k][e] * mesh[(size_t)c * Ng + idx[k]];
        }
        for (int e = 0; e < 3; e++) out[3 * j + e] = acc[e];
    }
}

/* ------------------------------------------------------------------------------------ */
/* 4. Force on the mesh (eq. 9 and 11; "1 forward and 3 inverse FFTs") */
/* ------------------------------------------------------------------------------------ */

/* signed integer mode m in [-N/2, N/2) of FFT index i */
static inline int mode_of(int i, int n) { return i < (n + 1) / 2 ? i : i - n; }

/* k-space pieces shared by the force and by its transpose:                              */
/*   k_d = 2 pi m_d / N_d;  k2 = |k|^2 (full, also on Nyquist planes);                   */
/*   kt_d = k_d except 0 on the Nyquist plane m_d = -N_d/2 (reading R10);                */
/*   dec = 1, or prod_e sinc(k_e/2)^-4 when deconvolve = 1 (reading R12, not in paper).  */
static inline void kvec(const int N[3], int deconv, int ix, int iy, int iz, double kt[3], double *k2, double *dec)
{
    int idx[3] = {ix, iy, iz};
    double kk = 0.0, dc = 1.0;
    for (int d = 0; d < 3; d++) {
        int m = mode_of(idx[d], N[d]);
        double k = 2.0 * PI_ * (double)m / (double)N[d];
        kk += k * k;
        kt[d] = (N[d] % 2 == 0 && m == -N[d] / 2) ? 0.0 : k;
        if (deconv && m != 0) {
            double h = 0.5 * k, s = sin(h) / h;
            dc /= (s * s) * (s * s);
        }
    }
    *k2 = kk; *dec = dc;
}

/* rho[Ng] (mass per mesh point) -> f[3][Ng] = -grad varphi on the mesh:                 */
/*   delta = rho/nbar - 1 (L79);  varphi(k) = -1.5 Om delta(k)/k^2, varphi(0) = 0 (eq.11) */
/*   f_d(k) = -i kt_d varphi(k) (L131);  f_d(g) = (1/Ng) sum_k f_d(k) e^{+ik.g}          */
/* If imag_max != NULL it receives max |Im f_d(g)| (must be rounding-level, reading R10). */
void orc_force_mesh(const int N[3], double om, int deconv, double nbar, const double *rho, double *f,
                    double *imag_max)
{
    size_t Ng = (size_t)N[0] * N[1] * N[2];
    cplx *phi = (cplx *)malloc(sizeof(cplx) * Ng);
    cplx *buf = (cplx *)malloc(sizeof(cplx) * Ng);
    for (size_t g = 0; g < Ng; g++) phi[g] = rho[g] / nbar - 1.0;
    orc_fft3d(N[0], N[1], N[2], phi, -1);
#pragma omp parallel for schedule(static)
    for (long ix = 0; ix < N[0]; ix++)
        for (int iy = 0; iy < N[1]; iy++)
            for (int iz = 0; iz < N[2]; iz++) {
                double kt[3], k2, dec;
                kvec(N, deconv, (int)ix, iy, iz, kt, &k2, &dec);
                size_t g = ((size_t)ix * N[1] + iy) * N[2] + iz;
                phi[g] = (k2 == 0.0) ? 0.0 : -1.5 * om * dec * phi[g] / k2;
            }
    double im = 0.0;
    for (int d = 0; d < 3; d++) {
#pragma omp parallel for schedule(static)
        for (long ix = 0; ix < N[0]; ix++)
            for (int iy = 0; iy < N[1]; iy++)
                for (int iz = 0; iz < N[2]; iz++) {
                    double kt[3], k2, dec;
                    kvec(N, deconv, (int)ix, iy, iz, kt, &k2, &dec);
                    size_t g = ((size_t)ix * N[1] + iy) * N[2] + iz;
                    buf[g] = -I * kt[d] * phi[g];
                }
        orc_fft3d(N[0], N[1], N[2], buf, +1);
        for (size_t g = 0; g < Ng; g++) {
            f[(size_t)d * Ng + g] = creal(buf[g]) / (double)Ng;
            double ai = fabs(cimag(buf[g])) / (double)Ng;
            if (ai > im) im = ai;
        }
    }
    if (imag_max) *imag_max = im;
    free(phi); free(buf);
}

/* transpose of orc_force_mesh with respect to rho (term B):      */
/*   Pi[3][Ng] -> psi[Ng],  psi(k) = sum_d (+i kt_d)(-1.5 Om / k^2) Pi_d(k) / nbar        */
/* i.e. the conjugated kernel (c_d real and odd in real space), components summed; the   */
/* 1/nbar is d(delta)/d(rho).                                                            */
void orc_force_mesh_T(const int N[3], double om, int deconv, double nbar, const double *Pi, double *psi)
{
    size_t Ng = (size_t)N[0] * N[1] * N[2];
    cplx *acc = (cplx *)calloc(Ng, sizeof(cplx));
    cplx *buf = (cplx *)malloc(sizeof(cplx) * Ng);
    for (int d = 0; d < 3; d++) {
        for (size_t g = 0; g < Ng; g++) buf[g] = Pi[(size_t)d * Ng + g];
        orc_fft3d(N[0], N[1], N[2], buf, -1);
#pragma omp parallel for schedule(static)
        for (long ix = 0; ix < N[0]; ix++)
            for (int iy = 0; iy < N[1]; iy++)
                for (int iz = 0; iz < N[2]; iz++) {
                    double kt[3], k2, dec;
                    kvec(N, deconv, (int)ix, iy, iz, kt, &k2, &dec);
                    size_t g = ((size_t)ix * N[1] + iy) * N[2] + iz;
                    if (k2 != 0.0) acc[g] += (I * kt[d]) * (-1.5 * om * dec / k2) * buf[g] / nbar;
                }
    }
    orc_fft3d(N[0], N[1], N[2], acc, +1);
    for (size_t g = 0; g < Ng; g++) psi[g] = creal(acc[g]) / (double)Ng;
    free(acc); free(buf);
}

/* acc = F(x) (L111-133): scatter -> force mesh -> gather.  If fmesh != NULL the three    */
/* force meshes are also returned there ([3][Ng]).                                       */
void orc_force(const int N[3], double om, int deconv, long np, const double *x, double *acc, double *fmesh)
{
    size_t Ng = (size_t)N[0] * N[1] * N[2];
    double nbar = (double)np / (double)Ng;
    double *rho = (double *)malloc(sizeof(double) * Ng);
    double *f = fmesh ? fmesh : (double *)malloc(sizeof(double) * 3 * Ng);
    orc_scatter(N, np, x, NULL, 1, rho);
    orc_force_mesh(N, om, deconv, nbar, rho, f, NULL);
    orc_gather(N, np, x, f, 3, acc);
    free(rho);
    if (!fmesh) free(f);
}

/* Force VJP (paper: alpha = -pi . d grad(varphi)/dx, L393/L397; computed "by custom     */
/* VJPs of scatter and gather", L410; formula derived in DESIGN.md):                     */
/*   alpha_{j,e} = sum_{j',d} pi_{j',d} d acc_{j',d} / d x_{j,e} = A + B                 */
/*   A_{j,e} = sum_d pi_{j,d} sum_g dW(g,x_j)/dx_e f_d(g)          (through the gather)  */
/*   B_{j,e} = sum_g dW(g,x_j)/dx_e psi(g),  psi = force_mesh^T( scatter(x, pi) )        */
void orc_force_vjp(const int N[3], double om, int deconv, long np, const double *x, const double *pi,
                   double *alpha)
{
    size_t Ng = (size_t)N[0] * N[1] * N[2];
    double nbar = (double)np / (double)Ng;
    double *rho = (double *)malloc(sizeof(double) * Ng);
    double *f = (double *)malloc(sizeof(double) * 3 * Ng);
    double *Pi = (double *)malloc(sizeof(double) * 3 * Ng);
    double *psi = (double *)malloc(sizeof(double) * Ng);
    double *tmp = (double *)malloc(sizeof(double) * 3 * (size_t)np);
    /* force meshes at x */
    orc_scatter(N, np, x, NULL, 1, rho);
    orc_force_mesh(N, om, deconv, nbar, rho, f, NULL);
    /* term A: all three components d at once (cot = pi) */
    orc_gather_grad(N, np, x, f, 3, pi, alpha);
    /* Pi_d(g) = sum_j pi_{j,d} W(g, x_j) */
    orc_scatter(N, np, x, pi, 3, Pi);
    /* term B */
    orc_force_mesh_T(N, om, deconv, nbar, Pi, psi);
    orc_gather_grad(N, np, x, psi, 1, NULL, tmp);
    for (long j = 0; j < 3 * np; j++) alpha[j] += tmp[j];
    free(rho); free(f); free(Pi); free(psi); free(tmp);
}

/* ------------------------------------------------------------------------------------ */
/* 5. Lattice, objective                                                                  */
/* ------------------------------------------------------------------------------------ */

/* x_j = q_j + s_j (eq. 1); q_j = (jx, jy, jz) * (N/L): a Cartesian lattice (L45) whose   */
/* site 0 sits on mesh point 0 (reading R6); j = (jx*Ly + jy)*Lz + jz.  In every config N/L is  */
/* an integer (2), so q is on mesh points; a finer lattice (L > N) is allowed and used by P9.   */
void orc_positions(const int N[3], const int L[3], const double *s, double *x)
{
    long np = (long)L[0] * L[1] * L[2];
#pragma omp parallel for schedule(static)
    for (long j = 0; j < np; j++) {
        long jz = j % L[2], jy = (j / L[2]) % L[1], jx = j / ((long)L[1] * L[2]);
        x[3 * j + 0] = (double)jx * ((double)N[0] / (double)L[0]) + s[3 * j + 0];
        x[3 * j + 1] = (double)jy * ((double)N[1] / (double)L[1]) + s[3 * j + 1];
        x[3 * j + 2] = (double)jz * ((double)N[2] / (double)L[2]) + s[3 * j + 2];
    }
}

/* Objective (configs; "MSE ... on their density fields"; reading R17):     */
/*   r = rho/nbar - 1 - delta_target;  J = 1/2 sum_g r^2;                                 */
/*   xi_j = dJ/dx_j = (1/nbar) sum_g dW(g,x_j)/dx r(g)  (scatter VJP, L410)               */
double orc_objective(const int N[3], long np, const double *x, const double *delta_target, double *xi)
{
    size_t Ng = (size_t)N[0] * N[1] * N[2];
    double nbar = (double)np / (double)Ng;
    double *r = (double *)malloc(sizeof(double) * Ng);
    orc_scatter(N, np, x, NULL, 1, r);
    double J = 0.0;
    for (size_t g = 0; g < Ng; g++) {
        r[g] = r[g] / nbar - 1.0 - delta_target[g];
        J += 0.5 * r[g] * r[g];
    }
    if (xi) {
        orc_gather_grad(N, np, x, r, 1, NULL, xi);
        for (long j = 0; j < 3 * np; j++) xi[j] /= nbar;
    }
    free(r);
    return J;
}

/* ------------------------------------------------------------------------------------ */
/* 6. Time integration                                                                    */
/* ------------------------------------------------------------------------------------ */

/* half-step scale factor (reading R3): a_{i-1/2} = (a_{i-1} + a_i)/2                     */
static double a_half(const double *a, int i) { return 0.5 * (a[i - 1] + a[i]); }

static void force_at(const int N[3], const int L[3], double om, int deconv, const double *s, double *acc)
{
    long np = (long)L[0] * L[1] * L[2];
    double *x = (double *)malloc(sizeof(double) * 3 * (size_t)np);
    orc_positions(N, L, s, x);
    orc_force(N, om, deconv, np, x, acc, NULL);
    free(x);
}

static void vjp_at(const int N[3], const int L[3], double om, int deconv, const double *s, const double *pi,
                   double *alpha)
{
    long np = (long)L[0] * L[1] * L[2];
    double *x = (double *)malloc(sizeof(double) * 3 * (size_t)np);
    orc_positions(N, L, s, x);
    orc_force_vjp(N, om, deconv, np, x, pi, alpha);
    free(x);
}

/* acc_0 = F(x_0)  ("initialize acc_0 with F_0 before the first time step", L175)         */
void orc_init_acc(const int N[3], const int L[3], double om, int deconv, const double *s, double *acc)
{
    force_at(N, L, om, deconv, s, acc);
}

/* One forward KDK step t_{i-1} -> t_i, eq. 16 (L172), state (s, p, acc) updated in place: */
/*   K: p += acc K(t_{i-1}, t_{i-1}, t_{i-1/2});  D: s += p D(t_{i-1/2}, t_{i-1}, t_i);    */
/*   F: acc = F(q + s);                            K: p += acc K(t_i, t_{i-1/2}, t_i)      */
void orc_step_fwd(const int N[3], const int L[3], double om, int deconv, const double *a, int i,
                  double *s, double *p, double *acc)
{
    long n3 = 3L * L[0] * L[1] * L[2];
    double ah = a_half(a, i);
    double K1 = orc_kick_factor(om, a[i - 1], a[i - 1], ah);
    double D = orc_drift_factor(om, ah, a[i - 1], a[i]);
    double K2 = orc_kick_factor(om, a[i], ah, a[i]);
    for (long j = 0; j < n3; j++) p[j] += acc[j] * K1;
    for (long j = 0; j < n3; j++) s[j] += p[j] * D;
    force_at(N, L, om, deconv, s, acc);
    for (long j = 0; j < n3; j++) p[j] += acc[j] * K2;
}

/* One adjoint step t_i -> t_{i-1} with reverse-time integration, eq. 49 (L393), in place: */
/*   K_i^{i-1/2}:  p += acc K';  xi -= alpha K'          K' = K(t_i, t_i, t_{i-1/2})        */
/*   D_i^{i-1}:    s += p D';    pi -= xi D'             D' = D(t_{i-1/2}, t_i, t_{i-1})    */
/*   F_{i-1}:      acc = F(q + s);  alpha = VJP(q + s, pi)                                  */
/*   K_{i-1/2}^{i-1}: p += acc K''; xi -= alpha K''      K'' = K(t_{i-1}, t_{i-1/2}, t_{i-1}) */
/*   O_{i-1}: nothing to add for a final-state objective (L369).                            */
void orc_step_adj(const int N[3], const int L[3], double om, int deconv, const double *a, int i,
                  double *s, double *p, double *acc, double *xi, double *pi, double *alpha)
{
    long n3 = 3L * L[0] * L[1] * L[2];
    double ah = a_half(a, i);
    double K1 = orc_kick_factor(om, a[i], a[i], ah);
    double D = orc_drift_factor(om, ah, a[i], a[i - 1]);
    double K2 = orc_kick_factor(om, a[i - 1], ah, a[i - 1]);
    for (long j = 0; j < n3; j++) { p[j] += acc[j] * K1; xi[j] -= alpha[j] * K1; }
    for (long j = 0; j < n3; j++) { s[j] += p[j] * D; pi[j] -= xi[j] * D; }
    force_at(N, L, om, deconv, s, acc);
    vjp_at(N, L, om, deconv, s, pi, alpha);
    for (long j = 0; j < n3; j++) { p[j] += acc[j] * K2; xi[j] -= alpha[j] * K2; }
}

/* Whole run (eq. 16, 50, 49, 51).  All arrays [np][3] doubles.         */
/* in:  s0, p0, delta_target[Ng]                                                           */
/* out: s_n, p_n (final state), J, xi0, pi0, dJ_ds0 = xi0 + pi0 G_D(a0)/D1(a0)             */
/*      (eq. 51's dJ/domega chain restricted to Zel'dovich ICs, reading R18),              */
/*      s_rec, p_rec = the state reconstructed at t_0 by the reverse integration (P10).    */
/* Any output pointer may be NULL.  n_adj < 0 runs all n adjoint steps; n_adj >= 0 runs    */
/* only that many (for bounded timing samples); outputs then refer to step n - n_adj.      */
double orc_run_fwd_adj(const int N[3], const int L[3], double om, int deconv, int n, const double *a,
                       const double *s0, const double *p0, const double *delta_target,
                       double *s_n, double *p_n, double *xi0, double *pi0, double *dJ_ds0,
                       double *s_rec, double *p_rec, int n_adj)
{
    long np = (long)L[0] * L[1] * L[2], n3 = 3 * np;
    double *s = (double *)malloc(sizeof(double) * n3), *p = (double *)malloc(sizeof(double) * n3);
    double *acc = (double *)malloc(sizeof(double) * n3), *x = (double *)malloc(sizeof(double) * n3);
    double *xi = (double *)malloc(sizeof(double) * n3), *pi = (double *)malloc(sizeof(double) * n3);
    double *alpha = (double *)malloc(sizeof(double) * n3);
    memcpy(s, s0, sizeof(double) * n3);
    memcpy(p, p0, sizeof(double) * n3);
    orc_init_acc(N, L, om, deconv, s, acc);
    for (int i = 1; i <= n; i++) orc_step_fwd(N, L, om, deconv, a, i, s, p, acc);
    if (s_n) memcpy(s_n, s, sizeof(double) * n3);
    if (p_n) memcpy(p_n, p, sizeof(double) * n3);
    /* eq. 50 (L397): xi_n = dJ/dx_n, pi_n = dJ/dp_n = 0, acc_n = F_n (already held),        */
    /* alpha_n = pi_n . dacc/dx = 0 because pi_n = 0.                                        */
    orc_positions(N, L, s, x);
    double J = orc_objective(N, np, x, delta_target, xi);
    for (long j = 0; j < n3; j++) { pi[j] = 0.0; alpha[j] = 0.0; }
    int last = (n_adj < 0) ? 1 : n - n_adj + 1;
    for (int i = n; i >= last; i--) orc_step_adj(N, L, om, deconv, a, i, s, p, acc, xi, pi, alpha);
    if (xi0) memcpy(xi0, xi, sizeof(double) * n3);
    if (pi0) memcpy(pi0, pi, sizeof(double) * n3);
    if (dJ_ds0) {
        double g[3], gd[2];
        orc_growth(om, a[0], g);
        orc_GD_GK(om, a[0], gd);
        for (long j = 0; j < n3; j++) dJ_ds0[j] = xi[j] + pi[j] * gd[0] / g[0];
    }
    if (s_rec) memcpy(s_rec, s, sizeof(double) * n3);
    if (p_rec) memcpy(p_rec, p, sizeof(double) * n3);
    free(s); free(p); free(acc); free(x); free(xi); free(pi); free(alpha);
    return J;
}

/* Forward only: final state and objective (used by finite differences, P11).              */
double orc_run_fwd(const int N[3], const int L[3], double om, int deconv, int n, const double *a,
                   const double *s0, const double *p0, const double *delta_target,
                   double *s_n, double *p_n)
{
    long np = (long)L[0] * L[1] * L[2], n3 = 3 * np;
    double *s = (double *)malloc(sizeof(double) * n3), *p = (double *)malloc(sizeof(double) * n3);
    double *acc = (double *)malloc(sizeof(double) * n3), *x = (double *)malloc(sizeof(double) * n3);
    memcpy(s, s0, sizeof(double) * n3);
    memcpy(p, p0, sizeof(double) * n3);
    orc_init_acc(N, L, om, deconv, s, acc);
    for (int i = 1; i <= n; i++) orc_step_fwd(N, L, om, deconv, a, i, s, p, acc);
    if (s_n) memcpy(s_n, s, sizeof(double) * n3);
    if (p_n) memcpy(p_n, p, sizeof(double) * n3);
    double J = 0.0;
    if (delta_target) {
        orc_positions(N, L, s, x);
        J = orc_objective(N, np, x, delta_target, NULL);
    }
    free(s); free(p); free(acc); free(x);
    return J;
}

/* Store-all backpropagation through eq. 16 (the "AD" side of PAPER.md L474: the same       */
/* discrete adjoint, eq. 47, but every x_i is taken from the saved forward history instead */
/* of being reconstructed by reverse integration).  Memory O(n); tiny inputs only (P12).   */
double orc_backprop_storeall(const int N[3], const int L[3], double om, int deconv, int n, const double *a,
                             const double *s0, const double *p0, const double *delta_target,
                             double *xi0, double *pi0)
{
    long np = (long)L[0] * L[1] * L[2], n3 = 3 * np;
    double *S = (double *)malloc(sizeof(double) * n3 * (size_t)(n + 1)); /* s_i for i = 0..n */
    double *p = (double *)malloc(sizeof(double) * n3), *acc = (double *)malloc(sizeof(double) * n3);
    double *x = (double *)malloc(sizeof(double) * n3);
    double *xi = (double *)malloc(sizeof(double) * n3), *pi = (double *)malloc(sizeof(double) * n3);
    double *alpha = (double *)malloc(sizeof(double) * n3);
    memcpy(S, s0, sizeof(double) * n3);
    memcpy(p, p0, sizeof(double) * n3);
    orc_init_acc(N, L, om, deconv, S, acc);
    for (int i = 1; i <= n; i++) {
        memcpy(S + (size_t)i * n3, S + (size_t)(i - 1) * n3, sizeof(double) * n3);
        orc_step_fwd(N, L, om, deconv, a, i, S + (size_t)i * n3, p, acc);
    }
    orc_positions(N, L, S + (size_t)n * n3, x);
    double J = orc_objective(N, np, x, delta_target, xi);
    for (long j = 0; j < n3; j++) { pi[j] = 0.0; alpha[j] = 0.0; }
    for (int i = n; i >= 1; i--) {
        /* the adjoint lines of eq. 49 only; state lines replaced by the stored history */
        double ah = a_half(a, i);
        double K1 = orc_kick_factor(om, a[i], a[i], ah);
        double D = orc_drift_factor(om, ah, a[i], a[i - 1]);
        double K2 = orc_kick_factor(om, a[i - 1], ah, a[i - 1]);
        for (long j = 0; j < n3; j++) xi[j] -= alpha[j] * K1;
        for (long j = 0; j < n3; j++) pi[j] -= xi[j] * D;
        vjp_at(N, L, om, deconv, S + (size_t)(i - 1) * n3, pi, alpha);
        for (long j = 0; j < n3; j++) xi[j] -= alpha[j] * K2;
    }
    memcpy(xi0, xi, sizeof(double) * n3);
    memcpy(pi0, pi, sizeof(double) * n3);
    free(S); free(p); free(acc); free(x); free(xi); free(pi); free(alpha);
    return J;
}

/* ------------------------------------------------------------------------------------ */
/* 7. Initial conditions from white noise by Lagrangian perturbation theory, and the VJP */
/*    that turns (xi_0, pi_0) into dJ/d(omega)   (eq. 2-6; L406 eq. 51;   */
/*    growth of second order: L520-555 A1-A8).  SURVEY section 8(f) row 1.                */
/*                                                                                        */
/*    omega(q): real white noise on the particle lattice (L89), q_j = j N/L (reading R6). */
/*    omega(k) = sum_q omega(q) e^{-ik.q}  (L81), k_d = 2 pi m_d / N_d per mesh cell,      */
/*      m_d in [-L_d/2, L_d/2).                                                           */
/*    delta1(k) = amp sqrt(P(k)) omega(k), P(k) = k^ns exp(-(rc k)^2), delta1(0) = 0       */
/*      (eq. 6; the volume factor is part of amp -- DESIGN.md reading R29).               */
/*    nabla^2 phi1 = delta1  ->  phi1(k) = -delta1(k)/k^2;  s1 = -grad phi1 (eq. 3-4):     */
/*      s1_d(k) = i kt_d delta1(k)/k^2.                                                   */
/*    phi1,ab(k) = -k_a k_b phi1(k) = k_a k_b delta1(k)/k^2 ;                              */
/*    S(q) = sum_{a<b} ( phi1,aa phi1,bb - phi1,ab^2 )  (eq. 4, second line);              */
/*    nabla^2 phi2 = S -> phi2(k) = -S(k)/k^2 ; s2 = -grad phi2: s2_d(k) = i kt_d S(k)/k^2.*/
/*    s0 = D1 s1 + D2 s2 ;  p0 = a^2 H (D1' s1 + D2' s2), H = E(a) (H0 = 1)   (eq. 2).     */
/*    Nyquist planes (reading R10 extended): the odd factors (i kt_d, and k_a k_b with     */
/*    a != b) are zero where m_d = -L_d/2; the even ones (k^2, k_a^2) are kept.            */
/* ------------------------------------------------------------------------------------ */

/* right-hand side of eq. A5, both lines (L537), y = (G1, G1', G2, G2'), ' = d/dlna       */
static void growth2_rhs(double om, double lna, const double y[4], double dy[4])
{
    double a = exp(lna);
    double hh = dlnH_of_a(om, a), oma = Om_of_a(om, a);
    dy[0] = y[1];
    dy[1] = -(4.0 + hh) * y[1] - (3.0 + hh - 1.5 * oma) * y[0];
    dy[2] = y[3];
    dy[3] = -(6.0 + hh) * y[3] - (8.0 + 2.0 * hh - 1.5 * oma) * y[2] + 1.5 * oma * y[0] * y[0];
}

/* A5 with the initial conditions A6 (G1 = 1, G1' = 0, G2 = 3/7, G2' = 0 at a = 1e-6),    */
/* RK4 in ln a as orc_growth.  out = {D2, D2'}: D2 = a^2 G2, D2' = a^2 (2 G2 + G2') (A8,   */
/* m = 2, garbling corrected as in reading R2).                                           */
void orc_growth2(double om, double a, double out[2])
{
    const double lna0 = log(1e-6), lna1 = log(a);
    long nstep = (long)ceil((lna1 - lna0) / 1e-3);
    if (nstep < 1) nstep = 1;
    double h = (lna1 - lna0) / (double)nstep;
    double y[4] = {1.0, 0.0, 3.0 / 7.0, 0.0};
    for (long i = 0; i < nstep; i++) {
        double t = lna0 + h * (double)i;
        double k1[4], k2[4], k3[4], k4[4], yt[4];
        growth2_rhs(om, t, y, k1);
        for (int c = 0; c < 4; c++) yt[c] = y[c] + 0.5 * h * k1[c];
        growth2_rhs(om, t + 0.5 * h, yt, k2);
        for (int c = 0; c < 4; c++) yt[c] = y[c] + 0.5 * h * k2[c];
        growth2_rhs(om, t + 0.5 * h, yt, k3);
        for (int c = 0; c < 4; c++) yt[c] = y[c] + h * k3[c];
        growth2_rhs(om, t + h, yt, k4);
        for (int c = 0; c < 4; c++) y[c] += h / 6.0 * (k1[c] + 2.0 * k2[c] + 2.0 * k3[c] + k4[c]);
    }
    out[0] = a * a * y[2];
    out[1] = a * a * (2.0 * y[2] + y[3]);
}

/* lattice mode (ix, iy, iz): k_d (full), kt_d (0 on the lattice Nyquist planes), k^2      */
static inline void lattice_kvec(const int N[3], const int L[3], int ix, int iy, int iz, double k[3], double kt[3], double *k2)
{
    int idx[3] = {ix, iy, iz};
    double kk = 0.0;
    for (int d = 0; d < 3; d++) {
        int m = mode_of(idx[d], L[d]);
        k[d] = 2.0 * PI_ * (double)m / (double)N[d];
        kt[d] = (L[d] % 2 == 0 && m == -L[d] / 2) ? 0.0 : k[d];
        kk += k[d] * k[d];
    }
    *k2 = kk;
}

/* sqrt(P(k)) amp, 0 at k = 0 */
static inline double ic_transfer(double amp, double ns, double rc, double k2)
{
    if (!(k2 > 0.0)) return 0.0;
    return amp * sqrt(pow(k2, 0.5 * ns) * exp(-rc * rc * k2));
}

/* multiplier of phi1,ab: k_a k_b / k^2 with the Nyquist rule above; ab = 0..5 for xx yy zz xy xz yz */
static const int kAB[6][2] = {{0, 0}, {1, 1}, {2, 2}, {0, 1}, {0, 2}, {1, 2}};
static inline double hess_mult(const double k[3], const double kt[3], double k2, int ab)
{
    int a = kAB[ab][0], b = kAB[ab][1];
    if (!(k2 > 0.0)) return 0.0;
    return (a == b ? k[a] * k[a] : kt[a] * kt[b]) / k2;
}

/* real field[np] -> spectrum (new array) ; spectrum -> real part of the inverse transform / np   */
static cplx *ic_spectrum_of(const int L[3], const double *f)
{
    long np = (long)L[0] * L[1] * L[2];
    cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)np);
    for (long i = 0; i < np; i++) w[i] = f[i];
    orc_fft3d(L[0], L[1], L[2], w, -1);
    return w;
}
static void ic_real_of(const int L[3], cplx *w, double *out, long ostride, double *imag_max)
{
    long np = (long)L[0] * L[1] * L[2];
    orc_fft3d(L[0], L[1], L[2], w, +1);
    double im = imag_max ? *imag_max : 0.0;
    for (long i = 0; i < np; i++) {
        out[i * ostride] = creal(w[i]) / (double)np;
        double v = fabs(cimag(w[i])) / (double)np;
        if (v > im) im = v;
    }
    if (imag_max) *imag_max = im;
}

/* s1[3][np], and when order == 2 phi[6][np] (xx yy zz xy xz yz) and s2[3][np], from omega[np] */
static void ic_fields(const int N[3], const int L[3], double amp, double ns, double rc, int order, const double *omega,
                      double *s1, double *phi, double *s2, double *imag_max)
{
    long np = (long)L[0] * L[1] * L[2];
    cplx *wk = ic_spectrum_of(L, omega);
    cplx *t = (cplx *)malloc(sizeof(cplx) * (size_t)np);
    /* delta1(k) in place */
    for (int ix = 0; ix < L[0]; ix++) for (int iy = 0; iy < L[1]; iy++) for (int iz = 0; iz < L[2]; iz++) {
        double k[3], kt[3], k2;
        lattice_kvec(N, L, ix, iy, iz, k, kt, &k2);
        wk[((size_t)ix * L[1] + iy) * L[2] + iz] *= ic_transfer(amp, ns, rc, k2);
    }
    for (int d = 0; d < 3; d++) {
        for (int ix = 0; ix < L[0]; ix++) for (int iy = 0; iy < L[1]; iy++) for (int iz = 0; iz < L[2]; iz++) {
            double k[3], kt[3], k2;
            size_t o = ((size_t)ix * L[1] + iy) * L[2] + iz;
            lattice_kvec(N, L, ix, iy, iz, k, kt, &k2);
            t[o] = k2 > 0.0 ? I * kt[d] / k2 * wk[o] : 0.0;
        }
        ic_real_of(L, t, s1 + (size_t)d * np, 1, imag_max);
    }
    if (order == 2) {
        for (int ab = 0; ab < 6; ab++) {
            for (int ix = 0; ix < L[0]; ix++) for (int iy = 0; iy < L[1]; iy++) for (int iz = 0; iz < L[2]; iz++) {
                double k[3], kt[3], k2;
                size_t o = ((size_t)ix * L[1] + iy) * L[2] + iz;
                lattice_kvec(N, L, ix, iy, iz, k, kt, &k2);
                t[o] = hess_mult(k, kt, k2, ab) * wk[o];
            }
            ic_real_of(L, t, phi + (size_t)ab * np, 1, imag_max);
        }
        double *S = (double *)malloc(sizeof(double) * (size_t)np);
        const double *pxx = phi, *pyy = phi + np, *pzz = phi + 2 * np, *pxy = phi + 3 * np, *pxz = phi + 4 * np, *pyz = phi + 5 * np;
        for (long i = 0; i < np; i++)
            S[i] = pxx[i] * pyy[i] + pxx[i] * pzz[i] + pyy[i] * pzz[i] - pxy[i] * pxy[i] - pxz[i] * pxz[i] - pyz[i] * pyz[i];
        cplx *Sk = ic_spectrum_of(L, S);
        for (int d = 0; d < 3; d++) {
            for (int ix = 0; ix < L[0]; ix++) for (int iy = 0; iy < L[1]; iy++) for (int iz = 0; iz < L[2]; iz++) {
                double k[3], kt[3], k2;
                size_t o = ((size_t)ix * L[1] + iy) * L[2] + iz;
                lattice_kvec(N, L, ix, iy, iz, k, kt, &k2);
                t[o] = k2 > 0.0 ? I * kt[d] / k2 * Sk[o] : 0.0;
            }
            ic_real_of(L, t, s2 + (size_t)d * np, 1, imag_max);
        }
        free(S); free(Sk);
    }
    free(wk); free(t);
}

/* the four time factors of eq. 2 at a0: {D1, D2, a^2 E D1', a^2 E D2'} */
void orc_ic_factors(double om, double a0, double out[4])
{
    double g1[3], g2[2];
    orc_growth(om, a0, g1);
    orc_growth2(om, a0, g2);
    double a2E = a0 * a0 * sqrt(E2_of_a(om, a0));
    out[0] = g1[0]; out[1] = g2[0]; out[2] = a2E * g1[1]; out[3] = a2E * g2[1];
}

/* omega[np] -> s0[np][3], p0[np][3] (eq. 2); order = 1 (Zel'dovich) or 2 (2LPT).          */
/* Returns the largest |imaginary part| met in any inverse transform (must be rounding).   */
double orc_ic(const int N[3], const int L[3], double om, double a0, double amp, double ns, double rc, int order,
              const double *omega, double *s0, double *p0)
{
    long np = (long)L[0] * L[1] * L[2];
    double *s1 = (double *)calloc((size_t)3 * np, sizeof(double)), *s2 = (double *)calloc((size_t)3 * np, sizeof(double));
    double *phi = (double *)calloc((size_t)6 * np, sizeof(double));
    double imag_max = 0.0, f[4];
    ic_fields(N, L, amp, ns, rc, order, omega, s1, phi, s2, &imag_max);
    orc_ic_factors(om, a0, f);
    if (order != 2) f[1] = f[3] = 0.0;
    for (long j = 0; j < np; j++)
        for (int d = 0; d < 3; d++) {
            s0[3 * j + d] = f[0] * s1[(size_t)d * np + j] + f[1] * s2[(size_t)d * np + j];
            p0[3 * j + d] = f[2] * s1[(size_t)d * np + j] + f[3] * s2[(size_t)d * np + j];
        }
    free(s1); free(s2); free(phi);
    return imag_max;
}

/* transposed multiplier applied to a real field and ACCUMULATED into a spectrum: acc(k) += conj(m(k)) FFT[f](k).   */
/* kind 0: m = i kt_d / k^2 (component d);  kind 1: m = hess_mult(ab = d)                                          */
static void ic_accumulate_T(const int N[3], const int L[3], const double *f, int kind, int d, cplx *acc)
{
    cplx *w = ic_spectrum_of(L, f);
    for (int ix = 0; ix < L[0]; ix++) for (int iy = 0; iy < L[1]; iy++) for (int iz = 0; iz < L[2]; iz++) {
        double k[3], kt[3], k2;
        size_t o = ((size_t)ix * L[1] + iy) * L[2] + iz;
        lattice_kvec(N, L, ix, iy, iz, k, kt, &k2);
        if (!(k2 > 0.0)) continue;
        if (kind == 0) acc[o] += -I * kt[d] / k2 * w[o];
        else acc[o] += hess_mult(k, kt, k2, d) * w[o];
    }
    free(w);
}

/* VJP of orc_ic: domega[np] = xi0 . d s0/d omega + pi0 . d p0/d omega  (eq. 51, second line; PAPER.md gives no      */
/* formula -- "computed by AD", L408 -- so this is the transpose of the steps above, taken one by one, backwards):   */
/*   c1 = D1 xi0 + (a^2 E D1') pi0, c2 = D2 xi0 + (a^2 E D2') pi0          (cotangents of s1, s2)                    */
/*   Sbar = sum_d M_d^T c2_d,   M_d = i kt_d / k^2  (real, odd kernel: transpose = conjugate multiplier)             */
/*   phibar_aa = Sbar (sum_{b != a} phi_bb),  phibar_ab = -2 Sbar phi_ab (a < b)                                     */
/*   delta1bar = sum_d M_d^T c1_d + sum_ab H_ab^T phibar_ab,   H_ab real and even: its own transpose                 */
/*   omegabar = T^T delta1bar, T = amp sqrt(P) real and even                                                         */
void orc_ic_vjp(const int N[3], const int L[3], double om, double a0, double amp, double ns, double rc, int order,
                const double *omega, const double *xi0, const double *pi0, double *domega)
{
    long np = (long)L[0] * L[1] * L[2];
    double f[4];
    orc_ic_factors(om, a0, f);
    cplx *dbar = (cplx *)calloc((size_t)np, sizeof(cplx));      /* delta1bar(k) */
    double *c = (double *)malloc(sizeof(double) * (size_t)np);
    for (int d = 0; d < 3; d++) {
        for (long j = 0; j < np; j++) c[j] = f[0] * xi0[3 * j + d] + f[2] * pi0[3 * j + d];
        ic_accumulate_T(N, L, c, 0, d, dbar);
    }
    if (order == 2) {
        double *s1 = (double *)calloc((size_t)3 * np, sizeof(double)), *s2 = (double *)calloc((size_t)3 * np, sizeof(double));
        double *phi = (double *)calloc((size_t)6 * np, sizeof(double));
        ic_fields(N, L, amp, ns, rc, 2, omega, s1, phi, s2, NULL);      /* phi1,ab of the forward pass */
        cplx *Sb = (cplx *)calloc((size_t)np, sizeof(cplx));
        for (int d = 0; d < 3; d++) {
            for (long j = 0; j < np; j++) c[j] = f[1] * xi0[3 * j + d] + f[3] * pi0[3 * j + d];
            ic_accumulate_T(N, L, c, 0, d, Sb);
        }
        double *Sbar = (double *)malloc(sizeof(double) * (size_t)np);
        ic_real_of(L, Sb, Sbar, 1, NULL);
        const double *pxx = phi, *pyy = phi + np, *pzz = phi + 2 * np;
        for (int ab = 0; ab < 6; ab++) {
            for (long j = 0; j < np; j++) {
                double v;
                if (ab == 0) v = pyy[j] + pzz[j];
                else if (ab == 1) v = pxx[j] + pzz[j];
                else if (ab == 2) v = pxx[j] + pyy[j];
                else v = -2.0 * phi[(size_t)ab * np + j];
                c[j] = Sbar[j] * v;
            }
            ic_accumulate_T(N, L, c, 1, ab, dbar);
        }
        free(s1); free(s2); free(phi); free(Sb); free(Sbar);
    }
    for (int ix = 0; ix < L[0]; ix++) for (int iy = 0; iy < L[1]; iy++) for (int iz = 0; iz < L[2]; iz++) {
        double k[3], kt[3], k2;
        lattice_kvec(N, L, ix, iy, iz, k, kt, &k2);
        dbar[((size_t)ix * L[1] + iy) * L[2] + iz] *= ic_transfer(amp, ns, rc, k2);
    }
    ic_real_of(L, dbar, domega, 1, NULL);
    free(dbar); free(c);
}

/* ------------------------------------------------------------------------------------ */
/* 8. Observations between the steps and the cosmological-parameter gradient             */
/*    (eq. 49 last two lines "O_{i-1}: xi_{i-1} += dJ/dx_{i-1}", L393, L369;     */
/*    eq. 51 first line, L406, for theta = Omega_m).  SURVEY section 8(f) rows 3 and 4.   */
/*                                                                                        */
/*    Objective: J = sum_k w_k J_k, J_k = 1/2 sum_g (delta(x_{i_k}) - target_k)^2, the     */
/*    mesh objective of section 5 evaluated on the SNAPSHOTS i_k in 0..n (the simplest     */
/*    observation operator of L179; the light cone of L187 is out of scope).               */
/*    Loop part of eq. 51 with theta = Omega_m (ICs and objective held fixed):             */
/*      dJ/dOm = - sum_i [ (pi_i.acc_i d/dOm + zeta_i) K(t_i,t_i,t_{i-1/2})                */
/*                        + xi_{i-1/2}.p_{i-1/2} dD(t_{i-1/2},t_i,t_{i-1})/dOm            */
/*                        + (pi_{i-1}.acc_{i-1} d/dOm + zeta_{i-1}) K(t_{i-1},t_{i-1/2},t_{i-1}) ] */
/*    where "pi.acc d/dOm K" is (pi.acc) dK/dOm, and zeta = pi . d acc/d Om = pi.acc / Om   */
/*    because acc = F(x) is linear in Om at fixed x (eq. 11).  dK/dOm, dD/dOm: central      */
/*    differences of the factor functions above (step 1e-4; they are smooth in Om).        */
/* ------------------------------------------------------------------------------------ */
static double dot3(long n3, const double *u, const double *v)
{
    double t = 0.0;
    for (long j = 0; j < n3; j++) t += u[j] * v[j];
    return t;
}

double orc_run_fwd_adj_obs(const int N[3], const int L[3], double om, int deconv, int n, const double *a,
                           const double *s0, const double *p0, int n_obs, const int *obs_step, const double *obs_w,
                           const double *targets, double *s_n, double *p_n, double *xi0, double *pi0, double *J_obs,
                           double *dJ_dOm)
{
    long np = (long)L[0] * L[1] * L[2], n3 = 3 * np;
    size_t ng = (size_t)N[0] * N[1] * N[2];
    double *s = (double *)malloc(sizeof(double) * n3), *p = (double *)malloc(sizeof(double) * n3);
    double *acc = (double *)malloc(sizeof(double) * n3), *x = (double *)malloc(sizeof(double) * n3);
    double *xi = (double *)calloc(n3, sizeof(double)), *pi = (double *)calloc(n3, sizeof(double));
    double *alpha = (double *)calloc(n3, sizeof(double)), *g = (double *)malloc(sizeof(double) * n3);
    double J = 0.0, dth = 0.0;
    const double h = 1e-4;
    memcpy(s, s0, sizeof(double) * n3);
    memcpy(p, p0, sizeof(double) * n3);
    orc_init_acc(N, L, om, deconv, s, acc);
    /* forward (eq. 16) with the observations O_i (eq. 17): J_k at the snapshots */
    for (int i = 0; i <= n; i++) {
        if (i > 0) orc_step_fwd(N, L, om, deconv, a, i, s, p, acc);
        for (int k = 0; k < n_obs; k++)
            if (obs_step[k] == i) {
                orc_positions(N, L, s, x);
                double Jk = orc_objective(N, np, x, targets + (size_t)k * ng, NULL);
                if (J_obs) J_obs[k] = Jk;
                J += obs_w[k] * Jk;
            }
    }
    if (s_n) memcpy(s_n, s, sizeof(double) * n3);
    if (p_n) memcpy(p_n, p, sizeof(double) * n3);
    /* eq. 50: xi_n = dJ/dx_n (zero unless t_n is observed), pi_n = 0, alpha_n = 0 */
    for (int k = 0; k < n_obs; k++)
        if (obs_step[k] == n) {
            orc_positions(N, L, s, x);
            orc_objective(N, np, x, targets + (size_t)k * ng, g);
            for (long j = 0; j < n3; j++) xi[j] += obs_w[k] * g[j];
        }
    for (int i = n; i >= 1; i--) {
        double ah = a_half(a, i);
        double K1 = orc_kick_factor(om, a[i], a[i], ah);                 /* K(t_i, t_i, t_{i-1/2})         */
        double D = orc_drift_factor(om, ah, a[i], a[i - 1]);             /* D(t_{i-1/2}, t_i, t_{i-1})     */
        double K2 = orc_kick_factor(om, a[i - 1], ah, a[i - 1]);         /* K(t_{i-1}, t_{i-1/2}, t_{i-1}) */
        double dK1 = (orc_kick_factor(om + h, a[i], a[i], ah) - orc_kick_factor(om - h, a[i], a[i], ah)) / (2 * h);
        double dD = (orc_drift_factor(om + h, ah, a[i], a[i - 1]) - orc_drift_factor(om - h, ah, a[i], a[i - 1])) / (2 * h);
        double dK2 = (orc_kick_factor(om + h, a[i - 1], ah, a[i - 1]) - orc_kick_factor(om - h, a[i - 1], ah, a[i - 1])) / (2 * h);
        double A = dot3(n3, pi, acc);                                    /* pi_i . acc_i                   */
        dth -= A * dK1 + (A / om) * K1;
        for (long j = 0; j < n3; j++) { p[j] += acc[j] * K1; xi[j] -= alpha[j] * K1; }
        dth -= dot3(n3, xi, p) * dD;                                     /* xi_{i-1/2} . p_{i-1/2}         */
        for (long j = 0; j < n3; j++) { s[j] += p[j] * D; pi[j] -= xi[j] * D; }
        force_at(N, L, om, deconv, s, acc);
        vjp_at(N, L, om, deconv, s, pi, alpha);
        A = dot3(n3, pi, acc);                                           /* pi_{i-1} . acc_{i-1}           */
        dth -= A * dK2 + (A / om) * K2;
        for (long j = 0; j < n3; j++) { p[j] += acc[j] * K2; xi[j] -= alpha[j] * K2; }
        /* O_{i-1} (eq. 49, last lines): xi_{i-1} += dJ/dx_{i-1}; dJ/dp = 0 for a density objective */
        for (int k = 0; k < n_obs; k++)
            if (obs_step[k] == i - 1) {
                orc_positions(N, L, s, x);
                orc_objective(N, np, x, targets + (size_t)k * ng, g);
                for (long j = 0; j < n3; j++) xi[j] += obs_w[k] * g[j];
            }
    }
    if (xi0) memcpy(xi0, xi, sizeof(double) * n3);
    if (pi0) memcpy(pi0, pi, sizeof(double) * n3);
    if (dJ_dOm) *dJ_dOm = dth;
    free(s); free(p); free(acc); free(x); free(xi); free(pi); free(alpha); free(g);
    return J;
}
