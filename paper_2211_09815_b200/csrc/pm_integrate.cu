// pm_integrate.cu -- fused kick/drift updates of the reversible KDK integrator, objective residual.
//
// PAPER.md eq. 16 (L172): K: p += acc K;  D: x += p D;  eq. 49 (L393): the adjoint step undoes them in
// reverse order with the time arguments swapped, D(tc,ta,tb) = -D(tc,tb,ta) (L389), and advances
// xi -= alpha K, pi -= xi D alongside.  The state is held in fixed point (x = q + s: int64 * 2^-XBITS cells,
// p: int64 * 2^-PBITS) so that "+= round(v)" followed by "+= round(-v)" restores it bit for bit: the
// reverse pass then re-evaluates F at exactly the forward positions (
// L371 names "more precise floating-point numbers" as the paper's remedy for fp32 irreversibility).
#include "pm_pos.cuh"

namespace pm {

static inline int ew_blocks(long long n)
{
    long long b = (n + 255) / 256;
    if (b > 148 * 16) b = 148 * 16;
    if (b < 1) b = 1;
    return (int)b;
}

// lattice site of particle j in state units (q_j = (jx, jy, jz) * N/L cells, R6)
__device__ __forceinline__ void lattice_site(const PosGeom &g, long long j, long long q[3])
{
    long long jz = j % g.L[2], t = j / g.L[2];
    long long jy = t % g.L[1], jx = t / g.L[1];
    q[0] = jx * g.qstep[0];
    q[1] = jy * g.qstep[1];
    q[2] = jz * g.qstep[2];
}

__global__ void __launch_bounds__(256) state_from_float_kernel(PosGeom g, long long np, const float *__restrict__ s,
                                                               const float *__restrict__ p, double xscale, double pscale,
                                                               long long *__restrict__ xf, long long *__restrict__ pf)
{
    long long stride = (long long)gridDim.x * blockDim.x;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < np; j += stride) {
        long long q[3];
        lattice_site(g, j, q);
#pragma unroll
        for (int d = 0; d < 3; d++) {
            xf[3 * j + d] = q[d] + __double2ll_rn((double)s[3 * j + d] * xscale);
            pf[3 * j + d] = __double2ll_rn((double)p[3 * j + d] * pscale);
        }
    }
}

__global__ void __launch_bounds__(256) state_to_float_kernel(PosGeom g, long long np, const long long *__restrict__ xf,
                                                             const long long *__restrict__ pf, double inv_xscale,
                                                             double inv_pscale, float *__restrict__ s, float *__restrict__ p)
{
    long long stride = (long long)gridDim.x * blockDim.x;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < np; j += stride) {
        long long q[3];
        lattice_site(g, j, q);
#pragma unroll
        for (int d = 0; d < 3; d++) {
            if (s) s[3 * j + d] = (float)((double)(xf[3 * j + d] - q[d]) * inv_xscale);
            if (p) p[3 * j + d] = (float)((double)pf[3 * j + d] * inv_pscale);
        }
    }
}

// Ks = K * 2^PBITS, Ds = D * 2^(XBITS - PBITS).  ADJ also advances xi, pi with the plain K, D.
// One thread per particle; a drift also adds the particle's new sort key to the histogram of the next sort.
template <bool ADJ>
__global__ void __launch_bounds__(256) kick_drift_kernel(PosGeom g, long long np, double Ks, double Ds, float K, float D,
                                                         long long *__restrict__ x, long long *__restrict__ p,
                                                         const float *__restrict__ acc, float *__restrict__ xi,
                                                         float *__restrict__ pi, const float *__restrict__ alpha,
                                                         int *__restrict__ hist)
{
    long long stride = (long long)gridDim.x * blockDim.x;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < np; j += stride) {
        unsigned int X[3];
#pragma unroll
        for (int d = 0; d < 3; d++) {
            const long long i = 3 * j + d;
            long long pv = p[i];
            if (Ks != 0.0) {
                pv += __double2ll_rn((double)acc[i] * Ks);
                p[i] = pv;
            }
            if (Ds != 0.0) {
                long long xv = x[i] + __double2ll_rn((double)pv * Ds);
                x[i] = xv;
                X[d] = record_coord(g, xv, d);
            }
            if (ADJ) {
                float v = xi[i];
                if (Ks != 0.0) {
                    v = fmaf(-alpha[i], K, v);
                    xi[i] = v;
                }
                if (Ds != 0.0) pi[i] = fmaf(-v, D, pi[i]);
            }
        }
        if (Ds != 0.0) hist_add(hist, key_of(g, X));
    }
}

// r = rho/nbar - 1 - target, in place in the padded mesh; J += 1/2 sum r^2 (fp64)
__global__ void __launch_bounds__(256) objective_kernel(int Nx, int Ny, int Nz, int zs, float inv_nbar, float *__restrict__ mesh,
                                                        const float *__restrict__ target, double *__restrict__ J)
{
    __shared__ double red[8];
    long long ng = (long long)Nx * Ny * Nz;
    long long stride = (long long)gridDim.x * blockDim.x;
    double part = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < ng; i += stride) {
        int iz = (int)(i % Nz);
        long long row = i / Nz;
        size_t o = (size_t)row * zs + iz;
        float r = fmaf(mesh[o], inv_nbar, -1.f) - target[i];
        mesh[o] = r;
        part += 0.5 * (double)r * (double)r;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = part;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < 8; k++) t += red[k];
        J[1 + blockIdx.x] = t;  // per-block partial; summed in a fixed order below (bit-reproducible J)
    }
}

__global__ void objective_final_kernel(int nblocks, double *__restrict__ J)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < nblocks; k++) t += J[1 + k];
        J[0] = t;
    }
}

__global__ void __launch_bounds__(256) combine_kernel(long long n3, const float *__restrict__ xi, const float *__restrict__ pi,
                                                      float ratio, float *__restrict__ out)
{
    long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n3; i += stride)
        out[i] = fmaf(pi[i], ratio, xi[i]);
}

int state_from_float(pm_ctx *c, const float *s, const float *p)
{
    long long np = c->g.np;
    Timer t(c, TC_CONVERT, 72.0 * np);
    state_from_float_kernel<<<ew_blocks(np), 256, 0, c->stream>>>(make_pos_geom(c->g), np, s, p, ldexp(1.0, XBITS),
                                                                  ldexp(1.0, PBITS), c->x, c->p);
    PM_LAUNCH_CHECK(c, "state_from_float_kernel");
    t.stop();
    return PM_OK;
}

int state_to_float(pm_ctx *c, float *s, float *p)
{
    long long np = c->g.np;
    Timer t(c, TC_CONVERT, 72.0 * np);
    state_to_float_kernel<<<ew_blocks(np), 256, 0, c->stream>>>(make_pos_geom(c->g), np, c->x, c->p, ldexp(1.0, -XBITS),
                                                                ldexp(1.0, -PBITS), s, p);
    PM_LAUNCH_CHECK(c, "state_to_float_kernel");
    t.stop();
    return PM_OK;
}

// a drift invalidates the sort and leaves the key histogram of the new positions in c->hist
static int drift_bookkeeping(pm_ctx *c, double D)
{
    if (D != 0.0) {
        if (c->hist_valid) return fail(c, PM_ESTATE, "kick_drift", "internal: key histogram already pending");
        c->sorted_valid = false;
        c->hist_valid = true;
    }
    return PM_OK;
}

int kick_drift(pm_ctx *c, double K, double D)
{
    long long np = c->g.np;
    double Ks = ldexp(K, PBITS), Ds = ldexp(D, XBITS - PBITS);
    PM_TRY(drift_bookkeeping(c, D));
    Timer t(c, TC_KICK_DRIFT, 3.0 * np * ((K != 0.0 ? 20.0 : 8.0) + (D != 0.0 ? 16.0 : 0.0)));
    kick_drift_kernel<false><<<ew_blocks(np), 256, 0, c->stream>>>(make_pos_geom(c->g), np, Ks, Ds, (float)K, (float)D, c->x, c->p,
                                                                   c->acc, nullptr, nullptr, nullptr, c->hist);
    PM_LAUNCH_CHECK(c, "kick_drift_kernel");
    t.stop();
    return PM_OK;
}

int kick_drift_adj(pm_ctx *c, double K, double D)
{
    long long np = c->g.np;
    double Ks = ldexp(K, PBITS), Ds = ldexp(D, XBITS - PBITS);
    PM_TRY(drift_bookkeeping(c, D));
    Timer t(c, TC_KICK_DRIFT, 3.0 * np * ((K != 0.0 ? 32.0 : 12.0) + (D != 0.0 ? 24.0 : 0.0)));
    kick_drift_kernel<true><<<ew_blocks(np), 256, 0, c->stream>>>(make_pos_geom(c->g), np, Ks, Ds, (float)K, (float)D, c->x, c->p,
                                                                  c->acc, c->xi, c->pi, c->alpha, c->hist);
    PM_LAUNCH_CHECK(c, "kick_drift_kernel<adj>");
    t.stop();
    return PM_OK;
}

int objective_residual(pm_ctx *c, float *mesh, const float *target, double nbar)
{
    const Geometry &g = c->g;
    Timer t(c, TC_OBJECTIVE, 12.0 * (double)g.ng);
    int nb = ew_blocks(g.ng);  // <= 148 * 16 < the 4096 doubles of scal
    objective_kernel<<<nb, 256, 0, c->stream>>>(g.N[0], g.N[1], g.N[2], g.zs, (float)(1.0 / nbar), mesh, target, c->scal);
    objective_final_kernel<<<1, 32, 0, c->stream>>>(nb, c->scal);
    c->n_own++;
    PM_LAUNCH_CHECK(c, "objective_kernel");
    t.stop();
    return PM_OK;
}

int combine_dJ_ds0(pm_ctx *c, float *out)
{
    long long n3 = 3 * c->g.np;
    Timer t(c, TC_CONVERT, 12.0 * n3);
    combine_kernel<<<ew_blocks(n3), 256, 0, c->stream>>>(n3, c->xi, c->pi, (float)c->p_over_s0, out);
    PM_LAUNCH_CHECK(c, "combine_kernel");
    t.stop();
    return PM_OK;
}

int fill_zero(pm_ctx *c, void *ptr, size_t bytes)
{
    PM_CUDA(c, cudaMemsetAsync(ptr, 0, bytes, c->stream));
    return PM_OK;
}

// ---- reductions and updates of the run with observations / the Omega_m gradient (eq. 49 last lines, eq. 51) ----------
// sum_j a_j b_j in fp64, per-block partials then one fixed-order sum: acc[0] += coef * sum (bit-reproducible)
__global__ void __launch_bounds__(256) dot_kernel(long long n, const float *__restrict__ a, const float *__restrict__ b,
                                                  const long long *__restrict__ bfix, double bscale, double *__restrict__ partial)
{
    __shared__ double red[8];
    const long long stride = (long long)gridDim.x * blockDim.x;
    double part = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        part += (double)a[i] * (bfix ? (double)bfix[i] * bscale : (double)b[i]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = part;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < 8; k++) t += red[k];
        partial[blockIdx.x] = t;
    }
}
__global__ void dot_final_kernel(int nblocks, const double *__restrict__ partial, double coef, double *__restrict__ acc)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < nblocks; k++) t += partial[k];
        acc[0] += coef * t;
    }
}
__global__ void __launch_bounds__(256) axpy_kernel(long long n, float w, const float *__restrict__ src, float *__restrict__ dst)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) dst[i] = fmaf(w, src[i], dst[i]);
}

// acc[0] += coef * sum_j a_j b_j over the 3 N_p components; b is a float array, or (bfix) the fixed-point momenta
int dot_accumulate(pm_ctx *c, const float *a, const float *b, const long long *bfix, double coef, double *acc)
{
    const long long n3 = 3 * c->g.np;
    const int nb = ew_blocks(n3);
    dot_kernel<<<nb, 256, 0, c->stream>>>(n3, a, b, bfix, ldexp(1.0, -PBITS), c->scal + 1);
    dot_final_kernel<<<1, 32, 0, c->stream>>>(nb, c->scal + 1, coef, acc);
    c->n_own += 2;
    PM_LAUNCH_CHECK(c, "dot_kernel");
    return PM_OK;
}

int axpy(pm_ctx *c, long long n, float w, const float *src, float *dst)
{
    axpy_kernel<<<ew_blocks(n), 256, 0, c->stream>>>(n, w, src, dst);
    c->n_own++;
    PM_LAUNCH_CHECK(c, "axpy_kernel");
    return PM_OK;
}

// Adam (the optimiser of the paper's Fig. 4 experiment, L482-488): m <- b1 m + (1 - b1) g, v <- b2 v + (1 - b2) g^2,
// w <- w - lr (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps); c1 = 1 / (1 - b1^t), c2 = 1 / (1 - b2^t) from the host
__global__ void __launch_bounds__(256) adam_kernel(long long n, float *__restrict__ w, const float *__restrict__ g, float *__restrict__ m,
                                                   float *__restrict__ v, float lr, float b1, float b2, float omb1, float omb2, float eps, float c1, float c2)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const float gi = g[i];
        const float mi = b1 * m[i] + omb1 * gi;          // omb = 1 - beta, formed in fp64 on the host (1 - 0.999f is off by 5e-5)
        const float vi = b2 * v[i] + omb2 * gi * gi;
        m[i] = mi;
        v[i] = vi;
        w[i] -= lr * (mi * c1) / (sqrtf(vi * c2) + eps);
    }
}

int adam_step(pm_ctx *c, long long n, float *w, const float *g, float *m, float *v, int t, double lr, double b1, double b2, double eps)
{
    const double c1 = 1.0 / (1.0 - pow(b1, (double)t)), c2 = 1.0 / (1.0 - pow(b2, (double)t));
    adam_kernel<<<ew_blocks(n), 256, 0, c->stream>>>(n, w, g, m, v, (float)lr, (float)b1, (float)b2, (float)(1.0 - b1), (float)(1.0 - b2), (float)eps, (float)c1, (float)c2);
    c->n_own++;
    PM_LAUNCH_CHECK(c, "adam_kernel");
    return PM_OK;
}

}  // namespace pm
