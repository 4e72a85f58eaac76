// pm_api.cu -- the C ABI of include/pm.h: argument checks, workspace carve-up, cuFFT plans, and the
// sequencing of the hot path (eq. 16 L172 forward; eq. 49-50 L393-397 adjoint; L400-408 run).
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "pm_pos.cuh"

namespace pm {

const char *const kTimingNames[TC_NCLASSES] = {
    "bin_count", "bin_scan", "bin_reorder", "scatter1", "scatter3", "gather", "gather_grad", "gather_fused", "gather_kick",
    "kspace_force", "kspace_adjoint", "fft_r2c", "fft_c2r", "fft_z_r2c", "fft_z_c2r", "fft_y", "kick_drift", "objective", "convert"};

static thread_local std::string g_err_noctx;

int fail(pm_ctx *c, int code, const char *what, const char *detail)
{
    std::string m = std::string(pm_strerror(code)) + ": " + (what ? what : "") + (detail ? std::string(" -- ") + detail : "");
    if (c) c->err = m; else g_err_noctx = m;
    return code;
}

bool pdl_enabled()
{
    static int v = -1;
    if (v < 0) {
        const char *e = getenv("PM_PDL");
        v = (e && atoi(e) == 0) ? 0 : 1;
    }
    return v == 1;
}

bool smem_attr_needed(pm_ctx *c, unsigned long long *mask)
{
    if (c->device < 0 || c->device >= 64) return true;
    const unsigned long long bit = 1ull << c->device;
    if (*mask & bit) return false;
    *mask |= bit;
    return true;
}

// after a stream synchronisation: did a work-queue watchdog fire (pm_cic.cu wq_pop)?  It cannot unless an invariant of
// the queue is broken; then the results are incomplete and the call reports it instead of hanging the GPU.
int check_watchdog(pm_ctx *c)
{
    int h[16];
    PM_CUDA(c, cudaMemcpy(h, c->sched, sizeof h, cudaMemcpyDeviceToHost));
    if (h[8] || h[10]) {
        cudaMemset(c->sched, 0, 64 * sizeof(int));
        return fail(c, PM_ECUDA, "work-queue watchdog", "a CIC kernel gave up waiting on its work queue; results are incomplete");
    }
    return PM_OK;
}

Timer::Timer(pm_ctx *ctx, int cls, double bytes) : c(ctx), idx(-1)
{
    if (cls == TC_FFT_R2C || cls == TC_FFT_C2R) c->n_fft++; else c->n_own++;
    if (!c->timing_on) return;
    TimingRec r;
    r.cls = cls;
    r.bytes = bytes;
    for (cudaEvent_t *e : {&r.e0, &r.e1}) {
        if (!c->event_pool.empty()) { *e = c->event_pool.back(); c->event_pool.pop_back(); }
        else if (cudaEventCreate(e) != cudaSuccess) return;
    }
    cudaEventRecord(r.e0, c->stream);
    c->trecs.push_back(r);
    idx = (int)c->trecs.size() - 1;
}

void Timer::stop()
{
    if (idx >= 0) cudaEventRecord(c->trecs[idx].e1, c->stream);
}

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

static int ceil_log2(int v)
{
    int k = 0;
    while ((1 << k) < v) k++;
    return k;
}

// validates params and fills the geometry; returns PM_OK or PM_EINVAL with text in *why
static int make_geometry(const pm_params *p, Geometry *g, const char **why)
{
    *why = "";
    if (!p) { *why = "params is NULL"; return PM_EINVAL; }
    int maxn = 0;
    for (int d = 0; d < 3; d++) {
        if (p->mesh[d] < 2 || p->mesh[d] > 4096) { *why = "mesh[d] must be in [2, 4096]"; return PM_EINVAL; }
        if (p->lattice[d] < 1) { *why = "lattice[d] must be >= 1"; return PM_EINVAL; }
        if (p->mesh[d] > maxn) maxn = p->mesh[d];
    }
    if (p->mesh[2] % 2) { *why = "mesh[2] must be even (in-place R2C layout)"; return PM_EINVAL; }
    if (!(p->omega_m > 0.0) || p->omega_m > 1.0) { *why = "omega_m must be in (0, 1]"; return PM_EINVAL; }
    if (p->n_steps < 0) { *why = "n_steps < 0"; return PM_EINVAL; }
    if (p->n_steps > 0 && !p->a) { *why = "a is NULL"; return PM_EINVAL; }
    if (p->flags & ~PM_FLAG_FP64_TRANSFORMS) { *why = "unknown bit in flags"; return PM_EINVAL; }
    if (p->deconvolve != 0 && p->deconvolve != 1) { *why = "deconvolve must be 0 or 1"; return PM_EINVAL; }
    if (p->a) {
        for (int i = 0; i <= p->n_steps; i++) {
            if (!(p->a[i] > 0.0) || !std::isfinite(p->a[i])) { *why = "a[i] must be finite and > 0"; return PM_EINVAL; }
            if (i > 0 && !(p->a[i] > p->a[i - 1])) { *why = "a must be strictly increasing"; return PM_EINVAL; }
        }
    }
    int fb = 32 - ceil_log2(maxn);
    g->fbits = fb > 24 ? 24 : fb;  // <= 24: the fraction and 1 - fraction stay exact in fp32
    g->np = 1;
    g->ng = 1;
    for (int d = 0; d < 3; d++) {
        g->N[d] = p->mesh[d];
        g->L[d] = p->lattice[d];
        long long M = (long long)g->N[d] << XBITS;
        if (M % (long long)g->L[d]) { *why = "(mesh[d] << 32) must be divisible by lattice[d]"; return PM_EINVAL; }
        g->qstep[d] = M / (long long)g->L[d];
        g->np *= g->L[d];
        g->ng *= g->N[d];
    }
    if (g->np >= (1ll << 31)) { *why = "more than 2^31 - 1 particles"; return PM_EINVAL; }
    g->nt[0] = (g->N[0] + TX - 1) / TX;
    g->nt[1] = (g->N[1] + TY - 1) / TY;
    g->nt[2] = (g->N[2] + TZ - 1) / TZ;
    g->zs = (g->N[2] + 2 + 3) / 4 * 4;
    g->mesh_stride = (long long)g->N[0] * g->N[1] * g->zs;
    g->nk = (long long)g->N[0] * g->N[1] * (g->N[2] / 2 + 1);
    long long ntiles = (long long)g->nt[0] * g->nt[1] * g->nt[2];
    if (ntiles * NCLS >= (1ll << 31)) { *why = "too many tiles"; return PM_EINVAL; }
    g->ntiles = (int)ntiles;
    g->nkeys = g->ntiles * NCLS;
    return PM_OK;
}

// the single definition of the workspace layout: with base == NULL only sizes are computed
struct Carve {
    size_t off = 0;
    char *base;
    explicit Carve(void *b) : base((char *)b) {}
    template <typename T> T *take(size_t count)
    {
        size_t o = off;
        off = align_up(off + sizeof(T) * count, 256);
        return base ? (T *)(base + o) : nullptr;
    }
};

// global integer accumulators for split scatter tiles (8 KB each): one per 32 tiles, at least 1024 (or every tile)
static int scatter_pool_slots(const Geometry &g)
{
    int n = g.ntiles / 32;
    if (n < 1024) n = 1024;
    if (n > g.ntiles) n = g.ntiles;
    return n;
}

static size_t fft_work_reserve(const Geometry &g) { return 2 * sizeof(float) * (size_t)g.mesh_stride + (32u << 20); }

static size_t carve_workspace(pm_ctx *c, const Geometry &g, void *base, bool fp64_transforms)
{
    Carve w(base);
    float *m = w.take<float>((size_t)g.mesh_stride * 7);
    uint4 *rec = w.take<uint4>((size_t)g.np);
    int *offsets = w.take<int>((size_t)g.nkeys + 1);
    int *cursor = w.take<int>((size_t)g.nkeys + 1);
    int *hist = w.take<int>((size_t)g.nkeys + 1);
    int *sched = w.take<int>(64);
    // work queues (one per stream), 8 ints per item.  Worst case of items: the scatter queues the chunks (2048 records)
    // of tiles whose record runs hold up to 8 np records in all (a particle is visited by its own tile and by up to 7
    // high-side neighbours), the gather np / 1024 chunks: np / 256 items cover both.
    const long long wq_ints = 16 + 8 * ((long long)g.np / 256 + g.ntiles + 64);
    int *wq = w.take<int>((size_t)(2 * wq_ints));
    const int spool_n = scatter_pool_slots(g);
    int *spool_ctl = w.take<int>(16 + (size_t)spool_n);
    unsigned *spool = w.take<unsigned>((size_t)spool_n * TX * TY * TZ);
    unsigned long long *scan_agg = w.take<unsigned long long>((size_t)(g.nkeys + 1) / 4096 + 2);
    long long *x = w.take<long long>((size_t)g.np * 3);
    long long *p = w.take<long long>((size_t)g.np * 3);
    float *acc = w.take<float>((size_t)g.np * 3);
    float *xi = w.take<float>((size_t)g.np * 3);
    float *pi = w.take<float>((size_t)g.np * 3);
    float *alpha = w.take<float>((size_t)g.np * 3);
    double *scal = w.take<double>(4096);
    int tabn = g.N[0] > g.N[1] ? g.N[0] : g.N[1];
    if (g.N[2] > tabn) tabn = g.N[2];
    double *ktab = w.take<double>((size_t)9 * tabn);
    void *ffttab = w.take<char>(fft_own_table_bytes(g));
    void *fftw = w.take<char>(fft_work_reserve(g));
    double *dm = nullptr;
    void *fftw64 = nullptr;
    if (fp64_transforms) {
        dm = w.take<double>(4 * fft64_mesh_doubles(g));
        fftw64 = w.take<char>(fft64_work_bytes(g));
    }
    if (c) {
        for (int k = 0; k < 4; k++) c->dmesh[k] = dm ? dm + (size_t)k * fft64_mesh_doubles(g) : nullptr;
        c->fft64_work = fftw64;
        c->fft64_work_bytes = fp64_transforms ? fft64_work_bytes(g) : 0;
        for (int k = 0; k < 7; k++) c->mesh[k] = m + (size_t)k * g.mesh_stride;
        c->rec = rec; c->offsets = offsets; c->cursor = cursor; c->hist = hist; c->sched = sched; c->wq = wq; c->wq_ints = wq_ints; c->spool_ctl = spool_ctl; c->spool = spool; c->spool_n = spool_n; c->scan_agg = scan_agg;
        c->x = x; c->p = p; c->acc = acc; c->xi = xi; c->pi = pi; c->alpha = alpha;
        c->scal = scal; c->ktab = ktab; c->ktabn = tabn;
        c->fft_tab = ffttab;
        c->fft_work = fftw; c->fft_work_bytes = fft_work_reserve(g);
    }
    return w.off;
}

#define PM_FFT(ctx, call)                                                      \
    do {                                                                       \
        cufftResult r_ = (call);                                               \
        if (r_ != CUFFT_SUCCESS) {                                             \
            char b_[32];                                                       \
            snprintf(b_, sizeof b_, "cufftResult %d", (int)r_);                \
            return pm::fail(ctx, PM_ECUFFT, #call, b_);                        \
        }                                                                      \
    } while (0)

static int make_plans(pm_ctx *c)
{
    const Geometry &g = c->g;
    long long n[3] = {g.N[0], g.N[1], g.N[2]};
    long long rembed[3] = {g.N[0], g.N[1], g.zs};
    long long cembed[3] = {g.N[0], g.N[1], g.zs / 2};
    long long rdist = g.mesh_stride, cdist = g.mesh_stride / 2;
    size_t need = 0, ws = 0;
    PM_FFT(c, cufftCreate(&c->plan_r2c1));
    PM_FFT(c, cufftCreate(&c->plan_c2r1));
    c->plans_ok = true;
    PM_FFT(c, cufftSetAutoAllocation(c->plan_r2c1, 0));
    PM_FFT(c, cufftSetAutoAllocation(c->plan_c2r1, 0));
    PM_FFT(c, cufftMakePlanMany64(c->plan_r2c1, 3, n, rembed, 1, rdist, cembed, 1, cdist, CUFFT_R2C, 1, &ws));
    need = ws;
    PM_FFT(c, cufftMakePlanMany64(c->plan_c2r1, 3, n, cembed, 1, cdist, rembed, 1, rdist, CUFFT_C2R, 1, &ws));
    if (ws > need) need = ws;
    if (need > c->fft_work_bytes) {
        char b[128];
        snprintf(b, sizeof b, "cuFFT work area %zu > reserved %zu", need, c->fft_work_bytes);
        return fail(c, PM_EWORKSPACE, "make_plans", b);
    }
    PM_FFT(c, cufftSetWorkArea(c->plan_r2c1, c->fft_work));
    PM_FFT(c, cufftSetWorkArea(c->plan_c2r1, c->fft_work));
    PM_FFT(c, cufftSetStream(c->plan_r2c1, c->stream));
    PM_FFT(c, cufftSetStream(c->plan_c2r1, c->stream));
    return PM_OK;
}

static int fft_r2c(pm_ctx *c, float *mesh)
{
    Timer t(c, TC_FFT_R2C, 8.0 * (double)c->g.ng);
    PM_FFT(c, cufftExecR2C(c->plan_r2c1, mesh, (cufftComplex *)mesh));
    t.stop();
    return PM_OK;
}

static int fft_c2r(pm_ctx *c, float *mesh)
{
    Timer t(c, TC_FFT_C2R, 8.0 * (double)c->g.ng);
    PM_FFT(c, cufftExecC2R(c->plan_c2r1, (cufftComplex *)mesh, mesh));
    t.stop();
    return PM_OK;
}

// per-axis k tables in fp64 on the host -> device (synchronous copy at init)
static int upload_ktab(pm_ctx *c)
{
    const Geometry &g = c->g;
    int tn = c->ktabn;
    std::vector<double> h((size_t)9 * tn, 0.0);
    const double PI = 3.14159265358979323846264338327950288;
    for (int d = 0; d < 3; d++) {
        int N = g.N[d];
        std::vector<int> order;  // frequency index held at memory position i (digit-reversed for the own FFT's x, y)
        fft_own_axis_order(c, d, order);
        for (int i = 0; i < N; i++) {
            int fi = order[i];
            int m = fi < (N + 1) / 2 ? fi : fi - N;
            double k = 2.0 * PI * (double)m / (double)N;
            bool nyq = (N % 2 == 0) && (m == -N / 2);
            double dec = 1.0;
            if (c->prm.deconvolve && m != 0) {
                double hh = 0.5 * k, sc = std::sin(hh) / hh;
                dec = 1.0 / (sc * sc * sc * sc);
            }
            h[(size_t)(3 * d + 0) * tn + i] = nyq ? 0.0 : k;
            h[(size_t)(3 * d + 1) * tn + i] = k * k;
            h[(size_t)(3 * d + 2) * tn + i] = dec;
        }
    }
    PM_CUDA(c, cudaMemcpy(c->ktab, h.data(), sizeof(double) * h.size(), cudaMemcpyHostToDevice));
    return PM_OK;
}

#ifdef PM_DEBUG
int dbg_prec_init(pm_ctx *c);      // pm_debug_prec.cu
void dbg_prec_destroy(pm_ctx *c);
#endif

}  // namespace pm

using namespace pm;

extern "C" {

const char *pm_strerror(int code)
{
    switch (code) {
        case PM_OK: return "PM_OK";
        case PM_EINVAL: return "PM_EINVAL (bad argument)";
        case PM_EWORKSPACE: return "PM_EWORKSPACE (workspace too small or misaligned)";
        case PM_ECUDA: return "PM_ECUDA (CUDA call failed)";
        case PM_ECUFFT: return "PM_ECUFFT (cuFFT call failed)";
        case PM_ESTATE: return "PM_ESTATE (call out of order)";
        default: return "unknown pm error code";
    }
}

const char *pm_last_error(const pm_ctx *ctx) { return ctx ? ctx->err.c_str() : g_err_noctx.c_str(); }

int pm_workspace_bytes(const pm_params *params, size_t *bytes)
{
    Geometry g;
    const char *why;
    if (!bytes) return fail(nullptr, PM_EINVAL, "pm_workspace_bytes", "bytes is NULL");
    int rc = make_geometry(params, &g, &why);
    if (rc != PM_OK) return fail(nullptr, rc, "pm_workspace_bytes", why);
    *bytes = carve_workspace(nullptr, g, nullptr, (params->flags & PM_FLAG_FP64_TRANSFORMS) != 0);
    return PM_OK;
}

int pm_init(pm_ctx **out, const pm_params *params, void *dev_workspace, size_t bytes, void *cuda_stream)
{
    if (!out) return fail(nullptr, PM_EINVAL, "pm_init", "out is NULL");
    *out = nullptr;
    Geometry g;
    const char *why;
    int rc = make_geometry(params, &g, &why);
    if (rc != PM_OK) return fail(nullptr, rc, "pm_init", why);
    if (!dev_workspace || ((uintptr_t)dev_workspace & 255)) return fail(nullptr, PM_EWORKSPACE, "pm_init", "dev_workspace NULL or not 256-byte aligned");
    const bool f64 = (params->flags & PM_FLAG_FP64_TRANSFORMS) != 0;
    size_t need = carve_workspace(nullptr, g, nullptr, f64);
    if (bytes < need) return fail(nullptr, PM_EWORKSPACE, "pm_init", "bytes < pm_workspace_bytes");
    pm_ctx *c = new (std::nothrow) pm_ctx();
    if (!c) return fail(nullptr, PM_EINVAL, "pm_init", "out of host memory");
    c->g = g;
    c->prm = *params;
    c->prm.a = nullptr;
    c->stream = (cudaStream_t)cuda_stream;
    c->plans_ok = false;
    c->plans64_ok = false;
    c->plans_ic_ok = false;
    c->fp64_transforms = f64;
    c->t_index = -1;
    c->have_adjoint = false;
    c->sorted_valid = false;
    c->hist_valid = false;
    c->timing_on = false;
    c->n_own = c->n_fft = 0;
    c->cur_np = 0;
    int n = params->n_steps;
    if (params->a) c->a.assign(params->a, params->a + n + 1);
    double om = params->omega_m;
    c->fac.resize((size_t)3 * n);
    for (int i = 1; i <= n; i++) pm_host_step_factors(om, c->a[i - 1], c->a[i], &c->fac[3 * (size_t)(i - 1)]);
    c->p_over_s0 = 0.0;
    if (!c->a.empty()) {
        double gr[4];
        growth_host(om, c->a[0], gr);
        c->p_over_s0 = gr[2] / gr[0];
    }
    carve_workspace(c, g, dev_workspace, f64);
    c->tma_ok = false;
    // fp64 transforms go through cuFFT's double-precision plans: the k tables then stay in natural order
    c->own_fft = !f64 && fft_own_supported(g);
    rc = f64 ? fft64_init(c) : (c->own_fft ? PM_OK : make_plans(c));
    if (rc == PM_OK) rc = cic_init_tensor_maps(c);
    if (rc == PM_OK) rc = upload_ktab(c);
    if (rc == PM_OK && !f64) rc = fft_own_init(c);
    c->scan_epoch = 0;
    c->wq_epoch = 0;
    if (rc == PM_OK && cudaMemsetAsync(c->wq, 0, sizeof(int) * (size_t)(2 * c->wq_ints), c->stream) != cudaSuccess) rc = fail(c, PM_ECUDA, "pm_init", "clearing the gather work queue");
    if (rc == PM_OK && (cudaMemsetAsync(c->spool_ctl, 0, sizeof(int) * (16 + (size_t)c->spool_n), c->stream) != cudaSuccess ||
                        cudaMemsetAsync(c->spool, 0, sizeof(unsigned) * (size_t)c->spool_n * TX * TY * TZ, c->stream) != cudaSuccess))
        rc = fail(c, PM_ECUDA, "pm_init", "clearing the scatter accumulator pool");
    c->overlap_ok = false;
    c->stream2 = nullptr;
    c->ev_fork = c->ev_xforce = c->ev_join = nullptr;
    {
        const char *e = getenv("PM_OVERLAP");
        if (!(e && atoi(e) == 0) && cudaStreamCreateWithFlags(&c->stream2, cudaStreamNonBlocking) == cudaSuccess) {
            bool ok = cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) == cudaSuccess;
            ok = ok && cudaEventCreateWithFlags(&c->ev_xforce, cudaEventDisableTiming) == cudaSuccess;
            ok = ok && cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) == cudaSuccess;
            c->overlap_ok = ok;  // whatever was created is destroyed by pm_destroy either way
        } else {
            c->stream2 = nullptr;
        }
        (void)cudaGetLastError();
    }
    {
        c->device = 0;
        c->num_sms = 148;
        if (cudaGetDevice(&c->device) == cudaSuccess) cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device);
    }
    if (rc == PM_OK && cudaMemsetAsync(c->sched, 0, 64 * sizeof(int), c->stream) != cudaSuccess) rc = fail(c, PM_ECUDA, "pm_init", "clearing the tile scheduler");
    if (rc == PM_OK && (cudaMemsetAsync(c->scan_agg, 0, sizeof(unsigned long long) * ((size_t)(g.nkeys + 1) / 4096 + 2), c->stream) != cudaSuccess ||
                        cudaMemsetAsync(c->hist, 0, sizeof(int) * ((size_t)g.nkeys + 1), c->stream) != cudaSuccess ||
                        cudaStreamSynchronize(c->stream) != cudaSuccess))
        rc = fail(c, PM_ECUDA, "pm_init", "clearing the key histogram");
#ifdef PM_DEBUG
    if (rc == PM_OK) rc = dbg_prec_init(c);
#endif
    if (rc != PM_OK) {
        g_err_noctx = c->err;
        pm_destroy(c);
        return rc;
    }
    *out = c;
    return PM_OK;
}

int pm_destroy(pm_ctx *c)
{
    if (!c) return PM_OK;
#ifdef PM_DEBUG
    dbg_prec_destroy(c);
#endif
    fft64_destroy(c);
    ic_destroy(c);
    if (c->plans_ok) {
        cufftDestroy(c->plan_r2c1);
        cufftDestroy(c->plan_c2r1);
    }
    for (auto &r : c->trecs) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
    for (auto e : c->event_pool) cudaEventDestroy(e);
    if (c->stream2) cudaStreamSynchronize(c->stream2);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_xforce) cudaEventDestroy(c->ev_xforce);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->stream2) cudaStreamDestroy(c->stream2);
    (void)cudaGetLastError();
    delete c;
    return PM_OK;
}

int pm_host_growth(double omega_m, double a, double out[4])
{
    if (!out || !(a > 0.0) || !(omega_m > 0.0) || omega_m > 1.0) return PM_EINVAL;
    growth_host(omega_m, a, out);
    return PM_OK;
}

int pm_host_step_factors(double omega_m, double a0, double a1, double out[3])
{
    if (!out || !(a0 > 0.0) || !(a1 > 0.0) || !(omega_m > 0.0) || omega_m > 1.0) return PM_EINVAL;
    double ah = 0.5 * (a0 + a1);  // a_{i-1/2}: DESIGN.md R3
    out[0] = kick_factor_host(omega_m, a0, a0, ah);
    out[1] = drift_factor_host(omega_m, ah, a0, a1);
    out[2] = kick_factor_host(omega_m, a1, ah, a1);
    return PM_OK;
}

int pm_host_fft_order(int32_t n, int32_t *out) { return fft_own_order_host((int)n, (int *)out); }

int pm_step_factors(const pm_ctx *c, int i, double out[3])
{
    if (!c || !out || i < 1 || i > c->prm.n_steps) return PM_EINVAL;
    for (int k = 0; k < 3; k++) out[k] = c->fac[3 * (i - 1) + k];
    return PM_OK;
}

}  // extern "C"

#include "pm_api_ops.inc"
