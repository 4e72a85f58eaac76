// pm_internal.cuh -- private declarations of libpm (CUDA, sm_100a).  Not part of the ABI.
// Shares nothing with oracle/ (the CPU fp64 oracle is test infrastructure with its own code).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>
#include <string>
#include <utility>
#include <vector>

#include "pm.h"

namespace pm {

// ---- tile geometry of the cell sort -----------------------------------------------------------------
// Particles are binned by mesh tile of TX x TY x TZ cells (z contiguous in memory: 32 cells = one
// 128-byte row of fp32) and, inside a tile, by a 3-bit class: bit 2/1/0 set when the particle sits in
// the LAST cell layer of the tile along x/y/z, i.e. when its CIC cloud reaches into the next tile.
constexpr int TX = 8, TY = 8, TZ = 32;
constexpr int NCLS = 8;
constexpr int GCHUNK = 1024;  // gather: tiles with more particles are split into chunks that any CTA may take
constexpr int PBITS = 36;  // momentum fixed point: p_fix = p * 2^PBITS (int64)
constexpr int XBITS = 32;  // position fixed point: x_fix = (q + s) * 2^XBITS (int64, absolute, not wrapped)

// ---- timing classes ---------------------------------------------------------------------------------
enum TimingClass {
    TC_BIN_COUNT = 0,
    TC_BIN_SCAN,
    TC_BIN_REORDER,
    TC_SCATTER1,
    TC_SCATTER3,
    TC_GATHER3,
    TC_GATHER_GRAD,
    TC_GATHER_FUSED,
    TC_GATHER_KICK,
    TC_KSPACE_FORCE,
    TC_KSPACE_ADJ,
    TC_FFT_R2C,
    TC_FFT_C2R,
    TC_FFT_Z_R2C,
    TC_FFT_Z_C2R,
    TC_FFT_Y,
    TC_KICK_DRIFT,
    TC_OBJECTIVE,
    TC_CONVERT,
    TC_NCLASSES
};
extern const char *const kTimingNames[TC_NCLASSES];

struct TimingRec {
    cudaEvent_t e0, e1;
    int cls;
    double bytes;
};

struct Geometry {
    int N[3];        // mesh
    int L[3];        // lattice
    int nt[3];       // tiles per axis
    int fbits;       // fraction bits of the absolute fixed-point coordinate
    int zs;          // floats per z-row of a (padded) internal mesh: Nz + 2 rounded up to a multiple of 4
                     // (16-byte rows: TMA global strides and vector loads need it; cuFFT takes it as inembed)
    long long np;    // particles of the lattice
    long long ng;    // Nx*Ny*Nz
    long long mesh_stride;  // floats per internal padded mesh: Nx*Ny*(Nz+2)
    long long nk;    // complex modes Nx*Ny*(Nz/2+1)
    int ntiles;      // nt[0]*nt[1]*nt[2]
    int nkeys;       // ntiles * NCLS
    long long qstep[3];  // lattice spacing in state units: (N << XBITS) / L
};

}  // namespace pm

struct pm_ctx {
    pm::Geometry g;
    pm_params prm;
    std::vector<double> a;       // n+1 scale factors
    std::vector<double> fac;     // 3 per step: K1, D, K2 (forward)
    double p_over_s0;            // G_D(a0)/D1(a0)
    cudaStream_t stream;         // the stream launches go to (the caller's; temporarily stream2 inside StreamScope)
    cudaStream_t stream2;        // second stream: the Pi branch of an adjoint step runs beside the force branch
    cudaEvent_t ev_fork, ev_xforce, ev_join;
    bool overlap_ok;             // stream2 and the events exist (and PM_OVERLAP != 0)
    cufftHandle plan_r2c1, plan_c2r1;
    bool plans_ok;
    // PM_FLAG_FP64_TRANSFORMS (pm_fft64.cu): double-precision plans, four fp64 meshes [Nx][Ny][Nz + 2], their work area
    cufftHandle plan_ic_r2c, plan_ic_c2r;   // transforms on the particle lattice (pm_ic.cu), created at the first pm_ic_* call
    bool plans_ic_ok;
    bool fp64_transforms;
    cufftHandle plan_d2z, plan_z2d;
    bool plans64_ok;
    double *dmesh[4];
    void *fft64_work;
    size_t fft64_work_bytes;
    // workspace carve-up (device pointers)
    float *mesh[7];              // padded in-place R2C layout, contiguous
    uint4 *rec;                  // sorted records {X, Y, Z, j}
    int *offsets;                // nkeys + 1 exclusive prefix of the key histogram
    int *cursor;                 // nkeys + 1 running cursors of the reorder pass
    int *hist;                   // nkeys + 1 key histogram; zero between sorts (the scan clears it)
    unsigned long long *scan_agg;  // scan scratch: per-block totals tagged with the launch epoch
    unsigned int scan_epoch;
    int *sched;                  // per stream (stream2: + 2): [0] tile counter, [1] finished CTAs of the persistent CIC kernels (zero
                                 // between launches), [8] work-queue watchdog flag (check_watchdog)
    int num_sms;
    int device;                  // CUDA device the ctx was created on
    int *wq;                     // work queue of the CIC kernels (chunks of heavy tiles): [0] head, [1] tail, [2] tiles published, items from [16]
    long long wq_ints;           // ints per queue (two queues: one per stream)
    unsigned int wq_epoch;       // tag of the items pushed by the current launch
    int *spool_ctl;              // scatter pool control: [0] next accumulator, [16 + p] arrived chunks
    unsigned *spool;             // scatter pool: spool_n accumulators of one tile (8 KB) each, zero between uses
    int spool_n;
    long long *x;                // [np][3] int64 absolute position (q + s) * 2^XBITS, not wrapped
    long long *p;                // [np][3] int64 momentum * 2^PBITS
    float *acc, *xi, *pi, *alpha;  // [np][3]
    double *scal;                // device scalars: [0] = J
    double *ktab;                // [3 axes][3: kt, k^2, dec][ktabn] per-axis k-space tables (fp64)
    int ktabn;
    long long cur_np;            // particles in the current sort
    CUtensorMap tmap_store;      // 4-D {z, y, x, mesh 0..6} view of the internal meshes with the tile box (scatter stores)
    bool tma_ok;                 // cuTensorMapEncodeTiled resolved and the internal maps encoded
    void *fft_work;
    bool own_fft;                // power-of-two mesh: own FFT passes with the k-space operators fused (pm_fft.cu)
    void *fft_tab;               // twiddle / position tables of the own FFT
    alignas(8) unsigned char fft_geom[320];  // pm::FftGeom (pm_fft.cu)
    size_t fft_work_bytes;
    // integrator bookkeeping
    int t_index;                 // state is at t_{t_index}; -1 = no state
    bool have_adjoint;
    bool sorted_valid;           // rec/offsets describe the current state's positions
    bool hist_valid;             // hist holds the key histogram of the current state's positions
    // instrumentation
    bool timing_on;
    std::vector<pm::TimingRec> trecs;
    std::vector<cudaEvent_t> event_pool;
    long long n_own, n_fft;
    std::string err;
};

namespace pm {

// record the last error text and return code
int fail(pm_ctx *c, int code, const char *what, const char *detail);
// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is per device: true when (slot, device of ctx) still needs it.
// slot = a function-local static 64-bit mask at the launch site (devices 0..63; beyond that the attribute is set every time)
bool smem_attr_needed(pm_ctx *c, unsigned long long *mask);
int check_watchdog(pm_ctx *c);

#define PM_CUDA(ctx, call)                                                        \
    do {                                                                          \
        cudaError_t e_ = (call);                                                  \
        if (e_ != cudaSuccess) return pm::fail(ctx, PM_ECUDA, #call, cudaGetErrorString(e_)); \
    } while (0)
#define PM_LAUNCH_CHECK(ctx, name)                                                \
    do {                                                                          \
        cudaError_t e_ = cudaGetLastError();                                      \
        if (e_ != cudaSuccess) return pm::fail(ctx, PM_ECUDA, name, cudaGetErrorString(e_)); \
    } while (0)
#define PM_TRY(expr)                 \
    do {                             \
        int rc_ = (expr);            \
        if (rc_ != PM_OK) return rc_; \
    } while (0)

// ---- programmatic dependent launch (PDL) ------------------------------------------------------------
// Kernels launched through launch_pdl may be scheduled while the previous kernel of the stream is still draining;
// each of them calls pdl_enter() before it touches anything a predecessor wrote (it also lets ITS successor in).
// What overlaps is the launch latency, the CTA ramp-up and the prologue with the predecessor's tail.  PM_PDL=0 disables.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_enter()
{
    pdl_trigger();
    pdl_wait();
}
#endif
bool pdl_enabled();
template <class... KArgs, class... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = pdl_enabled() ? 1 : 0;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

// RAII-ish bracket: t = Timer(ctx, cls, bytes); launch...; t.stop()
struct Timer {
    pm_ctx *c;
    int idx;
    Timer(pm_ctx *ctx, int cls, double bytes);
    void stop();
};

// ---- host growth (pm_growth.cc) ---------------------------------------------------------------------
void growth_host(double om, double a, double out[4]);  // D1, dD1/dlna, G_D, G_K
double drift_factor_host(double om, double ac, double aa, double ab);
double kick_factor_host(double om, double ac, double aa, double ab);

// ---- binning (pm_bin.cu) ----------------------------------------------------------------------------
// particles given as absolute float positions (x != NULL) or as the ctx state (x == NULL):
// bin_count adds their keys to c->hist (zero on entry); bin_sort scans c->hist (and clears it) and writes the records
int bin_count(pm_ctx *c, long long np, const float *x);
int bin_sort(pm_ctx *c, long long np, const float *x);

// ---- CIC (pm_cic.cu): operate on the sorted records of the last bin_particles -----------------------
// encode the two internal tensor maps (call once from pm_init); failure leaves tma_ok = false (plain loads)
int cic_init_tensor_maps(pm_ctx *c);
// val: [np][C] in ORIGINAL particle order or NULL.  mesh: C meshes, row stride zs, mesh stride ms.
// Internal meshes (pointers inside c->mesh[]) use the ctx's tensor maps; other pointers get a map encoded per call
// when their layout allows TMA (16-byte aligned base and strides), else the kernels' plain load/store path.
// mean (unit-mass scatter only): constant removed from every mesh point before the conversion to fp32
int scatter_sorted(pm_ctx *c, const float *val, int C, float *mesh, int zs, long long ms, double mean = 0.0);
struct KickArgs;  // pm_pos.cuh
// ka != NULL (C = 3): fused kick / kick / drift + key histogram on the interpolated acc (see gather_kernel)
int gather_sorted(pm_ctx *c, const float *mesh, int C, int zs, long long ms, float *out, const KickArgs *ka = nullptr);
int gather_grad_sorted(pm_ctx *c, const float *mesh, int C, int zs, long long ms, const float *cot,
                       float cot_scale, float *out);
// acc_j = sum_g W f_d ; alpha_j = sum_g dW (psi + sum_d pi_d f_d); meshes: psi = mesh4[0], f = mesh4[1..3]
int gather_fused_sorted(pm_ctx *c, const float *mesh4, int zs, long long ms, const float *pi, float *acc,
                        float *alpha, const KickArgs *ka = nullptr);

// ---- k-space (pm_kspace.cu) -------------------------------------------------------------------------
int kspace_force(pm_ctx *c, const float2 *rho_k, float2 *f_k /*3 meshes, stride ms/2*/, double nbar);
int kspace_adjoint(pm_ctx *c, const float2 *Pi_k /*3 meshes*/, float2 *psi_k, double nbar);

// ---- own FFT with fused k-space operators (pm_fft.cu) ------------------------------------------------
bool fft_own_supported(const Geometry &g);
size_t fft_own_table_bytes(const Geometry &g);
int fft_own_order_host(int n, int *out);
int fft_own_init(pm_ctx *c);                                  // needs c->ktab, c->fft_tab carved
void fft_own_axis_order(const pm_ctx *c, int axis, std::vector<int> &freq);  // frequency index stored at each memory position
int fft_own_force(pm_ctx *c, float *rho, float *f3, double nbar, int part = 0);     // part: see pm_fft.cu
int fft_own_adjoint(pm_ctx *c, float *Pi3, float *psi, double nbar, int part = 0);

// ---- transforms and k-space operators in fp64 (pm_fft64.cu; pm_params.flags bit 0) -----------------------
size_t fft64_mesh_doubles(const Geometry &g);
size_t fft64_work_bytes(const Geometry &g);
int fft64_init(pm_ctx *c);
void fft64_destroy(pm_ctx *c);
int fft64_force(pm_ctx *c, const float *rho, float *f3, double nbar);
int fft64_adjoint(pm_ctx *c, const float *Pi3, float *psi, double nbar);

// ---- initial conditions (pm_ic.cu) ---------------------------------------------------------------------
void ic_destroy(pm_ctx *c);

// ---- integrator elementwise kernels (pm_integrate.cu) -----------------------------------------------
int state_from_float(pm_ctx *c, const float *s, const float *p);
int state_to_float(pm_ctx *c, float *s, float *p);
// p += acc*K (first), then s += p*D  (K == 0 or D == 0 skip the respective half)
int kick_drift(pm_ctx *c, double K, double D);
// adjoint: p += acc*K; xi -= alpha*K; then s += p*D; pi -= xi*D
int kick_drift_adj(pm_ctx *c, double K, double D);
// r = rho/nbar - 1 - target in place in padded mesh; J into scal[0]
int objective_residual(pm_ctx *c, float *mesh, const float *target, double nbar);
int combine_dJ_ds0(pm_ctx *c, float *out);
int fill_zero(pm_ctx *c, void *ptr, size_t bytes);
int dot_accumulate(pm_ctx *c, const float *a, const float *b, const long long *bfix, double coef, double *acc);
int axpy(pm_ctx *c, long long n, float w, const float *src, float *dst);
int adam_step(pm_ctx *c, long long n, float *w, const float *g, float *m, float *v, int t, double lr, double b1, double b2, double eps);

}  // namespace pm
