/*
 * pm.h -- C ABI of libpm: the data-parallel hot path of the adjoint particle-mesh method of
 * "Differentiable Cosmological Simulation with the Adjoint Method" (arxiv 2211.09815),
 * hand-written CUDA for sm_100a (B200).  The 3-D transforms are the library's own passes on power-of-two
 * meshes from 16 to 1024 per axis (k-space operators fused in) and cuFFT's on every other mesh.
 *
 * Citations are /root/reference/PAPER.md line numbers (L..) with the equation they fall in.
 *
 * Conventions:
 *   - units: length = one mesh cell (l = 1 in eq. 10), time = 1/H0;
 *   - arrays are row-major; particle j = (jx*Ly + jy)*Lz + jz sits on lattice site
 *     q_j = (jx, jy, jz) * (mesh/lattice) cells (eq. 1); x = q + s is formed inside kernels;
 *   - real meshes handed over this ABI are UNPADDED [C][Nx][Ny][Nz] fp32, mesh point g at coordinate g;
 *   - every pointer named dev_* is a CUDA DEVICE pointer owned by the CALLER (e.g. a torch tensor),
 *     4-byte aligned at least; host_* is a HOST pointer.  The library never allocates or frees
 *     device memory except cuFFT's plan-internal scratch when no workspace is large enough (it
 *     is not: the work area comes from the caller's workspace, see pm_workspace_bytes);
 *   - every call enqueues its kernels on the ctx's stream and returns WITHOUT synchronising,
 *     except where noted.  Return value: PM_OK or a negative error code; nothing is enqueued
 *     when an argument error is returned.  No exception or abort crosses the ABI.
 *   - calls on one ctx are not thread-safe; separate ctxs are independent.
 *   - device memory = caller's tensors + pm_workspace_bytes(), a function of (mesh, lattice)
 *     only: it never depends on n_steps (L37, L400-402: no stored history).
 */
#ifndef PM_H_
#define PM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pm_ctx pm_ctx; /* opaque, host memory owned by the library */

typedef struct {
    int32_t mesh[3];     /* Nx, Ny, Nz mesh points per axis; each >= 2, Nz even; each <= 4096       */
    int32_t lattice[3];  /* particle lattice Lx, Ly, Lz; N_p = product; (mesh[d] << 32) % lattice[d] == 0
                            (true whenever lattice divides mesh, the case of every config)            */
    double omega_m;      /* flat matter + Lambda: Omega_Lambda = 1 - omega_m; 1.0 = Einstein-de Sitter */
    int32_t n_steps;     /* n >= 0 KDK steps                                                           */
    const double *a;     /* HOST: n_steps + 1 scale factors, strictly increasing, copied by pm_init     */
    int32_t deconvolve;  /* 0 = eq. 11 as printed (L127-131); 1 = also divide by the CIC window^2,
                            prod_d sinc(k_d/2)^-4 (reading R12; not in the paper)            */
    int32_t flags;       /* 0, or PM_FLAG_FP64_TRANSFORMS (below); any other bit is PM_EINVAL           */
} pm_params;

/* pm_params.flags.  PM_FLAG_FP64_TRANSFORMS: the 3-D transforms and the k-space operators of eq. 11 (L127-131) and of
   its transpose run in double precision (cuFFT D2Z / Z2D + fp64 kernels) -- the paper's "more precise floating-point
   numbers" remedy (L371; fp64 rows of Tables 1-2) applied to the one stage whose fp32 rounding limits the
   gradient (precision A/B).  Every particle and mesh array crossing the ABI stays fp32; the
   workspace grows by four fp64 meshes plus cuFFT's work area.  Slower; results stay bit-reproducible and reversible. */
enum { PM_FLAG_FP64_TRANSFORMS = 1 };

enum {
    PM_OK = 0,
    PM_EINVAL = -1,     /* bad argument (NULL, misaligned, sizes, non-monotone a, ...)                 */
    PM_EWORKSPACE = -2, /* dev_workspace too small or misaligned (needs 256-byte alignment)            */
    PM_ECUDA = -3,      /* a CUDA runtime call or kernel launch failed                                 */
    PM_ECUFFT = -4,     /* a cuFFT call failed                                                         */
    PM_ESTATE = -5      /* call out of order (e.g. pm_step_fwd(i) when the state is not at t_{i-1})    */
};

/* text for an error code; never NULL */
const char *pm_strerror(int code);
/* text of the last error recorded on ctx (includes the failing CUDA/cuFFT call); never NULL */
const char *pm_last_error(const pm_ctx *ctx);

/* Bytes of device workspace pm_init needs for these params.  Pure host query. */
int pm_workspace_bytes(const pm_params *params, size_t *bytes);

/* Create a context: validates params, precomputes the per-step drift/kick factors D, K in fp64 on
 * the host (eq. 15 L165-167 with G_D, G_K of eq. A7), carves dev_workspace (256-byte aligned,
 * >= pm_workspace_bytes) into meshes / sort buffers / integrator state / cuFFT work area, and
 * creates the cuFFT plans on cuda_stream (a cudaStream_t, may be NULL = default stream).  */
int pm_init(pm_ctx **out, const pm_params *params, void *dev_workspace, size_t bytes, void *cuda_stream);
/* Destroys the cuFFT plans and the host struct.  Does not touch dev_workspace. */
int pm_destroy(pm_ctx *ctx);

/* Host scalars (fp64); pure host functions, no GPU needed: */
/*   out[0..3] = D1, dD1/dlna, G_D = a^2 E D1', G_K = 1.5 Om D1 at scale factor a (App. A; eq. A7) */
int pm_host_growth(double omega_m, double a, double out[4]);
/*   the three factors of a forward KDK step a_prev -> a_next (eq. 16; eq. 15), with
 *   a_half = (a_prev + a_next)/2: out = {K(a_prev; a_prev, a_half), D(a_half; a_prev, a_next), K(a_next; a_half, a_next)} */
int pm_host_step_factors(double omega_m, double a_prev, double a_next, double out[3]);
/*   memory order of the library's own FFT passes along an axis of n points (n a power of two, 8 <= n <= 1024):
 *   out[p] = frequency index (0 .. n-1, e^{-2 pi i k g / n} convention) that memory position p holds after the
 *   forward decimation-in-frequency stages (radix 16, or 8 where a radix-2 stage would otherwise remain).  Pure host; the k-space tables are
 *   built from it and nothing in k-space crosses this ABI (R26). */
int pm_host_fft_order(int32_t n, int32_t *out);
/*   the factors stored in ctx for forward step i in 1..n; the adjoint step uses their exact negatives (L389) */
int pm_step_factors(const pm_ctx *ctx, int i, double out[3]);

/* ---- stand-alone particle <-> mesh operations (eq. 10; L133; VJPs L410) ----------------
 * dev_x[np][3]: ABSOLUTE positions in cells, any finite value (wrapped periodically); np <= N_p of ctx
 * (the sort buffers are sized for N_p).  Positions are binned by mesh tile (counting sort) first.     */

/* mesh_c(g) = sum_j val_{j,c} W(g, x_j); dev_val[np][C] or NULL (= unit mass, C must be 1); C in {1,3}.
 * dev_mesh[C][Nx][Ny][Nz] is OVERWRITTEN (no need to zero it). */
int pm_scatter(pm_ctx *ctx, int64_t np, const float *dev_x, const float *dev_val, int C, float *dev_mesh);
/* out_{j,c} = sum_g W(g, x_j) mesh_c(g); C in {1,3}; dev_out[np][C] */
int pm_gather(pm_ctx *ctx, int64_t np, const float *dev_x, const float *dev_mesh, int C, float *dev_out);
/* out_{j,e} = sum_c cot_{j,c} sum_g dW(g, x_j)/dx_e mesh_c(g); dev_cot[np][C] or NULL (= 1); dev_out[np][3].
 * This is the position-VJP of both pm_scatter and pm_gather (L410).  C in {1,3}. */
int pm_gather_grad(pm_ctx *ctx, int64_t np, const float *dev_x, const float *dev_mesh, int C,
                   const float *dev_cot, float *dev_out);
/* acc = F(x) (L111-133): scatter -> R2C -> Green's function * spectral gradient (eq. 11) -> 3 C2R -> gather.
 * nbar = np / N_g.  dev_acc[np][3]. */
int pm_force(pm_ctx *ctx, int64_t np, const float *dev_x, float *dev_acc);
/* alpha = pi . d acc / d x (the force VJP "alpha" of eq. 49, L393/L397); dev_pi, dev_alpha [np][3].
 * If dev_acc != NULL it also receives F(x). */
int pm_force_vjp(pm_ctx *ctx, int64_t np, const float *dev_x, const float *dev_pi, float *dev_acc,
                 float *dev_alpha);

/* ---- state-carrying reversible integrator (eq. 16; eq. 49-50) ------------------------
 * The state (s, p, acc) and the adjoint variables (xi, pi, alpha) live inside the workspace; s and p
 * are held in fixed point so that every kick and drift is undone EXACTLY by the reverse pass
 * (DESIGN.md "Reversibility"): absolute position int64 at 2^-32 cell, momentum int64 at 2^-36.       */

/* copy in s0, p0 [N_p][3] (displacement in cells, canonical momentum p = a^2 dx/dt in cells*H0),
 * set the time index to 0 and compute acc_0 = F(q + s_0) (L175) */
int pm_set_state(pm_ctx *ctx, const float *dev_s, const float *dev_p);
/* read back the current state as fp32; any pointer may be NULL */
int pm_get_state(pm_ctx *ctx, float *dev_s, float *dev_p, float *dev_acc);
/* forward KDK step t_{i-1} -> t_i (eq. 16); i must equal the current time index + 1 */
int pm_step_fwd(pm_ctx *ctx, int i);
/* objective on the current state (BASELINE.json configs; L478): r = rho/nbar - 1 - delta_target,
 * J = 1/2 sum_g r^2 accumulated in fp64; sets xi = dJ/dx (scatter VJP), pi = 0, alpha = 0 (eq. 50).
 * dev_delta_target[Nx][Ny][Nz] unpadded.  J stays on the device until pm_get_objective. */
int pm_objective(pm_ctx *ctx, const float *dev_delta_target);
/* SYNCHRONISES the stream and returns J */
int pm_get_objective(pm_ctx *ctx, double *host_J);
/* alternative to pm_objective: caller-provided adjoint initial conditions (eq. 50); computes
 * alpha = VJP(x, pi) at the current state unless dev_pi == NULL (pi = 0, alpha = 0) */
int pm_set_adjoint(pm_ctx *ctx, const float *dev_xi, const float *dev_pi);
/* adjoint step t_i -> t_{i-1} with reverse-time integration of the state (eq. 49); i must equal the
 * current time index */
int pm_step_adj(pm_ctx *ctx, int i);
/* read xi, pi (any may be NULL) and dJ/ds0 = xi + pi * G_D(a_0)/D1(a_0) (eq. 51 restricted to
 * Zel'dovich initial conditions p0 = (G_D/D1) s0, reading R18); all [N_p][3] */
int pm_get_adjoint(pm_ctx *ctx, float *dev_xi, float *dev_pi, float *dev_dJ_ds0);

/* Whole run (L400-408): set_state, n forward steps, objective, n adjoint steps.  Outputs (any may be
 * NULL): final state s_n, p_n; J (HOST; the call SYNCHRONISES once, at the end); xi_0, pi_0, dJ/ds0;
 * and the state (s, p) reconstructed at t_0 by the reverse integration (equals the input up to the
 * fixed-point quantisation of pm_set_state). */
int pm_run_fwd_adj(pm_ctx *ctx, const float *dev_s0, const float *dev_p0, const float *dev_delta_target,
                   float *dev_s_n, float *dev_p_n, double *host_J, float *dev_xi0, float *dev_pi0,
                   float *dev_dJ_ds0, float *dev_s_rec, float *dev_p_rec);
/* Same through HOST buffers: copies s0, p0, delta_target host->device, runs, copies every non-NULL
 * output device->host, synchronises.  Uses only workspace memory for staging.  When host_s_rec / host_p_rec are
 * requested the adjoint variables inside the ctx are overwritten (pm_get_adjoint then returns PM_ESTATE). */
int pm_run_fwd_adj_host(pm_ctx *ctx, const float *host_s0, const float *host_p0,
                        const float *host_delta_target, float *host_s_n, float *host_p_n, double *host_J,
                        float *host_xi0, float *host_pi0, float *host_dJ_ds0, float *host_s_rec, float *host_p_rec);

/* ---- observations between the steps and the cosmological-parameter gradient (eq. 49 last lines L393; eq. 51) ----
 * J = sum_k w_k J_k, J_k = 1/2 sum_g (delta(x_{i_k}) - target_k)^2 on the snapshots i_k in 0..n (host_obs_step, any order,
 * n_obs <= PM_MAX_OBS; dev_targets[n_obs][Nx][Ny][Nz]): the observation operator O_{i-1} of eq. 49 adds w_k dJ_k/dx to
 * xi_{i-1} between adjoint steps.  host_J = J, host_J_obs[k] = J_k (may be NULL).  host_dJ_dOm (may be NULL): the loop
 * part of eq. 51's first line for theta = Omega_m at fixed (s0, p0) -- sum over the steps of
 * (pi.acc d/dOm + zeta) K + xi.p dD/dOm with zeta = pi . d acc/d Om = pi.acc / Om (eq. 11 is linear in Om) and the
 * factor derivatives by central differences on the host; requesting it runs the adjoint steps unchained.
 * Other arguments and the single final synchronisation as pm_run_fwd_adj. */
enum { PM_MAX_OBS = 64 };
int pm_run_fwd_adj_obs(pm_ctx *ctx, const float *dev_s0, const float *dev_p0, int n_obs, const int32_t *host_obs_step,
                       const double *host_obs_w, const float *dev_targets, float *dev_s_n, float *dev_p_n,
                       double *host_J, double *host_J_obs, float *dev_xi0, float *dev_pi0, float *dev_dJ_ds0,
                       double *host_dJ_dOm);

/* ---- initial conditions from white noise, and dJ/d(omega) (eq. 2-6; eq. 51 second line L406) ----------------
 * dev_omega[Lx][Ly][Lz]: real white noise on the particle lattice (L89).  delta_1(k) = amp sqrt(P(k)) omega(k) with
 * P(k) = k^ns exp(-(rc k)^2), k in radians per mesh cell (eq. 6; the volume factor is part of amp; the configs' recipe is
 * ns = -1.5, rc = 2).  order 1: s0 = D1 s1, p0 = a^2 H D1' s1 (Zel'dovich); order 2 adds D2 s2, a^2 H D2' s2 (2LPT, eq. 2-4)
 * at a_0 = the ctx's first scale factor.  Transforms run on the lattice (cuFFT), the multipliers in fp64 per mode.
 * Both calls use the ctx's mesh buffers as scratch: call them outside a run (the integrator state is invalidated;
 * pm_set_state / pm_run_fwd_adj start a new one).  Outputs dev_s0, dev_p0 [N_p][3]; dev_domega [Lx][Ly][Lz]. */
int pm_ic_fwd(pm_ctx *ctx, const float *dev_omega, double amp, double ns, double rc, int order, float *dev_s0,
              float *dev_p0);
/* dev_domega = xi0 . d s0 / d omega + pi0 . d p0 / d omega: with (xi0, pi0) of pm_run_fwd_adj this is dJ/d omega. */
int pm_ic_vjp(pm_ctx *ctx, const float *dev_omega, double amp, double ns, double rc, int order, const float *dev_xi0,
              const float *dev_pi0, float *dev_domega);
/* Host: out = {D1, D2, a^2 E D1', a^2 E D2'} at a0, the four time factors of eq. 2 (D2 by RK4 on eq. A1). */
int pm_host_ic_factors(double omega_m, double a0, double out[4]);

/* ---- optimisation of the initial conditions (the paper's second workload, Fig. 4) ----------------------
 * One Adam update (Kingma & Ba 2015; the paper uses it with learning rate 0.1): t = 1, 2, ... is the iteration number,
 * dev_m / dev_v the running first / second moments (zero before t = 1), all arrays [n] floats. */
int pm_adam_step(pm_ctx *ctx, int64_t n, float *dev_w, const float *dev_g, float *dev_m, float *dev_v, int t, double lr,
                 double beta1, double beta2, double eps);
/* n_iter iterations of  omega -> pm_ic_fwd -> pm_run_fwd_adj (J, xi0, pi0) -> pm_ic_vjp (dJ/d omega) -> Adam(lr, 0.9,
 * 0.999, 1e-8) on the white-noise field dev_omega[Lx][Ly][Lz] (updated in place), towards dev_delta_target (the mesh
 * objective of pm_objective).  host_J_history[n_iter] (may be NULL) receives J BEFORE each update.  dev_scratch: at least
 * pm_optimize_ic_scratch_bytes(ctx) bytes of device memory owned by the caller.  Synchronises once per iteration (J).
 * No checkpoints are needed (L371, L381): the reverse pass retraces the forward one bit for bit. */
size_t pm_optimize_ic_scratch_bytes(const pm_ctx *ctx);
int pm_optimize_ic(pm_ctx *ctx, float *dev_omega, const float *dev_delta_target, double amp, double ns, double rc, int order,
                   int n_iter, double lr, void *dev_scratch, size_t scratch_bytes, double *host_J_history);

/* ---- an entry point that allocates nothing ---------------------------------------------------------------------------
 * pm_objective's reduction on caller-provided flat arrays, for callers that cannot allocate (CUDA graph capture, serving
 * loops): r_i = rho_i / nbar - 1 - delta_target_i, *dev_J = 1/2 sum_i r_i^2 (fp64, fixed order: bit-reproducible);
 * dev_resid[n] receives r when not NULL (may alias dev_rho).  No ctx, no workspace, no cudaMalloc / cudaFree: the per-block
 * partial sums live in a static device array of 128 KB that every GPU loading the library holds until exit, which limits
 * n to PM_NOALLOC_MAX_N (a 1024^3 mesh); larger n is PM_EINVAL with the limit in pm_last_error(NULL).  Enqueues two
 * kernels on cuda_stream and returns without synchronising.  All calls on a device share that array: calls that overlap
 * on the GPU (different streams, unordered) race on it -- order them.  pm_noalloc_setup resolves the array's device
 * address for the CURRENT device (the first pm_objective_noalloc on a device does it itself; call it beforehand where the
 * first call would fall inside a graph capture). */
#define PM_NOALLOC_MAX_N (1ll << 30)
int pm_noalloc_setup(void);
int pm_objective_noalloc(int64_t n, const float *dev_rho, const float *dev_delta_target, double nbar, float *dev_resid,
                         double *dev_J, void *cuda_stream);

/* ---- instrumentation ---------------------------------------------------------------------------------
 * When enabled, every kernel launch / cuFFT call of the library is bracketed by CUDA events on the
 * ctx's stream.  pm_timing_read SYNCHRONISES, sums the elapsed time per kernel class since the last
 * pm_timing_reset and returns how many classes there are.  names[k] points at static strings. */
enum { PM_TIMING_MAX_CLASSES = 32 };
int pm_timing_enable(pm_ctx *ctx, int on);
int pm_timing_reset(pm_ctx *ctx);
int pm_timing_read(pm_ctx *ctx, int max_classes, const char **names, double *ms, int64_t *launches,
                   double *algo_bytes);
/* number of kernels (own + cuFFT calls) launched on this ctx since pm_init */
int pm_launch_count(const pm_ctx *ctx, int64_t *own_kernels, int64_t *cufft_calls);

#ifdef __cplusplus
}
#endif
#endif /* PM_H_ */
