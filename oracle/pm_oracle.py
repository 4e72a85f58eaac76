"""ctypes wrapper around oracle/pm_oracle.c -- the CPU fp64 ORACLE.

TEST INFRASTRUCTURE ONLY.  May be imported by tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs; never by the product package
(paper_2211_09815_b200), which must fail loudly when its CUDA library is missing
rather than fall back to anything here.

This file holds no arithmetic of the method: it builds the C file with gcc, declares
the C prototypes and marshals numpy arrays.  Every function is documented, with its
PAPER.md citation, in pm_oracle.c.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pm_oracle.c")
_LIB = os.path.join(_HERE, "libpm_oracle.so")
_lib = None


def build(force=False):
    """Compile pm_oracle.c -> libpm_oracle.so (gcc, OpenMP).  Building is not using."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fcx-limited-range", "-fPIC", "-shared",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _i3(v):
    return (C.c_int * 3)(*[int(t) for t in v])


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_num_threads.restype = C.c_int
        L.orc_growth.argtypes = [C.c_double, C.c_double, _dp]
        L.orc_GD_GK.argtypes = [C.c_double, C.c_double, _dp]
        L.orc_drift_factor.argtypes = [C.c_double] * 4
        L.orc_drift_factor.restype = C.c_double
        L.orc_kick_factor.argtypes = [C.c_double] * 4
        L.orc_kick_factor.restype = C.c_double
        L.orc_fft1d.argtypes = [C.c_int, C.c_void_p, C.c_int]
        L.orc_fft3d.argtypes = [C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_int]
        L.orc_scatter.argtypes = [_ip, C.c_long, _dp, _dp, C.c_int, _dp]
        L.orc_gather.argtypes = [_ip, C.c_long, _dp, _dp, C.c_int, _dp]
        L.orc_gather_grad.argtypes = [_ip, C.c_long, _dp, _dp, C.c_int, _dp, _dp]
        L.orc_force_mesh.argtypes = [_ip, C.c_double, C.c_int, C.c_double, _dp, _dp, _dp]
        L.orc_force_mesh_T.argtypes = [_ip, C.c_double, C.c_int, C.c_double, _dp, _dp]
        L.orc_force.argtypes = [_ip, C.c_double, C.c_int, C.c_long, _dp, _dp, _dp]
        L.orc_force_vjp.argtypes = [_ip, C.c_double, C.c_int, C.c_long, _dp, _dp, _dp]
        L.orc_positions.argtypes = [_ip, _ip, _dp, _dp]
        L.orc_objective.argtypes = [_ip, C.c_long, _dp, _dp, _dp]
        L.orc_objective.restype = C.c_double
        L.orc_init_acc.argtypes = [_ip, _ip, C.c_double, C.c_int, _dp, _dp]
        L.orc_step_fwd.argtypes = [_ip, _ip, C.c_double, C.c_int, _dp, C.c_int, _dp, _dp, _dp]
        L.orc_step_adj.argtypes = [_ip, _ip, C.c_double, C.c_int, _dp, C.c_int] + [_dp] * 6
        L.orc_run_fwd_adj.argtypes = [_ip, _ip, C.c_double, C.c_int, C.c_int, _dp] + [_dp] * 10 + [C.c_int]
        L.orc_run_fwd_adj.restype = C.c_double
        L.orc_run_fwd.argtypes = [_ip, _ip, C.c_double, C.c_int, C.c_int, _dp] + [_dp] * 5
        L.orc_run_fwd.restype = C.c_double
        L.orc_backprop_storeall.argtypes = [_ip, _ip, C.c_double, C.c_int, C.c_int, _dp] + [_dp] * 5
        L.orc_backprop_storeall.restype = C.c_double
        L.orc_growth2.argtypes = [C.c_double, C.c_double, _dp]
        L.orc_ic_factors.argtypes = [C.c_double, C.c_double, _dp]
        L.orc_ic.argtypes = [_ip, _ip] + [C.c_double] * 5 + [C.c_int, _dp, _dp, _dp]
        L.orc_ic.restype = C.c_double
        L.orc_ic_vjp.argtypes = [_ip, _ip] + [C.c_double] * 5 + [C.c_int, _dp, _dp, _dp, _dp]
        L.orc_run_fwd_adj_obs.argtypes = [_ip, _ip, C.c_double, C.c_int, C.c_int, _dp, _dp, _dp, C.c_int, _ip, _dp, _dp] + [_dp] * 6
        L.orc_run_fwd_adj_obs.restype = C.c_double
        _lib = L
    return _lib


def num_threads():
    return lib().orc_num_threads()


# ---- growth ---------------------------------------------------------------------------
def growth(omega_m, a):
    """(D1, D1', D1'') at scale factor a, ' = d/dlna (App. A)."""
    out = np.zeros(3)
    lib().orc_growth(omega_m, a, _d(out))
    return out


def GD_GK(omega_m, a):
    out = np.zeros(2)
    lib().orc_GD_GK(omega_m, a, _d(out))
    return out


def drift_factor(omega_m, ac, aa, ab):
    return lib().orc_drift_factor(omega_m, ac, aa, ab)


def kick_factor(omega_m, ac, aa, ab):
    return lib().orc_kick_factor(omega_m, ac, aa, ab)


def p_over_s(omega_m, a0):
    """G_D(a0)/D1(a0): the Zel'dovich link p0 = (G_D/D1)(a0) s0 (eq. 2 at first order)."""
    return GD_GK(omega_m, a0)[0] / growth(omega_m, a0)[0]


# ---- FFT ------------------------------------------------------------------------------
def fft1d(x, sign=-1):
    y = np.ascontiguousarray(x, dtype=np.complex128).copy()
    lib().orc_fft1d(y.shape[0], y.ctypes.data_as(C.c_void_p), sign)
    return y


def fft3d(x, sign=-1):
    y = np.ascontiguousarray(x, dtype=np.complex128).copy()
    nx, ny, nz = y.shape
    lib().orc_fft3d(nx, ny, nz, y.ctypes.data_as(C.c_void_p), sign)
    return y


# ---- CIC ------------------------------------------------------------------------------
def scatter(N, x, val=None):
    """mesh[C, Nx, Ny, Nz] (C = 1 squeezed when val is None)."""
    x = _f64(x)
    npart = x.shape[0]
    if val is None:
        Cc = 1
    else:
        val = _f64(val).reshape(npart, -1)
        Cc = val.shape[1]
    mesh = np.zeros((Cc,) + tuple(N))
    lib().orc_scatter(_i3(N), npart, _d(x), _d(val), Cc, _d(mesh))
    return mesh[0] if val is None else mesh


def gather(N, x, mesh):
    """mesh [C, Nx, Ny, Nz] or [Nx, Ny, Nz] -> out [np, C]."""
    x = _f64(x)
    mesh = _f64(mesh)
    if mesh.ndim == 3:
        mesh = mesh[None]
    Cc = mesh.shape[0]
    out = np.zeros((x.shape[0], Cc))
    lib().orc_gather(_i3(N), x.shape[0], _d(x), _d(mesh), Cc, _d(out))
    return out


def gather_grad(N, x, mesh, cot=None):
    x = _f64(x)
    mesh = _f64(mesh)
    if mesh.ndim == 3:
        mesh = mesh[None]
    Cc = mesh.shape[0]
    if cot is not None:
        cot = _f64(cot).reshape(x.shape[0], Cc)
    out = np.zeros((x.shape[0], 3))
    lib().orc_gather_grad(_i3(N), x.shape[0], _d(x), _d(mesh), Cc, _d(cot), _d(out))
    return out


# ---- force ----------------------------------------------------------------------------
def force_mesh(N, omega_m, rho, nbar, deconv=0, return_imag=False):
    rho = _f64(rho)
    f = np.zeros((3,) + tuple(N))
    im = C.c_double(0.0)
    lib().orc_force_mesh(_i3(N), omega_m, deconv, nbar, _d(rho), _d(f), C.byref(im))
    return (f, im.value) if return_imag else f


def force_mesh_T(N, omega_m, Pi, nbar, deconv=0):
    Pi = _f64(Pi)
    psi = np.zeros(tuple(N))
    lib().orc_force_mesh_T(_i3(N), omega_m, deconv, nbar, _d(Pi), _d(psi))
    return psi


def force(N, omega_m, x, deconv=0, return_mesh=False):
    x = _f64(x)
    acc = np.zeros_like(x)
    fm = np.zeros((3,) + tuple(N)) if return_mesh else None
    lib().orc_force(_i3(N), omega_m, deconv, x.shape[0], _d(x), _d(acc), _d(fm))
    return (acc, fm) if return_mesh else acc


def force_vjp(N, omega_m, x, pi, deconv=0):
    x = _f64(x)
    pi = _f64(pi)
    alpha = np.zeros_like(x)
    lib().orc_force_vjp(_i3(N), omega_m, deconv, x.shape[0], _d(x), _d(pi), _d(alpha))
    return alpha


# ---- lattice / objective --------------------------------------------------------------
def positions(N, L, s):
    s = _f64(s)
    x = np.zeros_like(s)
    lib().orc_positions(_i3(N), _i3(L), _d(s), _d(x))
    return x


def objective(N, x, delta_target, want_xi=True):
    x = _f64(x)
    dt = _f64(delta_target)
    xi = np.zeros_like(x) if want_xi else None
    J = lib().orc_objective(_i3(N), x.shape[0], _d(x), _d(dt), _d(xi))
    return (J, xi) if want_xi else J


# ---- integrator -----------------------------------------------------------------------
def init_acc(N, L, omega_m, s, deconv=0):
    s = _f64(s)
    acc = np.zeros_like(s)
    lib().orc_init_acc(_i3(N), _i3(L), omega_m, deconv, _d(s), _d(acc))
    return acc


def step_fwd(N, L, omega_m, a, i, s, p, acc, deconv=0):
    """In place on float64 contiguous s, p, acc."""
    a = _f64(a)
    lib().orc_step_fwd(_i3(N), _i3(L), omega_m, deconv, _d(a), i, _d(s), _d(p), _d(acc))


def step_adj(N, L, omega_m, a, i, s, p, acc, xi, pi, alpha, deconv=0):
    a = _f64(a)
    lib().orc_step_adj(_i3(N), _i3(L), omega_m, deconv, _d(a), i,
                       _d(s), _d(p), _d(acc), _d(xi), _d(pi), _d(alpha))


def run_fwd_adj(N, L, omega_m, a, s0, p0, delta_target, deconv=0, n_adj=-1):
    a = _f64(a)
    n = a.shape[0] - 1
    s0 = _f64(s0)
    p0 = _f64(p0)
    dt = _f64(delta_target)
    out = {k: np.zeros_like(s0) for k in ("s_n", "p_n", "xi0", "pi0", "dJ_ds0", "s_rec", "p_rec")}
    J = lib().orc_run_fwd_adj(_i3(N), _i3(L), omega_m, deconv, n, _d(a), _d(s0), _d(p0), _d(dt),
                              _d(out["s_n"]), _d(out["p_n"]), _d(out["xi0"]), _d(out["pi0"]),
                              _d(out["dJ_ds0"]), _d(out["s_rec"]), _d(out["p_rec"]), n_adj)
    out["J"] = J
    return out


def run_fwd(N, L, omega_m, a, s0, p0, delta_target=None, deconv=0):
    a = _f64(a)
    n = a.shape[0] - 1
    s0 = _f64(s0)
    p0 = _f64(p0)
    dt = _f64(delta_target)
    s_n = np.zeros_like(s0)
    p_n = np.zeros_like(s0)
    J = lib().orc_run_fwd(_i3(N), _i3(L), omega_m, deconv, n, _d(a), _d(s0), _d(p0), _d(dt),
                          _d(s_n), _d(p_n))
    return s_n, p_n, J


def backprop_storeall(N, L, omega_m, a, s0, p0, delta_target, deconv=0):
    a = _f64(a)
    n = a.shape[0] - 1
    s0 = _f64(s0)
    p0 = _f64(p0)
    dt = _f64(delta_target)
    xi0 = np.zeros_like(s0)
    pi0 = np.zeros_like(s0)
    J = lib().orc_backprop_storeall(_i3(N), _i3(L), omega_m, deconv, n, _d(a), _d(s0), _d(p0), _d(dt),
                                    _d(xi0), _d(pi0))
    return J, xi0, pi0


# ---- initial conditions from white noise (eq. 2-6, eq. 51) ----
def growth2(omega_m, a):
    """[D2, dD2/dlna] (eq. A5 second line, A6, A8)."""
    out = np.zeros(2)
    lib().orc_growth2(omega_m, a, _d(out))
    return out


def ic_factors(omega_m, a0):
    """[D1, D2, a^2 E D1', a^2 E D2'] at a0: the four time factors of eq. 2."""
    out = np.zeros(4)
    lib().orc_ic_factors(omega_m, a0, _d(out))
    return out


def ic(N, L, omega_m, a0, amp, omega, order=2, ns=-1.5, rc=2.0, return_imag=False):
    """white noise omega[Lx, Ly, Lz] -> (s0[np, 3], p0[np, 3]) by 1LPT / 2LPT."""
    om = _f64(omega).reshape(-1)
    s0 = np.zeros((om.shape[0], 3))
    p0 = np.zeros_like(s0)
    im = lib().orc_ic(_i3(N), _i3(L), omega_m, a0, amp, ns, rc, order, _d(om), _d(s0), _d(p0))
    return (s0, p0, im) if return_imag else (s0, p0)


def ic_vjp(N, L, omega_m, a0, amp, omega, xi0, pi0, order=2, ns=-1.5, rc=2.0):
    """dJ/d omega [np] = xi0 . ds0/domega + pi0 . dp0/domega."""
    om = _f64(omega).reshape(-1)
    out = np.zeros_like(om)
    lib().orc_ic_vjp(_i3(N), _i3(L), omega_m, a0, amp, ns, rc, order, _d(om), _d(_f64(xi0)), _d(_f64(pi0)), _d(out))
    return out


# ---- observations between the steps, dJ/dOmega_m (eq. 49 last lines, eq. 51 first line) ----
def run_fwd_adj_obs(N, L, omega_m, a, s0, p0, obs_steps, obs_weights, targets, deconv=0):
    """J = sum_k w_k J_k(x_{i_k}); returns s_n, p_n, xi0, pi0, J, J_obs[k], dJ_dOm (loop part of eq. 51)."""
    a = _f64(a)
    n = a.shape[0] - 1
    s0 = _f64(s0)
    p0 = _f64(p0)
    steps = np.ascontiguousarray(obs_steps, dtype=np.int32)
    w = _f64(obs_weights)
    t = _f64(targets).reshape(len(steps), -1)
    out = {k: np.zeros_like(s0) for k in ("s_n", "p_n", "xi0", "pi0")}
    J_obs = np.zeros(len(steps))
    dth = np.zeros(1)
    J = lib().orc_run_fwd_adj_obs(_i3(N), _i3(L), omega_m, deconv, n, _d(a), _d(s0), _d(p0), len(steps),
                                  steps.ctypes.data_as(_ip), _d(w), _d(t), _d(out["s_n"]), _d(out["p_n"]),
                                  _d(out["xi0"]), _d(out["pi0"]), _d(J_obs), _d(dth))
    out.update(J=J, J_obs=J_obs, dJ_dOm=float(dth[0]))
    return out


# ---- Adam and the optimisation loop of the paper's Fig. 4 (L482-488), written out plainly (numpy, fp64) ----
def adam_step(w, g, m, v, t, lr=0.1, beta1=0.9, beta2=0.999, eps=1e-8):
    """Kingma & Ba (2015), Algorithm 1; returns the new (w, m, v).  t = 1, 2, ..."""
    m = beta1 * m + (1.0 - beta1) * g
    v = beta2 * v + (1.0 - beta2) * g * g
    mhat = m / (1.0 - beta1 ** t)
    vhat = v / (1.0 - beta2 ** t)
    return w - lr * mhat / (np.sqrt(vhat) + eps), m, v


def optimize_ic(N, L, omega_m, a, omega, target, amp, n_iter, lr=0.1, order=2, ns=-1.5, rc=2.0):
    """omega -> ic -> run_fwd_adj -> ic_vjp -> Adam, n_iter times; returns (omega_final, J history before each update)."""
    w = _f64(omega).reshape(-1).copy()
    m = np.zeros_like(w)
    v = np.zeros_like(w)
    hist = []
    for t in range(1, n_iter + 1):
        s0, p0 = ic(N, L, omega_m, a[0], amp, w.reshape(L), order=order, ns=ns, rc=rc)
        out = run_fwd_adj(N, L, omega_m, a, s0, p0, target)
        g = ic_vjp(N, L, omega_m, a[0], amp, w.reshape(L), out["xi0"], out["pi0"], order=order, ns=ns, rc=rc)
        hist.append(out["J"])
        w, m, v = adam_step(w, g, m, v, t, lr)
    return w.reshape(L), hist
