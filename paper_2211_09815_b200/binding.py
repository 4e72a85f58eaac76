"""Thin ctypes binding of libpm.so (include/pm.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; torch is used for device memory and the
stream.  There is NO CPU fallback: importing this module raises if libpm.so is missing, and every
call raises PMError on a non-zero return code.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# PM_LIB selects another build of the same library (e.g. the probe build libpm_debug.so of build.py --debug)
LIB_PATH = os.environ.get("PM_LIB") or os.path.join(_HERE, "libpm.so")

if not os.path.exists(LIB_PATH):
    # a fresh checkout on a box with nvcc: compile once (under a lock, ranks may import concurrently); never a fallback
    try:
        import fcntl
        from . import build as _build
        with open(os.path.join(_HERE, ".build.lock"), "w") as _lk:
            fcntl.flock(_lk, fcntl.LOCK_EX)
            if not os.path.exists(LIB_PATH):
                _build.build(force=True)
    except Exception:  # noqa: BLE001  (reported just below)
        pass
if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python -m paper_2211_09815_b200.build` "
        "(nvcc, sm_100a). There is no CPU fallback.")
_lib = C.CDLL(LIB_PATH)


class pm_params(C.Structure):
    _fields_ = [("mesh", C.c_int32 * 3), ("lattice", C.c_int32 * 3), ("omega_m", C.c_double),
                ("n_steps", C.c_int32), ("a", C.POINTER(C.c_double)), ("deconvolve", C.c_int32),
                ("flags", C.c_int32)]


PM_OK, PM_EINVAL, PM_EWORKSPACE, PM_ECUDA, PM_ECUFFT, PM_ESTATE = 0, -1, -2, -3, -4, -5
PM_TIMING_MAX_CLASSES = 32
PM_FLAG_FP64_TRANSFORMS = 1

_vp, _i64, _int, _dbl = C.c_void_p, C.c_int64, C.c_int, C.c_double
_SIGS = {
    "pm_strerror": (C.c_char_p, [_int]),
    "pm_last_error": (C.c_char_p, [_vp]),
    "pm_workspace_bytes": (_int, [C.POINTER(pm_params), C.POINTER(C.c_size_t)]),
    "pm_init": (_int, [C.POINTER(_vp), C.POINTER(pm_params), _vp, C.c_size_t, _vp]),
    "pm_destroy": (_int, [_vp]),
    "pm_host_growth": (_int, [_dbl, _dbl, C.POINTER(_dbl)]),
    "pm_host_step_factors": (_int, [_dbl, _dbl, _dbl, C.POINTER(_dbl)]),
    "pm_step_factors": (_int, [_vp, _int, C.POINTER(_dbl)]),
    "pm_host_fft_order": (_int, [C.c_int32, C.POINTER(C.c_int32)]),
    "pm_host_ic_factors": (_int, [_dbl, _dbl, C.POINTER(_dbl)]),
    "pm_ic_fwd": (_int, [_vp, _vp, _dbl, _dbl, _dbl, _int, _vp, _vp]),
    "pm_ic_vjp": (_int, [_vp, _vp, _dbl, _dbl, _dbl, _int, _vp, _vp, _vp]),
    "pm_run_fwd_adj_obs": (_int, [_vp, _vp, _vp, _int, C.POINTER(C.c_int32), C.POINTER(_dbl), _vp, _vp, _vp,
                                  C.POINTER(_dbl), C.POINTER(_dbl), _vp, _vp, _vp, C.POINTER(_dbl)]),
    "pm_adam_step": (_int, [_vp, _i64, _vp, _vp, _vp, _vp, _int, _dbl, _dbl, _dbl, _dbl]),
    "pm_optimize_ic_scratch_bytes": (C.c_size_t, [_vp]),
    "pm_optimize_ic": (_int, [_vp, _vp, _vp, _dbl, _dbl, _dbl, _int, _int, _dbl, _vp, C.c_size_t, C.POINTER(_dbl)]),
    "pm_noalloc_setup": (_int, []),
    "pm_objective_noalloc": (_int, [_i64, _vp, _vp, _dbl, _vp, _vp, _vp]),
    "pm_scatter": (_int, [_vp, _i64, _vp, _vp, _int, _vp]),
    "pm_gather": (_int, [_vp, _i64, _vp, _vp, _int, _vp]),
    "pm_gather_grad": (_int, [_vp, _i64, _vp, _vp, _int, _vp, _vp]),
    "pm_force": (_int, [_vp, _i64, _vp, _vp]),
    "pm_force_vjp": (_int, [_vp, _i64, _vp, _vp, _vp, _vp]),
    "pm_set_state": (_int, [_vp, _vp, _vp]),
    "pm_get_state": (_int, [_vp, _vp, _vp, _vp]),
    "pm_step_fwd": (_int, [_vp, _int]),
    "pm_objective": (_int, [_vp, _vp]),
    "pm_get_objective": (_int, [_vp, C.POINTER(_dbl)]),
    "pm_set_adjoint": (_int, [_vp, _vp, _vp]),
    "pm_step_adj": (_int, [_vp, _int]),
    "pm_get_adjoint": (_int, [_vp, _vp, _vp, _vp]),
    "pm_run_fwd_adj": (_int, [_vp] + [_vp] * 5 + [C.POINTER(_dbl)] + [_vp] * 5),
    "pm_run_fwd_adj_host": (_int, [_vp] + [_vp] * 5 + [C.POINTER(_dbl)] + [_vp] * 5),
    "pm_timing_enable": (_int, [_vp, _int]),
    "pm_timing_reset": (_int, [_vp]),
    "pm_timing_read": (_int, [_vp, _int, C.POINTER(C.c_char_p), C.POINTER(_dbl), C.POINTER(_i64), C.POINTER(_dbl)]),
    "pm_launch_count": (_int, [_vp, C.POINTER(_i64), C.POINTER(_i64)]),
}
EXPORTS = tuple(_SIGS)
for _name, (_res, _args) in _SIGS.items():
    _f = getattr(_lib, _name)  # AttributeError here = the library does not export what pm.h declares
    _f.restype = _res
    _f.argtypes = _args


class PMError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"libpm error {code}: {text}")
        self.code = code


def make_params(mesh, lattice, omega_m, a, deconvolve=0, flags=0):
    """Returns (pm_params, keepalive) -- keepalive owns the host array params.a points at."""
    a = [float(v) for v in a]
    arr = (C.c_double * len(a))(*a)
    p = pm_params()
    p.mesh[:] = [int(v) for v in mesh]
    p.lattice[:] = [int(v) for v in lattice]
    p.omega_m = float(omega_m)
    p.n_steps = len(a) - 1
    p.a = C.cast(arr, C.POINTER(C.c_double))
    p.deconvolve = int(deconvolve)
    p.flags = int(flags)
    return p, arr


def host_growth(omega_m, a):
    """[D1, dD1/dlna, G_D, G_K] at scale factor a (pure host)."""
    out = (_dbl * 4)()
    rc = _lib.pm_host_growth(float(omega_m), float(a), out)
    if rc != PM_OK:
        raise PMError(rc, "pm_host_growth")
    return list(out)


def host_step_factors(omega_m, a_prev, a_next):
    """[K1, D, K2] of the forward KDK step a_prev -> a_next (pure host)."""
    out = (_dbl * 3)()
    rc = _lib.pm_host_step_factors(float(omega_m), float(a_prev), float(a_next), out)
    if rc != PM_OK:
        raise PMError(rc, "pm_host_step_factors")
    return list(out)


def host_ic_factors(omega_m, a0):
    """[D1, D2, a^2 E D1', a^2 E D2'] at a0: the time factors of eq. 2 (pure host)."""
    out = (_dbl * 4)()
    rc = _lib.pm_host_ic_factors(float(omega_m), float(a0), out)
    if rc != PM_OK:
        raise PMError(rc, "pm_host_ic_factors")
    return list(out)


PM_NOALLOC_MAX_N = 1 << 30


def objective_noalloc(rho, delta_target, nbar, J, resid=None, stream=None):
    """pm_objective_noalloc: J[0] (float64 CUDA tensor of the caller) = 1/2 sum (rho / nbar - 1 - delta_target)^2 over the
    flat arrays; libpm allocates nothing for it (static device scratch, n <= PM_NOALLOC_MAX_N).  Asynchronous."""
    st = stream if stream is not None else torch.cuda.current_stream(rho.device)
    rc = _lib.pm_objective_noalloc(rho.numel(), _ptr(rho, "rho"), _ptr(delta_target, "delta_target"), float(nbar),
                                   _ptr(resid, "resid"), _ptr(J, "J", torch.float64), st.cuda_stream)
    if rc != PM_OK:
        raise PMError(rc, _lib.pm_last_error(None).decode())


def host_fft_order(n):
    """Frequency index held at each memory position after the own FFT's forward stages along an n-point axis (pure host)."""
    out = (C.c_int32 * int(n))()
    rc = _lib.pm_host_fft_order(int(n), out)
    if rc != PM_OK:
        raise PMError(rc, "pm_host_fft_order")
    return list(out)


def workspace_bytes(mesh, lattice, omega_m, a, deconvolve=0, flags=0):
    p, keep = make_params(mesh, lattice, omega_m, a, deconvolve, flags)
    n = C.c_size_t(0)
    rc = _lib.pm_workspace_bytes(C.byref(p), C.byref(n))
    if rc != PM_OK:
        raise PMError(rc, _lib.pm_last_error(None).decode())
    return n.value


def _ptr(t, name="tensor", dtype=torch.float32):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA torch tensor")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name} must be contiguous {dtype}")
    return t.data_ptr()


def _hptr(t, name="tensor"):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
        raise TypeError(f"{name} must be a contiguous float32 CPU torch tensor")
    return t.data_ptr()


class PM:
    """One libpm context.  Method names follow include/pm.h without the pm_ prefix."""

    def __init__(self, mesh, lattice, omega_m, a, deconvolve=0, device="cuda:0", stream=None, flags=0):
        if not torch.cuda.is_available():
            raise RuntimeError("libpm needs a CUDA device; there is no CPU fallback")
        self.mesh = tuple(int(v) for v in mesh)
        self.lattice = tuple(int(v) for v in lattice)
        self.np = self.lattice[0] * self.lattice[1] * self.lattice[2]
        self.ng = self.mesh[0] * self.mesh[1] * self.mesh[2]
        self.n_steps = len(a) - 1
        self.device = torch.device(device)
        self._params, self._keep = make_params(mesh, lattice, omega_m, a, deconvolve, flags)
        n = C.c_size_t(0)
        self._h = _vp(None)
        self._check(_lib.pm_workspace_bytes(C.byref(self._params), C.byref(n)), None)
        self.workspace_nbytes = n.value
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(n.value, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            rc = _lib.pm_init(C.byref(self._h), C.byref(self._params), self.workspace.data_ptr(), n.value,
                              self.stream.cuda_stream)
        self._check(rc, None)

    def _check(self, rc, h):
        if rc != PM_OK:
            raise PMError(rc, _lib.pm_last_error(h).decode())

    def _call(self, fn, *args):
        rc = fn(self._h, *args)
        if rc != PM_OK:
            raise PMError(rc, _lib.pm_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            _lib.pm_destroy(self._h)
            self._h = _vp(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _new(self, *shape):
        return torch.empty(*shape, dtype=torch.float32, device=self.device)

    # ---- host scalars ----
    def step_factors(self, i):
        out = (_dbl * 3)()
        self._call(_lib.pm_step_factors, int(i), out)
        return list(out)

    # ---- particle <-> mesh ----
    def scatter(self, x, val=None):
        C_ = 1 if val is None else (1 if val.dim() == 1 else val.shape[1])
        mesh = self._new(C_, *self.mesh)
        self._call(_lib.pm_scatter, x.shape[0], _ptr(x, "x"), _ptr(val, "val"), C_, mesh.data_ptr())
        return mesh[0] if val is None else mesh

    def gather(self, x, mesh):
        C_ = 1 if mesh.dim() == 3 else mesh.shape[0]
        out = self._new(x.shape[0], C_)
        self._call(_lib.pm_gather, x.shape[0], _ptr(x, "x"), _ptr(mesh, "mesh"), C_, out.data_ptr())
        return out

    def gather_grad(self, x, mesh, cot=None):
        C_ = 1 if mesh.dim() == 3 else mesh.shape[0]
        out = self._new(x.shape[0], 3)
        self._call(_lib.pm_gather_grad, x.shape[0], _ptr(x, "x"), _ptr(mesh, "mesh"), C_, _ptr(cot, "cot"),
                   out.data_ptr())
        return out

    def force(self, x):
        out = self._new(x.shape[0], 3)
        self._call(_lib.pm_force, x.shape[0], _ptr(x, "x"), out.data_ptr())
        return out

    def force_vjp(self, x, pi):
        acc = self._new(x.shape[0], 3)
        alpha = self._new(x.shape[0], 3)
        self._call(_lib.pm_force_vjp, x.shape[0], _ptr(x, "x"), _ptr(pi, "pi"), acc.data_ptr(), alpha.data_ptr())
        return acc, alpha

    def run_fwd_adj_obs(self, s0, p0, obs_steps, obs_weights, targets, want_dJ_dOm=False):
        """forward + adjoint run with the mesh objective on several snapshots (eq. 49's O operator) and, optionally,
        the loop part of dJ/dOmega_m (eq. 51).  targets: [n_obs, Nx, Ny, Nz] device tensor."""
        k = len(obs_steps)
        steps = (C.c_int32 * k)(*[int(v) for v in obs_steps])
        w = (_dbl * k)(*[float(v) for v in obs_weights])
        out = {n: self._new(self.np, 3) for n in ("s_n", "p_n", "xi0", "pi0", "dJ_ds0")}
        J, Jk, dth = _dbl(0.0), (_dbl * k)(), _dbl(0.0)
        self._check(_lib.pm_run_fwd_adj_obs(self._h, _ptr(s0, "s0"), _ptr(p0, "p0"), k, steps, w, _ptr(targets, "targets"),
                                            out["s_n"].data_ptr(), out["p_n"].data_ptr(), C.byref(J), Jk,
                                            out["xi0"].data_ptr(), out["pi0"].data_ptr(), out["dJ_ds0"].data_ptr(),
                                            C.byref(dth) if want_dJ_dOm else None), "pm_run_fwd_adj_obs")
        out.update(J=J.value, J_obs=list(Jk), dJ_dOm=dth.value if want_dJ_dOm else None)
        return out

    # ---- optimisation of the initial conditions (Fig. 4) ----
    def adam_step(self, w, g, m, v, t, lr=0.1, beta1=0.9, beta2=0.999, eps=1e-8):
        self._check(_lib.pm_adam_step(self._h, w.numel(), _ptr(w, "w"), _ptr(g, "g"), _ptr(m, "m"), _ptr(v, "v"), int(t),
                                      float(lr), float(beta1), float(beta2), float(eps)), "pm_adam_step")

    def optimize_ic(self, omega, target, amp, n_iter, lr=0.1, order=2, ns=-1.5, rc=2.0):
        """n_iter Adam iterations on the white noise omega (updated in place); returns the J history"""
        nb = _lib.pm_optimize_ic_scratch_bytes(self._h)
        scratch = torch.empty(nb, dtype=torch.uint8, device=self.device)
        hist = (_dbl * max(int(n_iter), 1))()
        self._check(_lib.pm_optimize_ic(self._h, _ptr(omega, "omega"), _ptr(target, "target"), float(amp), float(ns), float(rc),
                                        int(order), int(n_iter), float(lr), scratch.data_ptr(), nb, hist), "pm_optimize_ic")
        return list(hist)[: int(n_iter)]

    # ---- initial conditions (eq. 2-6) and dJ/d(omega) (eq. 51) ----
    def ic_fwd(self, omega, amp, order=2, ns=-1.5, rc=2.0):
        """white noise omega[Lx, Ly, Lz] -> (s0, p0) [N_p, 3] at the ctx's first scale factor"""
        s0, p0 = self._new(self.np, 3), self._new(self.np, 3)
        self._check(_lib.pm_ic_fwd(self._h, _ptr(omega, "omega"), float(amp), float(ns), float(rc), int(order),
                                   s0.data_ptr(), p0.data_ptr()), "pm_ic_fwd")
        return s0, p0

    def ic_vjp(self, omega, amp, xi0, pi0, order=2, ns=-1.5, rc=2.0):
        """dJ/d omega [Lx, Ly, Lz] from the adjoint run's (xi0, pi0)"""
        out = torch.empty(self.lattice, dtype=torch.float32, device=self.device)
        self._check(_lib.pm_ic_vjp(self._h, _ptr(omega, "omega"), float(amp), float(ns), float(rc), int(order),
                                   _ptr(xi0, "xi0"), _ptr(pi0, "pi0"), out.data_ptr()), "pm_ic_vjp")
        return out

    # ---- integrator ----
    def set_state(self, s, p):
        self._call(_lib.pm_set_state, _ptr(s, "s"), _ptr(p, "p"))

    def get_state(self, want_acc=False):
        s, p = self._new(self.np, 3), self._new(self.np, 3)
        acc = self._new(self.np, 3) if want_acc else None
        self._call(_lib.pm_get_state, s.data_ptr(), p.data_ptr(), _ptr(acc))
        return (s, p, acc) if want_acc else (s, p)

    def step_fwd(self, i):
        self._call(_lib.pm_step_fwd, int(i))

    def objective(self, delta_target):
        self._call(_lib.pm_objective, _ptr(delta_target, "delta_target"))

    def get_objective(self):
        J = _dbl(0.0)
        self._call(_lib.pm_get_objective, C.byref(J))
        return J.value

    def set_adjoint(self, xi, pi=None):
        self._call(_lib.pm_set_adjoint, _ptr(xi, "xi"), _ptr(pi, "pi"))

    def step_adj(self, i):
        self._call(_lib.pm_step_adj, int(i))

    def get_adjoint(self):
        xi, pi, g = self._new(self.np, 3), self._new(self.np, 3), self._new(self.np, 3)
        self._call(_lib.pm_get_adjoint, xi.data_ptr(), pi.data_ptr(), g.data_ptr())
        return xi, pi, g

    def run_fwd_adj(self, s0, p0, delta_target, out=None, want=("s_n", "p_n", "xi0", "pi0", "dJ_ds0", "s_rec", "p_rec")):
        """Whole run; returns a dict with J (float) and the requested device tensors."""
        if out is None:
            out = {k: self._new(self.np, 3) for k in want}
        J = _dbl(0.0)
        g = lambda k: _ptr(out.get(k))
        self._call(_lib.pm_run_fwd_adj, _ptr(s0, "s0"), _ptr(p0, "p0"), _ptr(delta_target, "delta_target"),
                   g("s_n"), g("p_n"), C.byref(J), g("xi0"), g("pi0"), g("dJ_ds0"), g("s_rec"), g("p_rec"))
        res = dict(out)
        res["J"] = J.value
        return res

    def run_fwd_adj_host(self, s0, p0, delta_target, out):
        """Host-buffer variant (CPU float32 tensors, ideally pinned); out: dict of CPU tensors to fill."""
        J = _dbl(0.0)
        g = lambda k: _hptr(out.get(k), k)
        self._call(_lib.pm_run_fwd_adj_host, _hptr(s0, "s0"), _hptr(p0, "p0"), _hptr(delta_target, "delta_target"),
                   g("s_n"), g("p_n"), C.byref(J), g("xi0"), g("pi0"), g("dJ_ds0"), g("s_rec"), g("p_rec"))
        return J.value

    # ---- instrumentation ----
    def timing_enable(self, on=True):
        self._call(_lib.pm_timing_enable, 1 if on else 0)

    def timing_reset(self):
        self._call(_lib.pm_timing_reset)

    def timing_read(self):
        n = PM_TIMING_MAX_CLASSES
        names = (C.c_char_p * n)()
        ms = (_dbl * n)()
        cnt = (_i64 * n)()
        by = (_dbl * n)()
        k = _lib.pm_timing_read(self._h, n, names, ms, cnt, by)
        if k < 0:
            raise PMError(k, _lib.pm_last_error(self._h).decode())
        return {names[i].decode(): dict(ms=ms[i], launches=cnt[i], algo_bytes=by[i]) for i in range(k)}

    def launch_count(self):
        a, b = _i64(0), _i64(0)
        self._call(_lib.pm_launch_count, C.byref(a), C.byref(b))
        return a.value, b.value
