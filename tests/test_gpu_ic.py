"""GPU parity of the device initial-condition generator and its VJP (pm_ic_fwd / pm_ic_vjp) against
the oracle's orc_ic / orc_ic_vjp (eq. 2-6, eq. 51), and of the whole chain
white noise -> 2LPT -> forward + adjoint run -> dJ/d(omega), the quantity of the paper's Fig. 3 (L474-480)."""
import numpy as np
import pytest

from paper_2211_09815_b200 import inputs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.sqrt(np.sum((a - b) ** 2) / max(np.sum(b ** 2), 1e-300)))


@pytest.fixture(scope="module")
def pmlib():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    from paper_2211_09815_b200 import binding
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


@pytest.mark.parametrize("mesh,lattice", [((32, 24, 16), (16, 12, 8)), ((18, 14, 10), (9, 7, 5)), ((64, 64, 64), (32, 32, 32))])
@pytest.mark.parametrize("order", [1, 2])
def test_ic_forward_and_vjp_parity(pmlib, orc, mesh, lattice, order):
    rng = np.random.default_rng(31)
    omega = rng.standard_normal(lattice).astype(np.float32)
    omm, a0 = 0.3, 1.0 / 16
    amp1 = 1.0
    s_ref, _ = orc.ic(mesh, lattice, omm, a0, amp1, omega, order=1)
    amp = 0.3 / np.sqrt(np.mean(np.sum(s_ref ** 2, axis=1)))         # rms displacement 0.3 cell, as in the configs
    s_o, p_o = orc.ic(mesh, lattice, omm, a0, amp, omega, order=order)
    pm = pmlib.PM(mesh, lattice, omm, [a0, 1.0])
    s0, p0 = pm.ic_fwd(dev(omega), amp, order=order)
    assert rel_l2(s0.cpu().numpy(), s_o) <= 1e-5
    assert rel_l2(p0.cpu().numpy(), p_o) <= 1e-5
    xi = rng.standard_normal((pm.np, 3)).astype(np.float32)
    pi = (rng.standard_normal((pm.np, 3)) * 30).astype(np.float32)    # p0 is ~1/15 of s0 at a0 = 1/16: comparable weights
    g = pm.ic_vjp(dev(omega), amp, dev(xi), dev(pi), order=order).cpu().numpy().reshape(-1)
    g_o = orc.ic_vjp(mesh, lattice, omm, a0, amp, omega, xi, pi, order=order)
    assert rel_l2(g, g_o) <= 1e-5
    pm.close()


def test_white_noise_to_gradient_chain_config0(pmlib, orc):
    """omega -> 2LPT -> 16 KDK steps -> J -> adjoint -> (xi0, pi0) -> dJ/d omega at configs[0]'s sizes, both sides from the
    same fp32 white noise: the oracle chain is orc.ic -> orc.run_fwd_adj -> orc.ic_vjp in fp64.  The device chain feeds its
    OWN fp32 (s0, p0) to its run; tolerance = north_star's gradient bar."""
    cfg = inputs.config(0)
    mesh, lattice, omm, a = cfg["mesh"], cfg["lattice"], cfg["omega_m"], cfg["a"]
    rng = np.random.default_rng(1)
    omega = rng.standard_normal(lattice).astype(np.float32)
    s_ref, _ = orc.ic(mesh, lattice, omm, a[0], 1.0, omega, order=1)
    amp = 0.3 / np.sqrt(np.mean(np.sum(s_ref ** 2, axis=1)))
    # target: a second noise field through the oracle
    omega_t = np.random.default_rng(2).standard_normal(lattice)
    s_t, p_t = orc.ic(mesh, lattice, omm, a[0], amp, omega_t, order=2)
    s_nt, _, _ = orc.run_fwd(mesh, lattice, omm, a, s_t, p_t)
    nbar = np.prod(lattice) / np.prod(mesh)
    target = (orc.scatter(mesh, orc.positions(mesh, lattice, s_nt)) / nbar - 1.0).astype(np.float32)
    # oracle chain
    s_o, p_o = orc.ic(mesh, lattice, omm, a[0], amp, omega, order=2)
    ref = orc.run_fwd_adj(mesh, lattice, omm, a, s_o, p_o, target)
    g_o = orc.ic_vjp(mesh, lattice, omm, a[0], amp, omega, ref["xi0"], ref["pi0"], order=2)
    # device chain
    pm = pmlib.PM(mesh, lattice, omm, a)
    om_d = dev(omega)
    s0, p0 = pm.ic_fwd(om_d, amp, order=2)
    out = pm.run_fwd_adj(s0, p0, dev(target))
    g = pm.ic_vjp(om_d, amp, out["xi0"], out["pi0"], order=2).cpu().numpy().reshape(-1)
    assert abs(out["J"] - ref["J"]) <= 1e-4 * abs(ref["J"])
    s_n = out["s_n"].cpu().numpy().astype(np.float64)
    assert np.sqrt(np.mean(np.sum((s_n - ref["s_n"]) ** 2, axis=1))) <= 1e-4
    assert rel_l2(g, g_o) <= 1e-3
    pm.close()
