"""GPU parity of the run with observations between the steps (eq. 49's O operator, L393) and of the loop part of
dJ/dOmega_m (eq. 51 first line, L406) against the oracle's orc_run_fwd_adj_obs."""
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


def _inputs(orc, mesh, lattice, omm, a, n_obs):
    s0 = inputs.zeldovich_displacement(lattice, mesh, seed=1, rms=0.3)
    p0 = (s0.astype(np.float64) * orc.p_over_s(omm, a[0])).astype(np.float32)
    targets = np.stack([inputs.lognormal_target(mesh, seed=2 + k, sigma=0.5) for k in range(n_obs)])
    return s0, p0, targets


@pytest.mark.parametrize("mesh,lattice,omm", [((32, 32, 32), (16, 16, 16), 0.3), ((24, 20, 36), (12, 10, 18), 1.0)])
def test_observations_and_omega_m_gradient_parity(pmlib, orc, mesh, lattice, omm):
    a = inputs.a_schedule(1.0 / 8, 6)
    steps, w = [2, 6, 4], [0.5, 1.0, 2.0]
    s0, p0, targets = _inputs(orc, mesh, lattice, omm, a, len(steps))
    ref = orc.run_fwd_adj_obs(mesh, lattice, omm, a, s0, p0, steps, w, targets)
    pm = pmlib.PM(mesh, lattice, omm, a)
    for want in (False, True):          # chained adjoint steps between observations / unchained with the reductions
        out = pm.run_fwd_adj_obs(dev(s0), dev(p0), steps, w, dev(targets), want_dJ_dOm=want)
        assert abs(out["J"] - ref["J"]) <= 1e-4 * abs(ref["J"])
        np.testing.assert_allclose(out["J_obs"], ref["J_obs"], rtol=1e-4)
        s_n = out["s_n"].cpu().numpy().astype(np.float64)
        assert np.sqrt(np.mean(np.sum((s_n - ref["s_n"]) ** 2, axis=1))) <= 1e-4
        assert rel_l2(out["xi0"].cpu().numpy(), ref["xi0"]) <= 1e-3
        assert rel_l2(out["pi0"].cpu().numpy(), ref["pi0"]) <= 1e-3
        if want:
            assert abs(out["dJ_dOm"] - ref["dJ_dOm"]) <= 1e-3 * abs(ref["dJ_dOm"])
    pm.close()


def test_single_final_observation_equals_the_plain_run(pmlib, orc):
    cfg = inputs.config(0)
    mesh, lattice, omm, a = cfg["mesh"], cfg["lattice"], cfg["omega_m"], cfg["a"]
    s0, p0, targets = _inputs(orc, mesh, lattice, omm, a, 1)
    pm = pmlib.PM(mesh, lattice, omm, a)
    plain = pm.run_fwd_adj(dev(s0), dev(p0), dev(targets[0]))
    obs = pm.run_fwd_adj_obs(dev(s0), dev(p0), [len(a) - 1], [1.0], dev(targets))
    assert obs["J"] == plain["J"]
    for k in ("s_n", "p_n", "xi0", "pi0", "dJ_ds0"):
        assert torch.equal(obs[k], plain[k]), k
    pm.close()


def test_observation_of_the_initial_snapshot(pmlib, orc):
    """an observation at t_0 is added after the last adjoint step (O_0): xi_0 then contains dJ_0/dx_0 directly"""
    mesh, lattice, omm = (32, 32, 32), (16, 16, 16), 0.3
    a = inputs.a_schedule(1.0 / 8, 4)
    steps, w = [0, 4], [1.5, 1.0]
    s0, p0, targets = _inputs(orc, mesh, lattice, omm, a, 2)
    ref = orc.run_fwd_adj_obs(mesh, lattice, omm, a, s0, p0, steps, w, targets)
    pm = pmlib.PM(mesh, lattice, omm, a)
    out = pm.run_fwd_adj_obs(dev(s0), dev(p0), steps, w, dev(targets), want_dJ_dOm=True)
    np.testing.assert_allclose(out["J_obs"], ref["J_obs"], rtol=1e-4)
    assert rel_l2(out["xi0"].cpu().numpy(), ref["xi0"]) <= 1e-3
    assert rel_l2(out["pi0"].cpu().numpy(), ref["pi0"]) <= 1e-3
    assert abs(out["dJ_dOm"] - ref["dJ_dOm"]) <= 1e-3 * abs(ref["dJ_dOm"])
    pm.close()
