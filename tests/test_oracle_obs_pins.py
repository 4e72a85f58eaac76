"""Pins of the oracle's run with observations between the steps and its Omega_m gradient (oracle/pm_oracle.c section 8).

PAPER.md eq. 49, last lines (L393): O_{i-1} adds dJ/dx_{i-1} to xi_{i-1}; eq. 51 first line (L406): the gradient with
respect to a cosmological parameter accumulated during the reverse pass (here theta = Omega_m, initial conditions fixed).

  O1  a single observation of the final snapshot with weight 1 is the plain run (orc_run_fwd_adj): same J, xi0, pi0
  O2  central differences of J = sum_k w_k J_k in every coordinate of s0 and p0 (two snapshots, unequal weights)
  O3  central difference of J in Omega_m at fixed (s0, p0), EdS-like and LambdaCDM
  O4  J is the weighted sum of the per-snapshot objectives evaluated by an independent forward run
"""
import numpy as np
import pytest

N, L = (8, 8, 8), (4, 4, 4)


def setup(orc, om, seed=5, n=3):
    rng = np.random.default_rng(seed)
    a = np.linspace(0.3, 0.9, n + 1)
    npart = int(np.prod(L))
    while True:
        s0 = 0.3 * rng.standard_normal((npart, 3))
        x = orc.positions(N, L, s0)
        if np.abs(x - np.rint(x)).min() > 1e-3:          # R7: stay away from the CIC kinks
            break
    p0 = orc.p_over_s(om, a[0]) * s0 * (1 + 0.1 * rng.standard_normal((npart, 3)))
    targets = rng.standard_normal((2,) + N) * 0.5
    return a, s0, p0, targets


def test_O1_single_final_observation_is_the_plain_run(orc):
    a, s0, p0, targets = setup(orc, 0.3)
    n = len(a) - 1
    ref = orc.run_fwd_adj(N, L, 0.3, a, s0, p0, targets[0])
    out = orc.run_fwd_adj_obs(N, L, 0.3, a, s0, p0, [n], [1.0], targets[:1])
    assert out["J"] == pytest.approx(ref["J"], rel=1e-14)
    np.testing.assert_allclose(out["xi0"], ref["xi0"], rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(out["pi0"], ref["pi0"], rtol=1e-12, atol=1e-14)


def test_O4_J_is_the_weighted_sum_of_snapshot_objectives(orc):
    a, s0, p0, targets = setup(orc, 0.3)
    out = orc.run_fwd_adj_obs(N, L, 0.3, a, s0, p0, [1, 3], [0.7, 1.3], targets)
    J = 0.0
    for k, (i, w) in enumerate(((1, 0.7), (3, 1.3))):
        s_i, _, Ji = orc.run_fwd(N, L, 0.3, a[: i + 1], s0, p0, targets[k])
        assert out["J_obs"][k] == pytest.approx(Ji, rel=1e-12)
        J += w * Ji
    assert out["J"] == pytest.approx(J, rel=1e-12)


def test_O2_gradient_against_central_differences(orc):
    om = 0.3
    a, s0, p0, targets = setup(orc, om)
    steps, w = [2, 3], [0.7, 1.3]
    out = orc.run_fwd_adj_obs(N, L, om, a, s0, p0, steps, w, targets)

    def J(s, p):
        return orc.run_fwd_adj_obs(N, L, om, a, s, p, steps, w, targets)["J"]

    eps = 1e-6
    rng = np.random.default_rng(9)
    for j, d in zip(rng.integers(0, s0.shape[0], 12), rng.integers(0, 3, 12)):
        sp, sm = s0.copy(), s0.copy()
        sp[j, d] += eps
        sm[j, d] -= eps
        fd = (J(sp, p0) - J(sm, p0)) / (2 * eps)
        assert out["xi0"][j, d] == pytest.approx(fd, rel=2e-6, abs=1e-7 * np.abs(out["xi0"]).max())
        pp, pm_ = p0.copy(), p0.copy()
        pp[j, d] += eps
        pm_[j, d] -= eps
        fd = (J(s0, pp) - J(s0, pm_)) / (2 * eps)
        assert out["pi0"][j, d] == pytest.approx(fd, rel=2e-6, abs=1e-7 * np.abs(out["pi0"]).max())


@pytest.mark.parametrize("om", [0.3, 0.9])
def test_O3_omega_m_gradient_against_central_difference(orc, om):
    a, s0, p0, targets = setup(orc, om, seed=7, n=4)
    steps, w = [2, 4], [1.0, 0.5]
    out = orc.run_fwd_adj_obs(N, L, om, a, s0, p0, steps, w, targets)
    h = 1e-5
    Jp = orc.run_fwd_adj_obs(N, L, om + h, a, s0, p0, steps, w, targets)["J"]
    Jm = orc.run_fwd_adj_obs(N, L, om - h, a, s0, p0, steps, w, targets)["J"]
    fd = (Jp - Jm) / (2 * h)
    assert abs(fd) > 1e-3 * abs(out["J"])                  # the derivative is not accidentally tiny
    assert out["dJ_dOm"] == pytest.approx(fd, rel=2e-6)
