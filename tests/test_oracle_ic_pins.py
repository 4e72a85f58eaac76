"""Pins of the oracle's initial-condition generator and its VJP (oracle/pm_oracle.c section 7).

PAPER.md eq. 2-6 (L57-89): s = D1 s1 + D2 s2, p = a^2 H (D1' s1 + D2' s2), s_m = -grad phi_m,
lap phi_1 = delta_1, lap phi_2 = sum_{a<b} (phi_1,aa phi_1,bb - phi_1,ab^2), delta_1(k) = sqrt(V P) omega(k);
eq. 51 (L406): dJ/d omega = xi_0 . dx_0/d omega + pi_0 . dp_0/d omega; growth of second order: A1-A8 (L520-555).

  I1  Einstein-de Sitter closed forms D2 = 3/7 a^2, D2' = 6/7 a^2 (A3, L528)
  I2  LambdaCDM: the oracle's G-form ODE (A5) against scipy's integration of the D-form ODE (A1, second line) with the
      initial conditions A3 -- another formulation and another integrator -- and against Bouchet et al.'s fit
  I3  every inverse transform is real to rounding (Hermitian symmetry of all multipliers, Nyquist rule included)
  I4  one plane wave: s1 = -(T/k) sin(kx), no second order (only one non-zero second derivative)
  I5  two crossed waves: closed form of the second-order displacement (sign, 1/k^2 factors, index structure)
  I6  -div s1 = delta_1 for band-limited noise, by the lattice's own spectral derivative written with numpy.fft
  I7  VJP against central differences of Phi(omega) = xi . s0 + pi . p0 on every component (Phi is quadratic in omega,
      so the central difference is exact up to rounding), on a non-cubic lattice with Nyquist planes
  I8  first order is linear: <c, A omega> = <A^T c, omega>
"""
import numpy as np
import pytest

N, L = (16, 12, 8), (8, 6, 4)


def lattice_coords(N, L):
    ax = [np.arange(L[d]) * (N[d] // L[d]) for d in range(3)]
    return np.meshgrid(*ax, indexing="ij")


def test_I1_eds_second_order_growth(orc):
    for a in (0.02, 0.3, 1.0):
        d2 = orc.growth2(1.0, a)
        np.testing.assert_allclose(d2, [3.0 / 7.0 * a * a, 6.0 / 7.0 * a * a], rtol=1e-10)
    f = orc.ic_factors(1.0, 0.25)                     # D1 = a, D1' = a, E = a^-3/2
    np.testing.assert_allclose(f, [0.25, 3 / 7 * 0.0625, 0.25 ** 1.5, 6 / 7 * 0.25 ** 2.5], rtol=1e-10)


def test_I2_lcdm_second_order_growth_by_another_route(orc):
    from scipy.integrate import solve_ivp
    om = 0.3

    def rhs(lna, y):                                   # eq. A1 in D (not G): y = (D1, D1', D2, D2')
        a = np.exp(lna)
        E2 = om / a ** 3 + 1 - om
        oma = om / a ** 3 / E2
        hh = -1.5 * oma
        return [y[1], -(2 + hh) * y[1] + 1.5 * oma * y[0], y[3], -(2 + hh) * y[3] + 1.5 * oma * y[2] + 1.5 * oma * y[0] ** 2]

    ai = 1e-5
    sol = solve_ivp(rhs, [np.log(ai), 0.0], [ai, ai, 3 / 7 * ai ** 2, 6 / 7 * ai ** 2], rtol=1e-11, atol=1e-20,
                    dense_output=True, method="DOP853")
    for a in (1 / 64, 0.25, 1.0):
        y = sol.sol(np.log(a))
        np.testing.assert_allclose(orc.growth2(om, a), [y[2], y[3]], rtol=2e-7)
        d1 = orc.growth(om, a)[0]
        np.testing.assert_allclose(d1, y[0], rtol=2e-7)
        oma = om / a ** 3 / (om / a ** 3 + 1 - om)
        assert abs(y[2] / (3 / 7 * d1 ** 2 * oma ** (-1 / 143)) - 1) < 5e-3      # Bouchet et al. 1995 fit


def test_I3_outputs_are_real(orc):
    rng = np.random.default_rng(3)
    om = rng.standard_normal(L)
    s0, p0, im = orc.ic(N, L, 0.3, 0.1, 0.7, om, order=2, return_imag=True)
    assert im <= 1e-13 * max(np.abs(s0).max() / orc.ic_factors(0.3, 0.1)[0], 1.0)
    assert np.abs(s0).max() > 1e-4


@pytest.mark.parametrize("order", [1, 2])
def test_I4_single_plane_wave(orc, order):
    x, y, z = lattice_coords(N, L)
    k0 = 2 * np.pi * 1 / N[0]
    amp, a0, omm = 0.37, 0.2, 0.3
    omega = np.cos(k0 * x)
    T = amp * np.sqrt(k0 ** -1.5 * np.exp(-(2.0 * k0) ** 2))
    f = orc.ic_factors(omm, a0)
    s0, p0 = orc.ic(N, L, omm, a0, amp, omega, order=order)
    s1x = (-(T / k0) * np.sin(k0 * x)).reshape(-1)
    np.testing.assert_allclose(s0[:, 0], f[0] * s1x, atol=1e-13)
    np.testing.assert_allclose(p0[:, 0], f[2] * s1x, atol=1e-13)
    assert np.abs(s0[:, 1:]).max() < 1e-13 and np.abs(p0[:, 1:]).max() < 1e-13


def test_I5_two_crossed_waves_second_order(orc):
    Nc, Lc = (16, 16, 8), (8, 8, 4)
    x, y, z = lattice_coords(Nc, Lc)
    k0 = 2 * np.pi * 1 / Nc[0]
    A, B, amp, a0, omm = 1.3, -0.6, 0.45, 0.3, 1.0
    omega = A * np.cos(k0 * x) + B * np.cos(k0 * y)
    T = amp * np.sqrt(k0 ** -1.5 * np.exp(-(2.0 * k0) ** 2))
    f = orc.ic_factors(omm, a0)
    s0, p0 = orc.ic(Nc, Lc, omm, a0, amp, omega, order=2)
    s1 = np.stack([-(T * A / k0) * np.sin(k0 * x), -(T * B / k0) * np.sin(k0 * y), 0 * x], axis=-1).reshape(-1, 3)
    c2 = -(T * T * A * B) / (2 * k0)
    s2 = np.stack([c2 * np.sin(k0 * x) * np.cos(k0 * y), c2 * np.cos(k0 * x) * np.sin(k0 * y), 0 * x], axis=-1).reshape(-1, 3)
    np.testing.assert_allclose(s0, f[0] * s1 + f[1] * s2, atol=1e-13)
    np.testing.assert_allclose(p0, f[2] * s1 + f[3] * s2, atol=1e-13)
    assert np.abs(f[1] * s2).max() > 1e-3                      # the second order is really there


def test_I6_divergence_of_first_order_is_minus_delta1(orc):
    rng = np.random.default_rng(8)
    Lc, Nc = (9, 7, 5), (18, 14, 10)                           # odd lattice: no Nyquist planes
    omega = rng.standard_normal(Lc)
    amp, a0 = 0.8, 0.5
    s0, _ = orc.ic(Nc, Lc, 1.0, a0, amp, omega, order=1)
    s1 = (s0 / orc.ic_factors(1.0, a0)[0]).reshape(Lc + (3,))
    k = [2 * np.pi * np.fft.fftfreq(Lc[d], d=1.0 / Lc[d]) / Nc[d] for d in range(3)]
    kx, ky, kz = np.meshgrid(*k, indexing="ij")
    k2 = kx ** 2 + ky ** 2 + kz ** 2
    div = sum(np.fft.ifftn(1j * kk * np.fft.fftn(s1[..., d])) for d, kk in enumerate((kx, ky, kz))).real
    with np.errstate(divide="ignore", invalid="ignore"):
        T = np.where(k2 > 0, amp * np.sqrt(k2 ** -0.75 * np.exp(-4.0 * k2)), 0.0)
    delta1 = np.fft.ifftn(T * np.fft.fftn(omega)).real
    np.testing.assert_allclose(-div, delta1, atol=1e-13)


@pytest.mark.parametrize("order", [1, 2])
def test_I7_vjp_against_central_differences(orc, order):
    rng = np.random.default_rng(12)
    omega = rng.standard_normal(L)
    npart = int(np.prod(L))
    xi, pi = rng.standard_normal((npart, 3)), rng.standard_normal((npart, 3))
    amp, a0, omm = 1.1, 0.15, 0.3

    def phi(w):
        s0, p0 = orc.ic(N, L, omm, a0, amp, w, order=order)
        return float(np.sum(xi * s0) + np.sum(pi * p0))

    g = orc.ic_vjp(N, L, omm, a0, amp, omega, xi, pi, order=order)
    fd = np.zeros(npart)
    eps = 1e-3
    flat = omega.reshape(-1)
    for j in range(npart):
        wp, wm = flat.copy(), flat.copy()
        wp[j] += eps
        wm[j] -= eps
        fd[j] = (phi(wp.reshape(L)) - phi(wm.reshape(L))) / (2 * eps)
    np.testing.assert_allclose(g, fd, rtol=0, atol=1e-9 * np.abs(fd).max())
    if order == 2:      # the second-order part of the gradient is not negligible in this test
        g1 = orc.ic_vjp(N, L, omm, a0, amp, omega, xi, pi, order=1)
        assert np.abs(g - g1).max() > 1e-4 * np.abs(g).max()


def test_I8_first_order_transpose_identity(orc):
    rng = np.random.default_rng(14)
    omega = rng.standard_normal(L)
    npart = int(np.prod(L))
    xi, pi = rng.standard_normal((npart, 3)), rng.standard_normal((npart, 3))
    s0, p0 = orc.ic(N, L, 0.3, 0.2, 0.9, omega, order=1)
    g = orc.ic_vjp(N, L, 0.3, 0.2, 0.9, omega, xi, pi, order=1)
    lhs = np.sum(xi * s0) + np.sum(pi * p0)
    np.testing.assert_allclose(lhs, np.sum(g * omega.reshape(-1)), rtol=1e-12)
