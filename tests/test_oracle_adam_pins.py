"""Pins of the oracle's Adam step (oracle/pm_oracle.py adam_step; the optimiser of PAPER.md Fig. 4).

  A1  first step: m_hat = g, v_hat = g^2, so every component moves by lr * g / (|g| + eps) = lr * sign(g) up to eps
  A2  constant gradient g: the bias corrections make every step equal to the first one
  A3  on f(w) = 1/2 w^2 from w = 1 with lr = 0.1 the iterate crosses zero and settles (|w| < 0.05 after 200 steps)
"""
import numpy as np


def test_A1_first_step_is_sign_descent(orc):
    g = np.array([3.0, -0.02, 1e-3, -7.0])
    w, m, v = orc.adam_step(np.zeros(4), g, np.zeros(4), np.zeros(4), 1, lr=0.1)
    np.testing.assert_allclose(w, -0.1 * np.sign(g), rtol=2e-5)
    np.testing.assert_allclose(m, 0.1 * g)
    np.testing.assert_allclose(v, 0.001 * g * g)


def test_A2_constant_gradient_gives_constant_steps(orc):
    g = np.array([0.5, -2.0])
    w, m, v = np.zeros(2), np.zeros(2), np.zeros(2)
    prev = w.copy()
    for t in range(1, 8):
        w, m, v = orc.adam_step(w, g, m, v, t, lr=0.05)
        np.testing.assert_allclose(w - prev, -0.05 * np.sign(g), rtol=1e-6)
        prev = w.copy()


def test_A3_quadratic_bowl(orc):
    w, m, v = np.array([1.0]), np.zeros(1), np.zeros(1)
    seen_negative = False
    for t in range(1, 201):
        w, m, v = orc.adam_step(w, w.copy(), m, v, t, lr=0.1)
        seen_negative |= bool(w[0] < 0)
    assert seen_negative and abs(w[0]) < 0.05
