"""Pins of the optimiser oracle (oracle/optim.py) against what the published update rules fix in closed form."""
import numpy as np
import pytest

from oracle import optim


def _g(seed=0, shape=(5, 7)):
    return np.random.default_rng(seed).standard_normal(shape) * 3.0


def test_adam_first_step_is_lr_times_sign():
    """t = 1: m^ = g, v^ = g^2, so the step is lr * g / (|g| + eps): the textbook scale-invariance of Adam."""
    g = _g()                                         # gradient of the LOSS; the oracle takes grad log p = -g
    z = np.zeros_like(g)
    z1, m1, v1 = optim.update(optim.ADAM, z, -g, np.zeros(5), z, z, 1, 1e-3, 0.9, 0.999, 1e-8)
    assert np.allclose(z1, -1e-3 * g / (np.abs(g) + 1e-8), rtol=1e-13)
    assert np.allclose(m1, 0.1 * g) and np.allclose(v1, 0.001 * g * g)


def test_adam_constant_gradient_keeps_unit_steps():
    """A constant gradient: m^ = g and v^ = g^2 at every t, so every step is lr * sign(g) and z(t) = -t lr sign(g)."""
    g = _g(1)
    z = np.zeros_like(g); m = np.zeros_like(g); v = np.zeros_like(g)
    for t in range(1, 40):
        z, m, v = optim.update(optim.ADAM, z, -g, np.zeros(5), m, v, t, 1e-2, 0.9, 0.999, 0.0)
    assert np.allclose(z, -39 * 1e-2 * np.sign(g), rtol=1e-12)


def test_adabelief_first_step_closed_form():
    """t = 1 with eps = eps_root = 0: m = (1-b1) g, s = (1-b2) b1^2 g^2, so the step is lr * sign(g) / b1."""
    g = _g(2); z = np.zeros_like(g)
    z1, m1, s1 = optim.update(optim.ADABELIEF, z, -g, np.zeros(5), z, z, 1, 1e-4, 0.95, 0.99, 0.0, 0.0)
    assert np.allclose(z1, -1e-4 * np.sign(g) / 0.95, rtol=1e-12)
    assert np.allclose(s1, 0.01 * (0.95 * g) ** 2, rtol=1e-13)


def test_adabelief_belief_term_vanishes_for_constant_gradient():
    """Constant gradient: g - m -> 0 geometrically, so s decays like b2^t and the steps GROW (large belief)."""
    g = np.full((1, 1), 2.0); z = np.zeros((1, 1)); m = z.copy(); s = z.copy()
    steps = []
    for t in range(1, 200):
        z0 = z.copy()
        z, m, s = optim.update(optim.ADABELIEF, z, -g, np.zeros(1), m, s, t, 1e-4, 0.95, 0.99, 1e-16, 1e-16)
        steps.append(float((z0 - z)[0, 0]))
    assert abs(g - m).max() < 2.0 * 0.95 ** 199 * 1.0001
    assert steps[-1] > steps[0] > 0


@pytest.mark.parametrize("kind", [optim.ADAM, optim.ADABELIEF])
def test_descends_a_quadratic_bowl(kind):
    """loss = 1/2 sum a_i z_i^2 (log p = -loss): both rules bring every coordinate close to the minimum."""
    a = np.array([[0.5, 2.0, 10.0]])
    z = np.array([[1.0, -2.0, 0.5]]); m = np.zeros_like(z); v = np.zeros_like(z)
    for t in range(1, 3001):
        z, m, v = optim.update(kind, z, -(a * z), np.zeros(1), m, v, t, 5e-3, 0.9, 0.999, 1e-8, 1e-16)
    assert np.all(np.abs(z) < 2e-2)


def test_non_finite_rows_are_left_unchanged():
    g = _g(3); z = _g(4); m = _g(5) * 0.1; v = np.abs(_g(6))
    logp = np.array([0.0, -np.inf, 0.0, np.nan, 0.0])
    g2 = g.copy(); g2[2, 3] = np.nan
    z1, m1, v1 = optim.update(optim.ADAM, z, g2, logp, m, v, 3, 1e-3, 0.9, 0.999, 1e-8)
    for r in (1, 2, 3):
        assert np.array_equal(z1[r], z[r]) and np.array_equal(m1[r], m[r]) and np.array_equal(v1[r], v[r])
    for r in (0, 4):
        assert not np.array_equal(z1[r], z[r])
    assert np.all(np.isfinite(z1))
