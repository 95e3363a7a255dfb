"""Pins for O3 (Darcy residual, Eq. 1): manufactured solutions fed as jets directly."""
import numpy as np

from oracle import pigan_oracle as orc


def _grid():
    rng = np.random.default_rng(5)
    xy = rng.uniform(-1, 1, size=(13, 2)); f = rng.normal(size=13)
    return xy[:, 0][None, :], xy[:, 1][None, :], f


def test_k_equal_one_u_paraboloid_gives_4_minus_f():
    # Y = 0, u = x^2 + y^2  =>  div(grad u) = 4, r = 4 - f exactly (BASELINE check 3)
    x, y, f = _grid()
    Yj = np.zeros((3, 1, 13)); Uj = np.stack([x * x + y * y, 2 * x, 2 * y, 2 + 0 * x, 2 + 0 * x])
    r, msq = orc.darcy_residual_ref(Yj, Uj, f)
    assert np.array_equal(r, 4.0 - f[None, :]) and np.isclose(msq, np.mean((4 - f) ** 2), rtol=1e-15)


def test_loglinear_k_u_paraboloid():
    # Y = a x + b y, u = x^2 + y^2  =>  r = exp(ax+by) (2 a x + 2 b y + 4) - f
    x, y, f = _grid(); a, b = 0.7, -0.4
    Yj = np.stack([a * x + b * y, a + 0 * x, b + 0 * x]); Uj = np.stack([x * x + y * y, 2 * x, 2 * y, 2 + 0 * x, 2 + 0 * x])
    r, _ = orc.darcy_residual_ref(Yj, Uj, f)
    assert np.allclose(r, np.exp(a * x + b * y) * (2 * a * x + 2 * b * y + 4) - f[None, :], rtol=1e-14)


def test_k_one_plus_x_u_x_squared_is_divergence_form():
    # k = 1 + x (Y = log(1+x)), u = x^2:  d/dx((1+x) 2x) = 2 + 4x -- distinguishes div(k grad u) from k lap u
    rng = np.random.default_rng(6); x = rng.uniform(0, 1, size=(1, 9)); f = np.zeros(9)
    Yj = np.stack([np.log1p(x), 1 / (1 + x), 0 * x]); Uj = np.stack([x * x, 2 * x, 0 * x, 2 + 0 * x, 0 * x])
    r, _ = orc.darcy_residual_ref(Yj, Uj, f)
    assert np.allclose(r, 2 + 4 * x, rtol=1e-14)


def test_second_derivatives_of_logk_are_ignored():
    # reading G9: log k carries 3 channels; extra planes, if passed, do not enter
    rng = np.random.default_rng(7)
    Yj = rng.normal(size=(5, 2, 6)); Uj = rng.normal(size=(5, 2, 6)); f = rng.normal(size=6)
    assert np.array_equal(orc.darcy_residual_ref(Yj, Uj, f)[0], orc.darcy_residual_ref(Yj[:3], Uj, f)[0])
