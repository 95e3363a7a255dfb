"""Pins for O8 (Adam): closed forms derived by hand from the update rule (reading G3)."""
import numpy as np

from oracle import pigan_oracle as orc

LR, B1, B2, EPS = 1e-2, 0.5, 0.9, 1e-8


def test_first_step_is_sign_like():
    # from m = v = 0: mhat = g, vhat = g^2  =>  dtheta = -lr g / (|g| + eps)
    th = np.array([1.0, -2.0, 0.5, 3.0]); g = np.array([0.3, -4.0, 1e-3, 0.0])
    t1, m1, v1 = orc.adam_update_ref(th, g, np.zeros(4), np.zeros(4), 1, LR, B1, B2, EPS)
    assert np.allclose(t1, th - LR * g / (np.abs(g) + EPS), rtol=1e-15)
    assert np.allclose(m1, (1 - B1) * g) and np.allclose(v1, (1 - B2) * g * g)
    assert t1[3] == th[3]


def test_constant_gradient_walks_linearly():
    # g_t = g for all t: m_t = (1-b1^t) g, v_t = (1-b2^t) g^2, so the bias correction cancels exactly and
    # theta_t = theta_0 - t lr g/(|g| + eps)
    th = np.array([0.7, -0.1]); g = np.array([2.5, -0.04]); m = np.zeros(2); v = np.zeros(2); th0 = th.copy()
    for t in range(1, 8):
        th, m, v = orc.adam_update_ref(th, g, m, v, t, LR, B1, B2, EPS)
        assert np.allclose(th, th0 - t * LR * g / (np.abs(g) + EPS), rtol=1e-13)


def test_sign_flip_second_step():
    # g_1 = g, g_2 = -g: m_2 = -(1-b1)^2 g, mhat_2 = -(1-b1)/(1+b1) g; v_2 = (1-b2^2) g^2, vhat_2 = g^2
    th = np.array([0.0]); g = np.array([3.0])
    t1, m, v = orc.adam_update_ref(th, g, np.zeros(1), np.zeros(1), 1, LR, B1, B2, 0.0)
    t2, m, v = orc.adam_update_ref(t1, -g, m, v, 2, LR, B1, B2, 0.0)
    assert np.isclose(t1[0], -LR) and np.isclose(t2[0] - t1[0], LR * (1 - B1) / (1 + B1), rtol=1e-14)


def test_skip_leaves_state_bit_identical():
    rng = np.random.default_rng(0); th, g, m, v = (rng.normal(size=5) for _ in range(4)); v = v * v
    t2, m2, v2 = orc.adam_update_ref(th, g, m, v, 3, LR, B1, B2, EPS, skip=True)
    assert np.array_equal(t2, th) and np.array_equal(m2, m) and np.array_equal(v2, v)


def test_three_steps_worked_by_hand():
    """tests/golden/adam_three_steps.txt: four elements, three steps, exact fractions derived by hand in the file."""
    import os
    from fractions import Fraction
    rows = []
    with open(os.path.join(os.path.dirname(__file__), "golden", "adam_three_steps.txt")) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                rows.append([float(Fraction(tok)) for tok in line.split()[1:]])
    rows = np.array(rows)
    assert rows.shape == (4, 9)
    th, m, v = rows[:, 0].copy(), np.zeros(4), np.zeros(4)
    for t in range(1, 4):
        th, m, v = orc.adam_update_ref(th, rows[:, t], m, v, t, 1.0, 0.5, 0.5, 1.0)
        assert np.allclose(th, rows[:, 3 + t], rtol=1e-14, atol=0), (t, th, rows[:, 3 + t])
    assert np.allclose(m, rows[:, 7], rtol=1e-14) and np.allclose(v, rows[:, 8], rtol=1e-14)
