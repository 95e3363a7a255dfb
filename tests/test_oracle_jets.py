"""Pins for O1/O2 (generator MLP and its second-order jet) -- SURVEY.md section 8(c) 'what pins the oracle'."""
import numpy as np
import pytest

from oracle import pigan_oracle as orc
from workloads import xavier_params


def _net(seed=0, m=3, L=3, H=9, bias_std=0.3):
    rng = np.random.default_rng(seed)
    shape = (2 + m, L, H)
    return shape, xavier_params(rng, *shape, bias_std=bias_std), rng


def test_param_count_matches_survey_table():
    # SURVEY.md section 8 table 'params per generator net' / 'params discriminator'
    assert orc.param_count(2 + 4, 3, 32) == 2369
    assert orc.param_count(2 + 30, 4, 128) == 53889
    assert orc.param_count(2 + 60, 4, 256) == 213761
    assert orc.param_count(2 + 1000, 6, 512) == 1827329
    assert orc.param_count(2 + 4000, 6, 1024) == 9348097
    assert orc.param_count(20, 3, 32) == 2817
    assert orc.param_count(10000, 6, 1024) == 15490049


def test_jets_match_central_differences_of_value_channel():
    shape, theta, rng = _net()
    xy = rng.uniform(0.1, 0.9, size=(11, 2)); z = rng.normal(size=(3, 3))
    out = orc.gen_jet_forward_ref(theta, *shape, xy, z, 2)
    val = lambda p: orc.gen_jet_forward_ref(theta, *shape, p, z, 0)[0]
    h = 1e-4
    ex, ey = np.array([h, 0.0]), np.array([0.0, h])
    assert np.allclose(out[0], val(xy), rtol=0, atol=1e-14)
    assert np.allclose(out[1], (val(xy + ex) - val(xy - ex)) / (2 * h), rtol=0, atol=1e-8)
    assert np.allclose(out[2], (val(xy + ey) - val(xy - ey)) / (2 * h), rtol=0, atol=1e-8)
    assert np.allclose(out[3], (val(xy + ex) - 2 * val(xy) + val(xy - ex)) / h ** 2, rtol=0, atol=2e-6)
    assert np.allclose(out[4], (val(xy + ey) - 2 * val(xy) + val(xy - ey)) / h ** 2, rtol=0, atol=2e-6)
    # the derivative channels are not trivially zero
    assert min(np.abs(out[c]).max() for c in range(1, 5)) > 1e-3


def test_jet_orders_are_prefixes():
    shape, theta, rng = _net(1)
    xy = rng.uniform(size=(5, 2)); z = rng.normal(size=(2, 3))
    o2 = orc.gen_jet_forward_ref(theta, *shape, xy, z, 2)
    o1 = orc.gen_jet_forward_ref(theta, *shape, xy, z, 1)
    o0 = orc.gen_jet_forward_ref(theta, *shape, xy, z, 0)
    assert o2.shape == (5, 2, 5) and o1.shape == (3, 2, 5) and o0.shape == (1, 2, 5)
    assert np.array_equal(o2[:3], o1) and np.array_equal(o1[:1], o0)


def test_one_hidden_unit_closed_form():
    # G = w2 tanh(wx x + wy y + wz.z + b) + b2  =>  G_x = w2 wx (1-t^2), G_xx = -2 w2 wx^2 t (1-t^2)  (BASELINE check 2)
    wx, wy, wz, b, w2, b2 = 0.7, -1.3, np.array([0.4, -0.2]), 0.15, 1.9, -0.6
    theta = np.concatenate([[wx, wy], wz, [b], [w2], [b2]])
    xy = np.array([[0.2, 0.9], [0.5, 0.5], [-0.3, 0.1]]); z = np.array([[1.0, 2.0], [-0.5, 0.3]])
    out = orc.gen_jet_forward_ref(theta, 4, 1, 1, xy, z, 2)
    for n in range(2):
        t = np.tanh(wx * xy[:, 0] + wy * xy[:, 1] + wz @ z[n] + b); s = 1 - t * t
        assert np.allclose(out[0, n], w2 * t + b2, atol=1e-15)
        assert np.allclose(out[1, n], w2 * wx * s, atol=1e-15)
        assert np.allclose(out[2, n], w2 * wy * s, atol=1e-15)
        assert np.allclose(out[3, n], -2 * w2 * wx ** 2 * t * s, atol=1e-15)
        assert np.allclose(out[4, n], -2 * w2 * wy ** 2 * t * s, atol=1e-15)


def test_no_spatial_weights_means_zero_derivatives():
    shape, theta, rng = _net(2)
    lay = orc.unpack_params(theta.copy(), *shape)
    lay[0][0][:, 0:2] = 0.0
    theta0 = orc.pack_grads(lay)
    xy = rng.uniform(size=(6, 2)); z = rng.normal(size=(2, 3))
    out = orc.gen_jet_forward_ref(theta0, *shape, xy, z, 2)
    assert np.all(out[1:] == 0.0)
    assert np.ptp(out[0], axis=1).max() < 1e-14  # value does not depend on the point either (BLAS rounding only)
    f = rng.normal(size=6)
    r, msq = orc.darcy_residual_ref(out[:3], out, f)
    assert np.allclose(r, -f[None, :], atol=0) and np.isclose(msq, np.mean(f * f))


def test_swapping_x_and_y_swaps_channels():
    shape, theta, rng = _net(3)
    lay = orc.unpack_params(theta, *shape)
    W1 = lay[0][0].copy(); W1[:, [0, 1]] = W1[:, [1, 0]]
    theta_sw = orc.pack_grads([(W1, lay[0][1])] + lay[1:])
    xy = rng.uniform(size=(7, 2)); z = rng.normal(size=(2, 3))
    a = orc.gen_jet_forward_ref(theta, *shape, xy, z, 2)
    b = orc.gen_jet_forward_ref(theta_sw, *shape, xy[:, ::-1], z, 2)
    assert np.allclose(a[[0, 1, 2, 3, 4]], b[[0, 2, 1, 4, 3]], atol=1e-14)


def test_jets_match_torch_float64_autograd():
    # library special case: torch.autograd differentiates the plain MLP twice (shares no code with the oracle)
    torch = pytest.importorskip("torch")
    shape, theta, rng = _net(4, m=2, L=2, H=5)
    xy = rng.uniform(size=(4, 2)); z = rng.normal(size=(2, 2))
    out = orc.gen_jet_forward_ref(theta, *shape, xy, z, 2)
    lay = [(torch.tensor(W), torch.tensor(b)) for W, b in orc.unpack_params(theta, *shape)]
    for n in range(2):
        for p in range(4):
            x = torch.tensor(xy[p, 0], requires_grad=True); y = torch.tensor(xy[p, 1], requires_grad=True)
            h = torch.cat([x[None], y[None], torch.tensor(z[n])])
            for W, b in lay[:-1]:
                h = torch.tanh(W @ h + b)
            o = (lay[-1][0] @ h + lay[-1][1])[0]
            gx, gy = torch.autograd.grad(o, (x, y), create_graph=True)
            gxx, = torch.autograd.grad(gx, x, retain_graph=True); gyy, = torch.autograd.grad(gy, y)
            got = out[:, n, p]
            assert np.allclose(got, [o.item(), gx.item(), gy.item(), gxx.item(), gyy.item()], rtol=1e-12, atol=1e-13)
