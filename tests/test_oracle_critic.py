"""Pins for O5/O6 (critic, gradient penalty, double backward)."""
import numpy as np
import pytest

from oracle import pigan_oracle as orc
from workloads import xavier_params


def test_one_hidden_unit_critic_closed_form_norm():
    # D = v tanh(w.X + c) + c2  =>  grad_X D = v (1 - t^2) w,  ||G|| = |v| (1 - t^2) ||w||
    w = np.array([0.3, -0.8, 0.5, 0.1]); c, v, c2 = 0.2, -1.7, 0.4
    theta = np.concatenate([w, [c], [v], [c2]])
    rng = np.random.default_rng(0)
    real = rng.normal(size=(3, 4)); fake = rng.normal(size=(3, 4)); eps = rng.uniform(size=3); lam = 10.0
    gp, nu, _ = orc.gradient_penalty_ref(theta, 4, 1, 1, real, fake, eps, lam)
    Xh = eps[:, None] * real + (1 - eps[:, None]) * fake
    t = np.tanh(Xh @ w + c)
    expect = abs(v) * (1 - t * t) * np.linalg.norm(w)
    assert np.allclose(nu, expect, rtol=1e-14)
    assert np.isclose(gp, lam * np.mean((expect - 1) ** 2), rtol=1e-14)
    assert np.allclose(orc.disc_forward_ref(theta, 4, 1, 1, Xh), v * t + c2, rtol=1e-15)


def test_eps_endpoints(tiny):
    t = tiny; c = t["cfg"]
    a = orc.gradient_penalty_ref(t["theta_D"], *c.disc_shape, t["real"], t["real"] * 0 + 3.0, np.ones(c.N), 10.0)
    b = orc.gradient_penalty_ref(t["theta_D"], *c.disc_shape, t["real"], t["real"], t["eps"], 10.0)
    assert np.isclose(a[0], b[0], rtol=1e-14) and np.allclose(a[2], b[2], rtol=1e-12, atol=1e-16)   # eps = 1 -> real
    a = orc.gradient_penalty_ref(t["theta_D"], *c.disc_shape, t["real"] * 0 - 2.0, t["real"], np.zeros(c.N), 10.0)
    assert np.isclose(a[0], b[0], rtol=1e-14) and np.allclose(a[2], b[2], rtol=1e-12, atol=1e-16)   # eps = 0 -> fake


def test_critic_gradients_match_finite_differences_of_LD(tiny):
    t = tiny; c = t["cfg"]
    _, _, gD, losses = orc.train_step_grads_ref(c.gen_shape, c.disc_shape, t["theta_Y"], t["theta_u"], t["theta_D"],
                                                t["xy_colloc"], t["f"], t["xy_sensors"], t["z"], t["real"], t["eps"], 10.0, 1.0)
    Ys = orc.gen_jet_forward_ref(t["theta_Y"], *c.gen_shape, t["xy_sensors"], t["z"], 0)[0]
    Us = orc.gen_jet_forward_ref(t["theta_u"], *c.gen_shape, t["xy_sensors"], t["z"], 0)[0]
    fake = np.concatenate([Ys, Us], axis=1)
    LD = lambda th: orc.critic_loss_ref(c.disc_shape, th, t["real"], fake, t["eps"], 10.0)
    assert np.isclose(losses[0], LD(t["theta_D"]), rtol=1e-7)
    fd = np.zeros_like(gD); h = 1e-5
    for i in range(gD.size):
        tp = t["theta_D"].copy(); tp[i] += h; tm = t["theta_D"].copy(); tm[i] -= h
        fd[i] = (LD(tp) - LD(tm)) / (2 * h)
    assert np.abs(gD - fd).max() / np.abs(fd).max() < 2e-5
    assert gD[-1] == 0.0        # invariant: dL_D/dc_out = 1/N sum(1) - 1/N sum(1) = 0 exactly; GP ignores c_out


def test_critic_matches_torch_float64_double_backward():
    # library special case (S8c pins): torch.autograd.grad(create_graph=True) in float64
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(3)
    shape = (6, 3, 5); lam = 10.0; B = 4
    theta = xavier_params(rng, *shape, bias_std=0.2)
    real = rng.normal(size=(B, 6)); fake = rng.normal(size=(B, 6)); eps = rng.uniform(size=B)
    gp, nu, dgp = orc.gradient_penalty_ref(theta, *shape, real, fake, eps, lam)
    lay = [(torch.tensor(W, requires_grad=True), torch.tensor(b, requires_grad=True)) for W, b in orc.unpack_params(theta, *shape)]
    def D(X):
        g = X
        for W, b in lay[:-1]:
            g = torch.tanh(g @ W.T + b)
        return (g @ lay[-1][0].T + lay[-1][1])[:, 0]
    e = torch.tensor(eps)[:, None]
    Xh = (e * torch.tensor(real) + (1 - e) * torch.tensor(fake)).requires_grad_(True)
    gx, = torch.autograd.grad(D(Xh).sum(), Xh, create_graph=True)
    tnu = gx.norm(dim=1); tgp = lam * ((tnu - 1) ** 2).mean()
    tgp.backward()
    ref = np.concatenate([np.concatenate([W.grad.numpy().ravel(), (b.grad.numpy() if b.grad is not None else np.zeros(b.shape)).ravel()]) for W, b in lay])
    assert np.isclose(gp, tgp.item(), rtol=1e-14) and np.allclose(nu, tnu.detach().numpy(), rtol=1e-13)
    assert np.abs(dgp - ref).max() / np.abs(ref).max() < 1e-12


def test_zero_gradient_norm_gives_zero_seed():
    # reading G12: nu = 0 exactly (v_out = 0) -> penalty lam*(0-1)^2 and a zero (not NaN) gradient seed
    rng = np.random.default_rng(4); shape = (4, 2, 3)
    lay = orc.unpack_params(xavier_params(rng, *shape, bias_std=0.1), *shape)
    lay[-1] = (np.zeros_like(lay[-1][0]), lay[-1][1])
    theta = orc.pack_grads(lay)
    gp, nu, d = orc.gradient_penalty_ref(theta, *shape, rng.normal(size=(2, 4)), rng.normal(size=(2, 4)), np.array([0.3, 0.6]), 10.0)
    assert np.all(nu == 0) and gp == 10.0 and np.all(np.isfinite(d))
