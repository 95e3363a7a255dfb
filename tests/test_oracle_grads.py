"""Pins for O3/O4/O7 (generator gradients) and the step-level invariants."""
import numpy as np

from oracle import pigan_oracle as orc


def _step(t, **kw):
    c = t["cfg"]
    args = dict(theta_Y=t["theta_Y"], theta_u=t["theta_u"], theta_D=t["theta_D"], xy_colloc=t["xy_colloc"], f=t["f"],
                xy_sensors=t["xy_sensors"], z=t["z"], real_snap=t["real"], eps=t["eps"])
    args.update(kw)
    return orc.train_step_grads_ref(c.gen_shape, c.disc_shape, **args)


def _fd(fun, theta, h=1e-6):
    g = np.zeros_like(theta)
    for i in range(theta.size):
        tp = theta.copy(); tp[i] += h; tm = theta.copy(); tm[i] -= h
        g[i] = (fun(tp) - fun(tm)) / (2 * h)
    return g


def test_generator_gradients_match_finite_differences_of_LG(tiny):
    t = tiny; c = t["cfg"]
    gY, gu, _, losses = _step(t, pde_weight=0.7)
    LG = lambda thY, thu: orc.generator_loss_ref(c.gen_shape, c.disc_shape, thY, thu, t["theta_D"], t["xy_colloc"],
                                                 t["f"], t["xy_sensors"], t["z"], pde_weight=0.7)
    assert np.isclose(losses[4], LG(t["theta_Y"], t["theta_u"]), rtol=1e-13)
    fdY = _fd(lambda th: LG(th, t["theta_u"]), t["theta_Y"])
    fdu = _fd(lambda th: LG(t["theta_Y"], th), t["theta_u"])
    assert np.abs(gY - fdY).max() / np.abs(fdY).max() < 1e-6
    assert np.abs(gu - fdu).max() / np.abs(fdu).max() < 1e-6
    # every parameter group really receives gradient (a dropped term would show as zeros)
    for g in (gY, gu):
        for gW, gb in orc.unpack_params(g, *c.gen_shape):
            assert np.abs(gW).max() > 1e-6 and np.abs(gb).max() > 1e-6


def test_losses_vector_is_consistent(tiny):
    t = tiny; c = t["cfg"]
    _, _, _, L = _step(t, gp_lambda=10.0, pde_weight=1.3)
    assert np.isclose(L[0], L[1] - L[2] + L[3], rtol=1e-14)
    assert np.isclose(L[4], -L[1] + 1.3 * L[5], rtol=1e-14)
    Yc = orc.gen_jet_forward_ref(t["theta_Y"], *c.gen_shape, t["xy_colloc"], t["z"], 1)
    Uc = orc.gen_jet_forward_ref(t["theta_u"], *c.gen_shape, t["xy_colloc"], t["z"], 2)
    assert np.isclose(L[5], orc.darcy_residual_ref(Yc, Uc, t["f"])[1], rtol=1e-13)
    assert np.isclose(L[2], orc.disc_forward_ref(t["theta_D"], *c.disc_shape, t["real"]).mean(), rtol=1e-14)


def test_generator_gradient_is_linear_in_pde_weight(tiny):
    g0 = _step(tiny, pde_weight=0.0); g1 = _step(tiny, pde_weight=1.0); g2 = _step(tiny, pde_weight=2.0)
    for k in (0, 1):
        assert np.allclose(g2[k] - g1[k], g1[k] - g0[k], rtol=1e-10, atol=1e-14)
    assert np.allclose(g0[2], g2[2], atol=0)                      # theta_D gradient does not see w_pde


def test_sample_additivity(tiny):
    # both losses are means over samples: the gradient of the batch is the mean of the per-sample gradients
    t = tiny
    full = _step(t)
    parts = [_step(t, z=t["z"][n:n + 1], real_snap=t["real"][n:n + 1], eps=t["eps"][n:n + 1]) for n in range(2)]
    for k in range(3):
        assert np.allclose(full[k], 0.5 * (parts[0][k] + parts[1][k]), rtol=1e-11, atol=1e-15)
    assert np.allclose(full[3], 0.5 * (parts[0][3] + parts[1][3]), rtol=1e-12)


def test_sensor_rows_only_feed_the_value_channel(tiny):
    # with w_pde = 0 the generator gradient comes only through D(X_fake): FD of -mean D(fake) pins O7
    t = tiny; c = t["cfg"]
    gY, gu, _, _ = _step(t, pde_weight=0.0)
    def negD(thY):
        Ys = orc.gen_jet_forward_ref(thY, *c.gen_shape, t["xy_sensors"], t["z"], 0)[0]
        Us = orc.gen_jet_forward_ref(t["theta_u"], *c.gen_shape, t["xy_sensors"], t["z"], 0)[0]
        return -orc.disc_forward_ref(t["theta_D"], *c.disc_shape, np.concatenate([Ys, Us], 1)).mean()
    fd = _fd(negD, t["theta_Y"])
    assert np.abs(gY - fd).max() / np.abs(fd).max() < 1e-6
