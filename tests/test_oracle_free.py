"""Pins for the NEXT-2 oracle (f at per-realization free sensors fed to the critic; R9)."""
import numpy as np

from oracle import pigan_oracle as orc


def _setup(rng, N=2, Fp=4, S=3, m=2, L=2, H=4, LD=2, HD=5):
    gen_shape, disc_shape = (2 + m, L, H), (2 * S + 3 * Fp, LD, HD)
    thY = rng.normal(0, 0.6, size=orc.param_count(*gen_shape)); thU = rng.normal(0, 0.6, size=orc.param_count(*gen_shape))
    thD = rng.normal(0, 0.4, size=orc.param_count(*disc_shape))
    xy_free = rng.uniform(size=(N, Fp, 2)); xy_s = rng.uniform(size=(S, 2)); z = rng.normal(size=(N, m))
    real = rng.normal(size=(N, 2 * S + 3 * Fp)); eps = rng.uniform(size=N)
    return gen_shape, disc_shape, thY, thU, thD, xy_free, xy_s, z, real, eps


def test_snapshot_layout_and_f_is_eq1_of_the_generator():
    rng = np.random.default_rng(2)
    gen_shape, disc_shape, thY, thU, thD, xy_free, xy_s, z, real, eps = _setup(rng)
    X, _ = orc.free_snapshot_ref(gen_shape, thY, thU, xy_free, xy_s, z)
    S, Fp = 3, 4
    assert X.shape == (2, 2 * S + 3 * Fp)
    assert np.array_equal(X[:, 2 * S + Fp:2 * S + 2 * Fp], xy_free[:, :, 0]) and np.array_equal(X[:, 2 * S + 2 * Fp:], xy_free[:, :, 1])
    # f = div(k grad u) with k = exp(G_Y), by central differences of the VALUE channels only (Eq. 1)
    h = 1e-4
    for n in range(2):
        def ku(dx, dy):
            p = xy_free[n] + np.array([dx, dy])
            return (np.exp(orc.gen_jet_forward_ref(thY, *gen_shape, p, z[n:n + 1], 0)[0, 0]), orc.gen_jet_forward_ref(thU, *gen_shape, p, z[n:n + 1], 0)[0, 0])
        k0, u0 = ku(0, 0)
        div = 0.0
        for ax in ((h, 0), (0, h)):
            kp, up = ku(*ax); km, um = ku(-ax[0], -ax[1])
            div = div + (0.5 * (kp + k0) * (up - u0) - 0.5 * (k0 + km) * (u0 - um)) / h ** 2      # conservative second difference
        assert np.allclose(X[n, 2 * S:2 * S + Fp], div, rtol=0, atol=5e-6 * max(1.0, np.abs(div).max()))


def test_gradients_match_finite_differences():
    rng = np.random.default_rng(4)
    gen_shape, disc_shape, thY, thU, thD, xy_free, xy_s, z, real, eps = _setup(rng)
    for w_pde in (0.0, 0.8):
        gY, gU, gD, losses = orc.train_step_grads_free_ref(gen_shape, disc_shape, thY, thU, thD, xy_free, xy_s, z, real, eps, 10.0, w_pde)
        assert np.isclose(losses[4], orc.free_generator_loss_ref(gen_shape, disc_shape, thY, thU, thD, xy_free, xy_s, z, w_pde), rtol=1e-13)
        h = 1e-6
        for th, g, which in ((thY, gY, 0), (thU, gU, 1)):
            fd = np.empty_like(g)
            for i in range(th.size):
                e = np.zeros_like(th); e[i] = h
                a = [thY, thU]; b = [thY, thU]
                a[which] = th + e; b[which] = th - e
                fd[i] = (orc.free_generator_loss_ref(gen_shape, disc_shape, a[0], a[1], thD, xy_free, xy_s, z, w_pde) -
                         orc.free_generator_loss_ref(gen_shape, disc_shape, b[0], b[1], thD, xy_free, xy_s, z, w_pde)) / (2 * h)
            assert np.abs(fd - g).max() <= 5e-7 * max(1.0, np.abs(g).max()), (w_pde, which, np.abs(fd - g).max())
        # L_D: the critic part is the pinned WGAN-GP of the base oracle on these snapshots
        X, _ = orc.free_snapshot_ref(gen_shape, thY, thU, xy_free, xy_s, z)
        assert np.isclose(losses[0], orc.critic_loss_ref(disc_shape, thD, real, X, eps, 10.0), rtol=1e-6)


def test_reduces_to_the_base_step_when_the_critic_ignores_f():
    """Zero first-layer critic weights on the f and coordinate columns, the same points for every sample and w_pde > 0:
    the generator gradients equal those of the pinned base oracle (f_target = 0) with the critic restricted to 2S inputs."""
    rng = np.random.default_rng(6)
    N, Fp, S, m, L, H, LD, HD = 2, 9, 3, 2, 3, 4, 2, 5
    gen_shape = (2 + m, L, H)
    thY = rng.normal(0, 0.6, size=orc.param_count(*gen_shape)); thU = rng.normal(0, 0.6, size=orc.param_count(*gen_shape))
    base_D = (2 * S, LD, HD); free_D = (2 * S + 3 * Fp, LD, HD)
    thD = rng.normal(0, 0.4, size=orc.param_count(*base_D))
    layers = orc.unpack_params(thD, *base_D)
    W1 = np.concatenate([layers[0][0], np.zeros((HD, 3 * Fp))], axis=1)
    thD_free = np.concatenate([W1.reshape(-1), layers[0][1]] + [np.concatenate([W.reshape(-1), b]) for W, b in layers[1:]])
    pts = rng.uniform(size=(Fp, 2)); xy_free = np.broadcast_to(pts, (N, Fp, 2)).copy()
    xy_s = rng.uniform(size=(S, 2)); z = rng.normal(size=(N, m)); eps = rng.uniform(size=N)
    real = rng.normal(size=(N, 2 * S)); real_free = np.concatenate([real, rng.normal(size=(N, 3 * Fp))], axis=1)
    gY, gU, gD, losses = orc.train_step_grads_free_ref(gen_shape, free_D, thY, thU, thD_free, xy_free, xy_s, z, real_free, eps, 10.0, 0.7)
    bY, bU, bD, blosses = orc.train_step_grads_ref(gen_shape, base_D, thY, thU, thD, pts, np.zeros(Fp), xy_s, z, real, eps, 10.0, 0.7)
    assert np.allclose(gY, bY, rtol=1e-10, atol=1e-14) and np.allclose(gU, bU, rtol=1e-10, atol=1e-14)
    assert np.allclose(losses[[1, 4, 5]], blosses[[1, 4, 5]], rtol=1e-12)
