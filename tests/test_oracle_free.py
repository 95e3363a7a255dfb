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


def test_score_mean_small_by_cancellation_is_ill_conditioned_in_f():
    """DESIGN.md reading R9, shown with the fp64 oracle alone.  In the 16-bit NEXT-2 parity case `c2-free` (tests/test_gpu_parity.py)
    mean D(fake) is 1.7 % of the critic's score scale.  Perturbing the f entries of X_fake by ONE FP16 half-ulp (2^-11, relative to
    max|f|; FP16 is the paper's activation precision) in the worst direction moves mean D(fake) by far more than 1e-3 of
    itself -- and by far less than 1e-3 of the score scale.  So no arithmetic that stores f (let alone the jets it is built from)
    in FP16 can promise north_star's 1e-3 on this number; the score-scale ruler is the one such a case is held to."""
    import dataclasses

    import workloads as wl
    from parity_util import free_case, free_score_sensitivity
    cfg, F = dataclasses.replace(wl.CONFIGS["c2"], name="c2-free", N=8, S=32), 64
    inp, disc_shape, xy_free, real = free_case(cfg, F)
    B, gf, f = free_score_sensitivity(cfg, F, inp, disc_shape, xy_free)
    S = cfg.S
    X, _ = orc.free_snapshot_ref(cfg.gen_shape, inp["theta_Y"], inp["theta_u"], xy_free, inp["xy_sensors"], inp["z"])
    D_fake = orc.disc_forward_ref(inp["theta_D"], *disc_shape, X).mean()
    D_real = orc.disc_forward_ref(inp["theta_D"], *disc_shape, real).mean()
    scale = max(abs(D_fake), abs(D_real))
    assert abs(D_fake) < 0.05 * scale                                        # small by cancellation
    Xp = X.copy()
    Xp[:, 2 * S:2 * S + F] += 2.0 ** -11 * np.abs(f).max() * np.sign(gf)     # one FP16 half-ulp of max|f|, worst direction
    moved = abs(orc.disc_forward_ref(inp["theta_D"], *disc_shape, Xp).mean() - D_fake)
    assert np.isclose(moved, B * 2.0 ** -11, rtol=0.05)                      # the first-order bound B is what actually happens
    assert moved > 10 * 1e-3 * abs(D_fake)                                   # > 10x north_star's ruler applied to the loss itself
    assert moved < 0.6 * 1e-3 * scale                                        # inside 1e-3 of the score scale
