"""Pins for the NEXT-1 oracle (shared-trunk generator with two heads and skip connections; R7, R8).
None of them re-types the trunk's own formulas: finite differences, reduction to the already pinned two-MLP oracle, and a
special case in which the skip path is the only path."""
import numpy as np

from oracle import pigan_oracle as orc
from workloads import collocation_grid


def _rand_trunk(rng, in_dim, L, H, scale=0.6):
    return rng.normal(0.0, scale, size=orc.trunk_param_count(in_dim, L, H))


def test_trunk_param_count_and_packing():
    assert orc.trunk_param_count(6, 3, 32) == 2369 + 32 + 1            # one extra output row and bias
    lay = orc.unpack_trunk_params(np.arange(orc.trunk_param_count(5, 2, 4), dtype=float), 5, 2, 4)
    assert [w.shape for w, _ in lay] == [(4, 5), (4, 4), (2, 4)] and lay[-1][1].shape == (2,)


def test_jets_match_finite_differences_with_skips():
    rng = np.random.default_rng(3)
    in_dim, L, H = 5, 5, 6                                             # skips act at l = 3 and l = 5
    th = _rand_trunk(rng, in_dim, L, H)
    xy = rng.uniform(0.1, 0.9, size=(7, 2)); z = rng.normal(size=(2, 3))
    J = orc.trunk_jet_forward_ref(th, in_dim, L, H, xy, z, 2, True)
    h = 1e-4
    def val(dx, dy):
        return orc.trunk_jet_forward_ref(th, in_dim, L, H, xy + np.array([dx, dy]), z, 0, True)[:, 0]
    v0 = val(0, 0)
    assert np.allclose(J[:, 0], v0, rtol=0, atol=1e-14)
    assert np.allclose(J[:, 1], (val(h, 0) - val(-h, 0)) / (2 * h), atol=1e-7)
    assert np.allclose(J[:, 2], (val(0, h) - val(0, -h)) / (2 * h), atol=1e-7)
    assert np.allclose(J[:, 3], (val(h, 0) - 2 * v0 + val(-h, 0)) / h ** 2, atol=2e-6)
    assert np.allclose(J[:, 4], (val(0, h) - 2 * v0 + val(0, -h)) / h ** 2, atol=2e-6)
    # the skips do change the function
    assert np.abs(J - orc.trunk_jet_forward_ref(th, in_dim, L, H, xy, z, 2, False)).max() > 1e-3


def _split_into_two_mlps(th, in_dim, L, H):
    """Two plain MLPs that share every hidden weight with the trunk and take one head each."""
    lay = orc.unpack_trunk_params(th, in_dim, L, H)
    out = []
    for k in range(2):
        parts = [np.concatenate([W.reshape(-1), b]) for W, b in lay[:-1]]
        parts.append(np.concatenate([lay[-1][0][k], lay[-1][1][k:k + 1]]))
        out.append(np.concatenate(parts))
    return out


def test_without_skips_the_trunk_is_two_mlps_sharing_hidden_weights(tiny):
    cfg = tiny["cfg"]
    rng = np.random.default_rng(5)
    th = _rand_trunk(rng, *cfg.gen_shape, scale=0.5)
    thY, thU = _split_into_two_mlps(th, *cfg.gen_shape)
    J = orc.trunk_jet_forward_ref(th, *cfg.gen_shape, tiny["xy_colloc"], tiny["z"], 2, False)
    assert np.allclose(J[0], orc.gen_jet_forward_ref(thY, *cfg.gen_shape, tiny["xy_colloc"], tiny["z"], 2), rtol=1e-13, atol=1e-14)
    assert np.allclose(J[1], orc.gen_jet_forward_ref(thU, *cfg.gen_shape, tiny["xy_colloc"], tiny["z"], 2), rtol=1e-13, atol=1e-14)
    args = (tiny["theta_D"], tiny["xy_colloc"], tiny["f"], tiny["xy_sensors"], tiny["z"], tiny["real"], tiny["eps"], 10.0, 0.7)
    gG, gD, losses = orc.train_step_grads_trunk_ref(cfg.gen_shape, cfg.disc_shape, th, *args, skip=False)
    gY, gU, gD2, losses2 = orc.train_step_grads_ref(cfg.gen_shape, cfg.disc_shape, thY, thU, *args)
    assert np.allclose(losses, losses2, rtol=1e-12) and np.allclose(gD, gD2, rtol=1e-11, atol=1e-15)
    n_hidden = gY.size - (cfg.H + 1)
    assert np.allclose(gG[:n_hidden], gY[:n_hidden] + gU[:n_hidden], rtol=1e-10, atol=1e-14)      # shared weights: the two nets' gradients add
    H = cfg.H
    assert np.allclose(gG[n_hidden:n_hidden + H], gY[n_hidden:n_hidden + H], rtol=1e-10, atol=1e-14)          # head 0 weights
    assert np.allclose(gG[n_hidden + H:n_hidden + 2 * H], gU[n_hidden:n_hidden + H], rtol=1e-10, atol=1e-14)  # head 1 weights
    assert np.allclose(gG[-2], gY[-1], rtol=1e-10, atol=1e-14) and np.allclose(gG[-1], gU[-1], rtol=1e-10, atol=1e-14)


def test_skip_is_the_only_path_when_the_skipped_block_is_dead():
    """W_3 = 0, b_3 = 0 makes t^3 = 0, so h^3 = h^1 and the trunk equals the pinned one-hidden-layer MLP (per head)."""
    rng = np.random.default_rng(7)
    in_dim, L, H = 4, 3, 5
    th = _rand_trunk(rng, in_dim, L, H)
    lay = orc.unpack_trunk_params(th, in_dim, L, H)
    off3 = H * in_dim + H + (H * H + H)
    th[off3:off3 + H * H + H] = 0.0
    xy = rng.uniform(size=(6, 2)); z = rng.normal(size=(3, 2))
    J = orc.trunk_jet_forward_ref(th, in_dim, L, H, xy, z, 2, True)
    for k in range(2):
        one = np.concatenate([lay[0][0].reshape(-1), lay[0][1], lay[3][0][k], lay[3][1][k:k + 1]])
        assert np.allclose(J[k], orc.gen_jet_forward_ref(one, in_dim, 1, H, xy, z, 2), rtol=1e-13, atol=1e-14)


def test_trunk_gradients_match_finite_differences_of_L_G():
    rng = np.random.default_rng(11)
    gen_shape, disc_shape = (2 + 2, 5, 4), (2 * 3, 2, 5)
    th = _rand_trunk(rng, *gen_shape, scale=0.7)
    thD = rng.normal(0.0, 0.5, size=orc.param_count(*disc_shape))
    xy_c = collocation_grid(3).astype(np.float64); xy_s = rng.uniform(size=(3, 2)); z = rng.normal(size=(2, 2))
    f = rng.normal(size=9); real = rng.normal(size=(2, 6)); eps = rng.uniform(size=2)
    gG, _, losses = orc.train_step_grads_trunk_ref(gen_shape, disc_shape, th, thD, xy_c, f, xy_s, z, real, eps, 10.0, 0.7, skip=True)
    assert np.isclose(losses[4], orc.trunk_generator_loss_ref(gen_shape, disc_shape, th, thD, xy_c, f, xy_s, z, 0.7, True), rtol=1e-13)
    h = 1e-6
    fd = np.empty_like(gG)
    for i in range(th.size):
        e = np.zeros_like(th); e[i] = h
        fd[i] = (orc.trunk_generator_loss_ref(gen_shape, disc_shape, th + e, thD, xy_c, f, xy_s, z, 0.7, True) -
                 orc.trunk_generator_loss_ref(gen_shape, disc_shape, th - e, thD, xy_c, f, xy_s, z, 0.7, True)) / (2 * h)
    assert np.abs(fd - gG).max() <= 2e-7 * max(1.0, np.abs(gG).max()), np.abs(fd - gG).max()
