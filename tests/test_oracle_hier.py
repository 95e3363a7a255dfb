"""Pins for the NEXT-3 oracle (hierarchical multi-discriminator loss; R10)."""
import numpy as np

from oracle import pigan_oracle as orc


def _args(tiny):
    return (tiny["xy_colloc"], tiny["f"], tiny["xy_sensors"], tiny["z"], tiny["real"], tiny["eps"], 10.0, 0.7)


def test_hierarchy_weights_of_the_papers_example():
    # "one subdomain at level 1, 19 subdomains at level 2, and 480 subdomains at level 3": weights 1/3, 1/57, 1/1440
    w = orc.hierarchy_weights([1, 19, 480])
    assert w.shape == (500,) and np.isclose(w[0], 1 / 3) and np.isclose(w[1], 1 / 57) and np.isclose(w[-1], 1 / 1440)
    assert np.isclose(w.sum(), 1.0)                         # every level carries 1 / levels: a weighted AVERAGE


def test_one_critic_on_the_whole_snapshot_is_the_base_step(tiny):
    cfg = tiny["cfg"]
    idx = np.arange(2 * cfg.S)[None, :]
    gY, gU, gD, losses = orc.train_step_grads_hier_ref(cfg.gen_shape, cfg.disc_shape, tiny["theta_Y"], tiny["theta_u"], [tiny["theta_D"]], idx, [1.0], *_args(tiny))
    bY, bU, bD, blosses = orc.train_step_grads_ref(cfg.gen_shape, cfg.disc_shape, tiny["theta_Y"], tiny["theta_u"], tiny["theta_D"], *_args(tiny))
    assert np.allclose(gY, bY, rtol=1e-12, atol=1e-16) and np.allclose(gU, bU, rtol=1e-12, atol=1e-16) and np.allclose(gD[0], bD, rtol=1e-12, atol=1e-16)
    assert np.allclose(losses, blosses, rtol=1e-13)


def test_two_copies_of_a_critic_with_half_weights_change_nothing_for_the_generator(tiny):
    cfg = tiny["cfg"]
    idx = np.arange(2 * cfg.S)[None, :]
    gY1, gU1, gD1, l1 = orc.train_step_grads_hier_ref(cfg.gen_shape, cfg.disc_shape, tiny["theta_Y"], tiny["theta_u"], [tiny["theta_D"]], idx, [1.0], *_args(tiny))
    gY2, gU2, gD2, l2 = orc.train_step_grads_hier_ref(cfg.gen_shape, cfg.disc_shape, tiny["theta_Y"], tiny["theta_u"], [tiny["theta_D"]] * 2,
                                                      np.repeat(idx, 2, axis=0), [0.5, 0.5], *_args(tiny))
    assert np.allclose(gY1, gY2, rtol=1e-12, atol=1e-16) and np.allclose(gU1, gU2, rtol=1e-12, atol=1e-16)
    assert np.allclose(gD2[0], gD1[0]) and np.allclose(gD2[1], gD1[0])       # each critic's own loss carries no weight
    assert np.isclose(l2[0], 2 * l1[0]) and np.isclose(l2[4], l1[4]) and np.isclose(l2[3], 2 * l1[3])


def test_generator_gradient_matches_finite_differences_with_overlapping_subdomains(tiny):
    cfg = tiny["cfg"]
    rng = np.random.default_rng(9)
    S = cfg.S
    d_sub = 4
    disc_shape = (d_sub, 2, 5)
    sens = [np.array([0, 1]), np.array([1, 3]), np.array([2, 3])]                    # sensors per subdomain (overlapping)
    subsets = np.stack([np.concatenate([s, S + s]) for s in sens])                  # their log k and u entries
    thDs = [rng.normal(0, 0.5, size=orc.param_count(*disc_shape)) for _ in sens]
    w = orc.hierarchy_weights([1, 2])
    gY, gU, gD, losses = orc.train_step_grads_hier_ref(cfg.gen_shape, disc_shape, tiny["theta_Y"], tiny["theta_u"], thDs, subsets, w, *_args(tiny))

    def L_G(thY, thU):                                                              # the plain definition
        Yc = orc.gen_jet_forward_ref(thY, *cfg.gen_shape, tiny["xy_colloc"], tiny["z"], 1)
        Uc = orc.gen_jet_forward_ref(thU, *cfg.gen_shape, tiny["xy_colloc"], tiny["z"], 2)
        _, msq = orc.darcy_residual_ref(Yc, Uc, tiny["f"])
        X = np.concatenate([orc.gen_jet_forward_ref(thY, *cfg.gen_shape, tiny["xy_sensors"], tiny["z"], 0)[0],
                            orc.gen_jet_forward_ref(thU, *cfg.gen_shape, tiny["xy_sensors"], tiny["z"], 0)[0]], axis=1)
        return sum(-w[k] * orc.disc_forward_ref(thDs[k], *disc_shape, X[:, subsets[k]]).mean() for k in range(3)) + 0.7 * msq

    assert np.isclose(losses[4], L_G(tiny["theta_Y"], tiny["theta_u"]), rtol=1e-13)
    h = 1e-6
    for th, g, which in ((tiny["theta_Y"], gY, 0), (tiny["theta_u"], gU, 1)):
        fd = np.empty_like(g)
        for i in range(th.size):
            e = np.zeros_like(th); e[i] = h
            a = [tiny["theta_Y"], tiny["theta_u"]]; b = [tiny["theta_Y"], tiny["theta_u"]]
            a[which] = th + e; b[which] = th - e
            fd[i] = (L_G(*a) - L_G(*b)) / (2 * h)
        assert np.abs(fd - g).max() <= 5e-7 * max(1.0, np.abs(g).max())
    # each critic's gradient is the pinned single-critic WGAN-GP gradient on its sub-snapshot
    X = np.concatenate([orc.gen_jet_forward_ref(tiny["theta_Y"], *cfg.gen_shape, tiny["xy_sensors"], tiny["z"], 0)[0],
                        orc.gen_jet_forward_ref(tiny["theta_u"], *cfg.gen_shape, tiny["xy_sensors"], tiny["z"], 0)[0]], axis=1)
    # (the VALUE, critic by critic, with DISTINCT subsets: a wrong real[:, idx] or fake[:, idx] for k > 0 fails here).
    # g_Dk = d/dtheta [mean D_k(fake_k) - mean D_k(real_k)] + d GP_k/dtheta: the Wasserstein part by central differences of the plain
    # forward disc_forward_ref in every parameter of critic k, the penalty part from gradient_penalty_ref (pinned on its own by
    # closed forms and torch fp64 double backward in test_oracle_critic.py) evaluated on critic k's sub-snapshots.
    for k in range(3):
        real_k, fake_k = tiny["real"][:, subsets[k]], X[:, subsets[k]]
        W = lambda th: orc.disc_forward_ref(th, *disc_shape, fake_k).mean() - orc.disc_forward_ref(th, *disc_shape, real_k).mean()
        fd = np.empty_like(thDs[k])
        for i in range(thDs[k].size):
            e = np.zeros_like(thDs[k]); e[i] = h
            fd[i] = (W(thDs[k] + e) - W(thDs[k] - e)) / (2 * h)
        _, _, gp_own = orc.gradient_penalty_ref(thDs[k], *disc_shape, real_k, fake_k, tiny["eps"], 10.0)
        assert np.abs(gD[k]).max() > 0 and gD[k].shape == fd.shape
        assert np.abs(fd + gp_own - gD[k]).max() <= 5e-7 * max(1.0, np.abs(gD[k]).max()), (k, np.abs(fd + gp_own - gD[k]).max())
        # and it is NOT the gradient on another critic's columns (the subsets are distinct, so the pin can tell them apart)
        other = subsets[(k + 1) % 3]
        _, _, gp_other = orc.gradient_penalty_ref(thDs[k], *disc_shape, tiny["real"][:, other], X[:, other], tiny["eps"], 10.0)
        assert np.abs(gp_other - gp_own).max() > 1e-3 * np.abs(gp_own).max()
