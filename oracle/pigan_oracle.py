"""fp64 CPU oracle for the PI-GAN hot path (arXiv 1910.13444).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference`` legs may
import this module.  The CUDA library under ``paper_1910_13444_b200/`` shares no code with it and never calls it.

Everything is plain numpy in float64.  Each function restates, step by step and in the paper's notation, what the
hot path computes; ``@`` (matmul) is the only library primitive used as a step.  No blocking, fusion or
reordering beyond a loop over latent samples n (both losses are sums over samples, so this is the definition).

Citations: ``P:<line>`` = /root/reference/PAPER.md line; ``S8c Ok`` = SURVEY.md section 8(c) step Ok, which fixes the
reading where the paper is silent (DESIGN.md section 3 lists every such reading).

  * generator (x, random vector) -> log k, u with tanh fully-connected layers ........ P:139
  * induced network for f = div(k grad u) by differentiating the generator in x ....... P:93 (Eq. 1)
  * snapshot = log k and u at the sensors, fed to the discriminator as one input ...... P:139
  * WGAN-GP critic loss (two-sided gradient penalty of ref. [24]) ..................... P:83
  * FP32 master weights / optimiser update (Adam by BASELINE.json) .................... P:155

Flat parameter packing (same as include/pigan.h): for l = 1..n_hidden+1: W_l row-major [out][in], then b_l [out].
Generator W_1 columns are ordered [x, y, z_1..z_m].

Parity pins (tests/test_oracle_*.py): central finite differences of the value channel; the closed-form jet of a
one-hidden-unit network; manufactured Darcy solutions; finite differences of L_G and L_D on tiny inputs; the
closed-form gradient norm of a one-hidden-unit critic; torch float64 double-backward as a library special case;
invariants (output-bias gradient of L_D is exactly 0, eps = 0/1, sample additivity, linearity in w_pde); Adam
closed form and a hand-computed three-step fixture (tests/golden/adam_three_steps.txt).
Parity against the paper's *trained* results (Figs. 5-11) is UNPINNED: no datasets, weights or code exist here.
"""
from __future__ import annotations

import numpy as np

F64 = np.float64


# --------------------------------------------------------------------------------------------------------------
# parameter packing
# --------------------------------------------------------------------------------------------------------------
def param_count(in_dim: int, n_hidden: int, width: int) -> int:
    """H(in)+H + (L-1)(H^2+H) + H+1 (scalar linear output; S8 table 'params per generator net')."""
    return width * in_dim + width + (n_hidden - 1) * (width * width + width) + width + 1


def unpack_params(theta, in_dim: int, n_hidden: int, width: int):
    """theta (flat) -> [(W_1,b_1), ..., (W_{L+1}, b_{L+1})], W_l is [out][in]."""
    theta = np.asarray(theta, dtype=F64)
    assert theta.shape == (param_count(in_dim, n_hidden, width),), theta.shape
    layers, off, fan_in = [], 0, in_dim
    for l in range(n_hidden + 1):
        fan_out = width if l < n_hidden else 1
        W = theta[off:off + fan_out * fan_in].reshape(fan_out, fan_in); off += fan_out * fan_in
        b = theta[off:off + fan_out]; off += fan_out
        layers.append((W, b)); fan_in = fan_out
    return layers


def pack_grads(grads) -> np.ndarray:
    """[(gW_1, gb_1), ...] -> flat vector in the parameter packing order."""
    return np.concatenate([np.concatenate([gW.reshape(-1), gb.reshape(-1)]) for gW, gb in grads])


# --------------------------------------------------------------------------------------------------------------
# O1 + O2: generator MLP and its second-order spatial jet
# --------------------------------------------------------------------------------------------------------------
N_CHANNELS = {0: 1, 1: 3, 2: 5}      # jet_order -> C; channels are (value, d/dx, d/dy, d2/dx2, d2/dy2)


def _jet_forward_one_sample(layers, xy, z_n, C, keep_tape=False):
    """One latent sample z_n at all points xy [P,2].  Returns out [C,P] (and the tape for the reverse sweep).

    S8c O1: a^1 = W_1[:,0] x + W_1[:,1] y + W_1[:,2:] z + b_1; h^l = tanh(a^l); a^{l+1} = W_{l+1} h^l + b_{l+1};
            output o = a^{L+1} (linear).
    S8c O2: layer 1: a_x = W_1[:,0], a_y = W_1[:,1], a_xx = a_yy = 0.  At each hidden layer with t = tanh a,
            s = 1 - t^2, q = -2ts:  h = t, h_x = s a_x, h_y = s a_y, h_xx = s a_xx + q a_x^2, h_yy = s a_yy + q a_y^2.
            Next pre-activations a_c <- W h_c, bias on the value channel only.
    """
    W1, b1 = layers[0]
    P = xy.shape[0]
    H = W1.shape[0]
    x, y = xy[:, 0:1], xy[:, 1:2]
    a = [None] * C
    a[0] = x * W1[:, 0][None, :] + y * W1[:, 1][None, :] + (W1[:, 2:] @ z_n + b1)[None, :]     # [P,H]
    if C >= 3:
        a[1] = np.broadcast_to(W1[:, 0], (P, H)).copy()
        a[2] = np.broadcast_to(W1[:, 1], (P, H)).copy()
    if C >= 5:
        a[3] = np.zeros((P, H), dtype=F64)
        a[4] = np.zeros((P, H), dtype=F64)
    tape = []
    for l in range(1, len(layers)):
        t = np.tanh(a[0]); s = 1.0 - t * t; q = -2.0 * t * s
        h = [None] * C
        h[0] = t
        if C >= 3:
            h[1] = s * a[1]; h[2] = s * a[2]
        if C >= 5:
            h[3] = s * a[3] + q * a[1] * a[1]
            h[4] = s * a[4] + q * a[2] * a[2]
        if keep_tape:
            tape.append((t, a[1:], h))
        W, b = layers[l]
        a = [h[c] @ W.T for c in range(C)]
        a[0] = a[0] + b[None, :]
    out = np.stack([a[c][:, 0] for c in range(C)])                                             # [C,P]
    return (out, tape) if keep_tape else out


def gen_jet_forward_ref(theta, in_dim, n_hidden, width, xy, z, jet_order):
    """out [C][n_samples][n_pts]: generator value and spatial derivatives (oracle of pigan_gen_jet_forward)."""
    layers = unpack_params(theta, in_dim, n_hidden, width)
    xy = np.asarray(xy, dtype=F64); z = np.asarray(z, dtype=F64)
    C = N_CHANNELS[jet_order]
    out = np.empty((C, z.shape[0], xy.shape[0]), dtype=F64)
    for n in range(z.shape[0]):
        out[:, n, :] = _jet_forward_one_sample(layers, xy, z[n], C)
    return out


def _jet_backward_one_sample(layers, xy, z_n, tape, o_hat, C, grads):
    """Reverse sweep for one sample.  o_hat [C,P] = adjoints of the outputs; accumulates into grads (S8c O4).

    Given h_hat_c and the stored t, a_x, a_y, a_xx, a_yy, with q' = -2s(1 - 3t^2):
      a_hat_xx = s h_hat_xx; a_hat_yy = s h_hat_yy; a_hat_x = s h_hat_x + 2 q a_x h_hat_xx; a_hat_y likewise;
      a_hat = s h_hat + q (a_x h_hat_x + a_y h_hat_y + a_xx h_hat_xx + a_yy h_hat_yy) + q' (a_x^2 h_hat_xx + a_y^2 h_hat_yy).
    Linear part: W_hat_l += sum_rows sum_c a_hat_c (x) h_c^{l-1}; b_hat_l += sum_rows a_hat (value channel only);
      h_hat_c^{l-1} = W_l^T a_hat_c.
    First layer: W_hat_1[:,0] = sum (a_hat x_p + a_hat_x); W_hat_1[:,1] = sum (a_hat y_p + a_hat_y);
      W_hat_1[:,2:] = (sum_p a_hat) (x) z_n; b_hat_1 = sum a_hat.
    """
    a_hat = [o_hat[c][:, None] for c in range(C)]                     # adjoints of a^{L+1}_c, [P,1]
    for l in range(len(layers) - 1, 0, -1):
        t, a_der, h = tape[l - 1]
        W, _ = layers[l]
        gW, gb = grads[l]
        for c in range(C):
            gW += a_hat[c].T @ h[c]
        gb += a_hat[0].sum(axis=0)
        h_hat = [a_hat[c] @ W for c in range(C)]
        s = 1.0 - t * t; q = -2.0 * t * s; qp = -2.0 * s * (1.0 - 3.0 * t * t)
        new = [None] * C
        val = s * h_hat[0]
        if C >= 3:
            a_x, a_y = a_der[0], a_der[1]
            val = val + q * (a_x * h_hat[1] + a_y * h_hat[2])
            new[1] = s * h_hat[1]; new[2] = s * h_hat[2]
        if C >= 5:
            a_xx, a_yy = a_der[2], a_der[3]
            val = val + q * (a_xx * h_hat[3] + a_yy * h_hat[4]) + qp * (a_x * a_x * h_hat[3] + a_y * a_y * h_hat[4])
            new[1] = new[1] + 2.0 * q * a_x * h_hat[3]
            new[2] = new[2] + 2.0 * q * a_y * h_hat[4]
            new[3] = s * h_hat[3]; new[4] = s * h_hat[4]
        new[0] = val
        a_hat = new
    gW1, gb1 = grads[0]
    col = a_hat[0].sum(axis=0)                                        # sum over points, [H]
    gW1[:, 0] += (a_hat[0] * xy[:, 0:1]).sum(axis=0)
    gW1[:, 1] += (a_hat[0] * xy[:, 1:2]).sum(axis=0)
    if C >= 3:
        gW1[:, 0] += a_hat[1].sum(axis=0)
        gW1[:, 1] += a_hat[2].sum(axis=0)
    gW1[:, 2:] += np.outer(col, z_n)
    gb1 += col


def _zero_grads(layers):
    return [(np.zeros_like(W), np.zeros_like(b)) for W, b in layers]


# --------------------------------------------------------------------------------------------------------------
# O3: Darcy residual  r = div(k grad u) - f  with k = exp(Y)     (Eq. 1)
# --------------------------------------------------------------------------------------------------------------
def darcy_residual_ref(logk_jet, u_jet, f):
    """r[n][p] = exp(Y)(Y_x u_x + Y_y u_y + u_xx + u_yy) - f[p];  returns (r, mean r^2).

    div(k grad u) = grad k . grad u + k lap u and grad k = k grad(log k), which is Eq. 1 expanded for k = exp(Y).
    logk_jet is [>=3][N][P] (value, x, y), u_jet is [5][N][P].
    """
    Y = np.asarray(logk_jet, dtype=F64); U = np.asarray(u_jet, dtype=F64); f = np.asarray(f, dtype=F64)
    k = np.exp(Y[0])
    D = Y[1] * U[1] + Y[2] * U[2] + U[3] + U[4]
    r = k * D - f[None, :]
    return r, float(np.mean(r * r))


def _residual_adjoints(Yj, Uj, f_row, w_pde, NP):
    """S8c O3 for one sample: r_hat = 2 w_pde r / (N P);
    Y_hat = r_hat k D, Y_hat_x = r_hat k u_x, Y_hat_y = r_hat k u_y;
    u_hat = 0, u_hat_x = r_hat k Y_x, u_hat_y = r_hat k Y_y, u_hat_xx = u_hat_yy = r_hat k."""
    k = np.exp(Yj[0]); D = Yj[1] * Uj[1] + Yj[2] * Uj[2] + Uj[3] + Uj[4]
    r = k * D - f_row
    rh = 2.0 * w_pde * r / NP
    Y_hat = np.stack([rh * k * D, rh * k * Uj[1], rh * k * Uj[2]])
    U_hat = np.stack([np.zeros_like(r), rh * k * Yj[1], rh * k * Yj[2], rh * k, rh * k])
    return r, Y_hat, U_hat


# --------------------------------------------------------------------------------------------------------------
# O5-O7: discriminator (critic), gradient penalty and its double backward
# --------------------------------------------------------------------------------------------------------------
def _disc_forward(layers, X):
    """g^0 = X; g^l = tanh(V_l g^{l-1} + c_l); D = v_out . g^{L_D} + c_out.  Returns ([g^0..g^{L_D}], D[B])."""
    g = [X]
    for l in range(len(layers) - 1):
        V, c = layers[l]
        g.append(np.tanh(g[-1] @ V.T + c[None, :]))
    V, c = layers[-1]
    return g, (g[-1] @ V.T + c[None, :])[:, 0]


def disc_forward_ref(theta_d, in_dim, n_hidden, width, snap):
    """score[B] (oracle of pigan_disc_forward)."""
    layers = unpack_params(theta_d, in_dim, n_hidden, width)
    return _disc_forward(layers, np.asarray(snap, dtype=F64))[1]


def _disc_backward(layers, g, seed, grads):
    """Ordinary backprop of sum_b seed[b] D(X_b); accumulates weight grads (if grads is not None), returns d/dX."""
    LD = len(layers) - 1
    a_hat = seed[:, None]                                  # adjoint of the output pre-activation, [B,1]
    if grads is not None:
        grads[LD][0][...] += a_hat.T @ g[LD]; grads[LD][1][...] += a_hat.sum(axis=0)
    g_hat = a_hat @ layers[LD][0]
    for l in range(LD, 0, -1):
        a_hat = g_hat * (1.0 - g[l] * g[l])
        if grads is not None:
            grads[l - 1][0][...] += a_hat.T @ g[l - 1]; grads[l - 1][1][...] += a_hat.sum(axis=0)
        g_hat = a_hat @ layers[l - 1][0]
    return g_hat


def _gradient_penalty(layers, Xhat, lam, grads):
    """S8c O5 + O6.  gp = lam * mean_n (||grad_X D(xhat_n)||_2 - 1)^2 ; accumulates d gp / d theta into grads.

    O5: forward stores g^l, s^l = 1 - (g^l)^2.  Backward-to-input: gbar^{L_D} = v_out; for l = L_D..1:
        abar^l = gbar^l * s^l, gbar^{l-1} = V_l^T abar^l;  G = gbar^0;  nu = ||G||_2 (no epsilon; nu = 0 -> seed 0).
    O6: seed adj(gbar^0) = (lam/N) 2 (nu - 1) G / nu.
        Ascending l = 1..L_D: adj(abar^l) = V_l adj(gbar^{l-1}); V_hat_l += abar^l (x) adj(gbar^{l-1});
            adj(s^l) = adj(abar^l) * gbar^l; adj(gbar^l) = adj(abar^l) * s^l.  Top: v_hat_out += adj(gbar^{L_D}).
        Descending l = L_D..1 with running adj(g) (starts 0): adj(g^l) += -2 g^l * adj(s^l); adj(a^l) = adj(g^l) * s^l;
            V_hat_l += adj(a^l) (x) g^{l-1}; c_hat_l += adj(a^l); adj(g^{l-1}) = V_l^T adj(a^l).
    """
    B = Xhat.shape[0]
    LD = len(layers) - 1
    g, _ = _disc_forward(layers, Xhat)
    s = [None] + [1.0 - g[l] * g[l] for l in range(1, LD + 1)]
    gbar = [None] * (LD + 1); abar = [None] * (LD + 1)
    gbar[LD] = np.broadcast_to(layers[LD][0][0], (B, layers[LD][0].shape[1])).copy()
    for l in range(LD, 0, -1):
        abar[l] = gbar[l] * s[l]
        gbar[l - 1] = abar[l] @ layers[l - 1][0]
    G = gbar[0]
    nu = np.sqrt((G * G).sum(axis=1))
    gp = lam * float(np.mean((nu - 1.0) ** 2))
    if grads is not None:
        safe = np.where(nu > 0.0, nu, 1.0)
        adj_gbar = (lam / B) * 2.0 * ((nu - 1.0) / safe)[:, None] * G
        adj_gbar[nu == 0.0] = 0.0
        adj_s = [None] * (LD + 1)
        for l in range(1, LD + 1):
            adj_abar = adj_gbar @ layers[l - 1][0].T
            grads[l - 1][0][...] += abar[l].T @ adj_gbar
            adj_s[l] = adj_abar * gbar[l]
            adj_gbar = adj_abar * s[l]
        grads[LD][0][...] += adj_gbar.sum(axis=0, keepdims=True)
        adj_g = np.zeros_like(g[LD])
        for l in range(LD, 0, -1):
            adj_g = adj_g + (-2.0 * g[l]) * adj_s[l]
            adj_a = adj_g * s[l]
            grads[l - 1][0][...] += adj_a.T @ g[l - 1]
            grads[l - 1][1][...] += adj_a.sum(axis=0)
            adj_g = adj_a @ layers[l - 1][0]
    return gp, nu


def gradient_penalty_ref(theta_d, in_dim, n_hidden, width, real, fake, eps, lam):
    """(gp, grad_norm[B], d gp / d theta_D) with xhat_n = eps_n real_n + (1 - eps_n) fake_n  (ref. [24] via P:83)."""
    layers = unpack_params(theta_d, in_dim, n_hidden, width)
    real = np.asarray(real, dtype=F64); fake = np.asarray(fake, dtype=F64); eps = np.asarray(eps, dtype=F64)
    Xhat = eps[:, None] * real + (1.0 - eps[:, None]) * fake
    grads = _zero_grads(layers)
    gp, nu = _gradient_penalty(layers, Xhat, lam, grads)
    return gp, nu, pack_grads(grads)


# --------------------------------------------------------------------------------------------------------------
# the whole step: both gradient sets at the same current weights (S8c definition of L_D, L_G; reading G16)
# --------------------------------------------------------------------------------------------------------------
def train_step_grads_ref(gen_shape, disc_shape, theta_Y, theta_u, theta_D, xy_colloc, f, xy_sensors, z,
                         real_snap, eps, gp_lambda=10.0, pde_weight=1.0):
    """Oracle of pigan_train_step_grads.

    gen_shape = (in_dim = 2 + m, n_hidden, width) for both G_logk and G_u; disc_shape likewise with in_dim = 2S.
    L_D = mean D(fake) - mean D(real) + lam mean (||grad D(xhat)|| - 1)^2     (X_fake held constant)
    L_G = -mean D(fake) + w_pde mean_{n,p} r(n,p)^2                           (theta_D held constant)
    Returns g_Y, g_u, g_D (flat) and losses = [L_D, mean D(fake), mean D(real), GP, L_G, L_pde].
    """
    lay_Y = unpack_params(theta_Y, *gen_shape); lay_u = unpack_params(theta_u, *gen_shape)
    lay_D = unpack_params(theta_D, *disc_shape)
    xy_c = np.asarray(xy_colloc, dtype=F64); xy_s = np.asarray(xy_sensors, dtype=F64)
    f = np.asarray(f, dtype=F64); z = np.asarray(z, dtype=F64)
    real = np.asarray(real_snap, dtype=F64); eps = np.asarray(eps, dtype=F64)
    N, P, S = z.shape[0], xy_c.shape[0], xy_s.shape[0]

    # a6: sensor evaluation + snapshot  X_fake[n] = [Y(s_1..S; z_n), u(s_1..S; z_n)]   (S8c G6, G7, G14)
    X_fake = np.empty((N, 2 * S), dtype=F64)
    sens_tapes = []
    for n in range(N):
        oY, tY = _jet_forward_one_sample(lay_Y, xy_s, z[n], 1, keep_tape=True)
        ou, tu = _jet_forward_one_sample(lay_u, xy_s, z[n], 1, keep_tape=True)
        X_fake[n, :S] = oY[0]; X_fake[n, S:] = ou[0]
        sens_tapes.append((tY, tu))

    # a7-a9: critic losses and gradient w.r.t. theta_D
    gD = _zero_grads(lay_D)
    g_fake, D_fake = _disc_forward(lay_D, X_fake)
    g_real, D_real = _disc_forward(lay_D, real)
    _disc_backward(lay_D, g_fake, np.full(N, 1.0 / N), gD)
    _disc_backward(lay_D, g_real, np.full(N, -1.0 / N), gD)
    Xhat = eps[:, None] * real + (1.0 - eps[:, None]) * X_fake
    gp, _ = _gradient_penalty(lay_D, Xhat, gp_lambda, gD)
    L_D = float(D_fake.mean() - D_real.mean() + gp)

    # O7: generator's critic term, dL_G/dX_fake[n] = -(1/N) grad_X D(X_fake[n]); theta_D gets nothing from it
    dX = _disc_backward(lay_D, g_fake, np.full(N, -1.0 / N), None)

    # a1-a5, a10: collocation jets, residual, reverse sweep; sensors seeded through the value channel
    gY = _zero_grads(lay_Y); gu = _zero_grads(lay_u)
    sum_r2 = 0.0
    for n in range(N):
        Yj, tY = _jet_forward_one_sample(lay_Y, xy_c, z[n], 3, keep_tape=True)
        Uj, tU = _jet_forward_one_sample(lay_u, xy_c, z[n], 5, keep_tape=True)
        r, Y_hat, U_hat = _residual_adjoints(Yj, Uj, f, pde_weight, N * P)
        sum_r2 += float((r * r).sum())
        _jet_backward_one_sample(lay_Y, xy_c, z[n], tY, Y_hat, 3, gY)
        _jet_backward_one_sample(lay_u, xy_c, z[n], tU, U_hat, 5, gu)
        tYs, tus = sens_tapes[n]
        _jet_backward_one_sample(lay_Y, xy_s, z[n], tYs, dX[n:n + 1, :S], 1, gY)
        _jet_backward_one_sample(lay_u, xy_s, z[n], tus, dX[n:n + 1, S:], 1, gu)
    L_pde = sum_r2 / (N * P)
    L_G = float(-D_fake.mean() + pde_weight * L_pde)
    losses = np.array([L_D, D_fake.mean(), D_real.mean(), gp, L_G, L_pde], dtype=F64)
    return pack_grads(gY), pack_grads(gu), pack_grads(gD), losses


def generator_loss_ref(gen_shape, disc_shape, theta_Y, theta_u, theta_D, xy_colloc, f, xy_sensors, z, pde_weight=1.0):
    """L_G written as its plain definition (used by the finite-difference pins only)."""
    S = np.asarray(xy_sensors).shape[0]
    Yc = gen_jet_forward_ref(theta_Y, *gen_shape, xy_colloc, z, 1)
    Uc = gen_jet_forward_ref(theta_u, *gen_shape, xy_colloc, z, 2)
    _, mean_sq = darcy_residual_ref(Yc, Uc, f)
    Ys = gen_jet_forward_ref(theta_Y, *gen_shape, xy_sensors, z, 0)[0]
    Us = gen_jet_forward_ref(theta_u, *gen_shape, xy_sensors, z, 0)[0]
    X_fake = np.concatenate([Ys, Us], axis=1)
    assert X_fake.shape[1] == 2 * S
    return float(-disc_forward_ref(theta_D, *disc_shape, X_fake).mean() + pde_weight * mean_sq)


def critic_loss_ref(disc_shape, theta_D, real, fake, eps, lam):
    """L_D written as its plain definition, with the input gradient taken by central differences of D in X
    (used by the finite-difference pins only; independent of the O5/O6 sweeps)."""
    real = np.asarray(real, dtype=F64); fake = np.asarray(fake, dtype=F64); eps = np.asarray(eps, dtype=F64)
    Xhat = eps[:, None] * real + (1.0 - eps[:, None]) * fake
    h = 1e-6
    G = np.empty_like(Xhat)
    for j in range(Xhat.shape[1]):
        e = np.zeros(Xhat.shape[1]); e[j] = h
        G[:, j] = (disc_forward_ref(theta_D, *disc_shape, Xhat + e) - disc_forward_ref(theta_D, *disc_shape, Xhat - e)) / (2 * h)
    nu = np.sqrt((G * G).sum(axis=1))
    return float(disc_forward_ref(theta_D, *disc_shape, fake).mean() - disc_forward_ref(theta_D, *disc_shape, real).mean()
                 + lam * np.mean((nu - 1.0) ** 2))


# --------------------------------------------------------------------------------------------------------------
# O8: Adam (S8c G3: epsilon outside the square root, 1-based step, bias correction)
# --------------------------------------------------------------------------------------------------------------
def adam_update_ref(theta, g, m, v, step, lr, beta1, beta2, adam_eps, skip=False):
    """m <- b1 m + (1-b1) g; v <- b2 v + (1-b2) g^2; mhat = m/(1-b1^t); vhat = v/(1-b2^t);
    theta <- theta - lr mhat / (sqrt(vhat) + eps).  skip=True leaves (theta, m, v) untouched.  Returns new copies."""
    theta = np.array(theta, dtype=F64); g = np.asarray(g, dtype=F64)
    m = np.array(m, dtype=F64); v = np.array(v, dtype=F64)
    if skip:
        return theta, m, v
    m = beta1 * m + (1.0 - beta1) * g
    v = beta2 * v + (1.0 - beta2) * g * g
    mhat = m / (1.0 - beta1 ** step)
    vhat = v / (1.0 - beta2 ** step)
    theta = theta - lr * mhat / (np.sqrt(vhat) + adam_eps)
    return theta, m, v


# ==============================================================================================================
# NEXT-1: the paper's own generator -- ONE set of weights, separate log k and u outputs in the final
# layer, residual connections that skip intermediate layers.  DESIGN.md readings R7 (heads) and R8 (skips):
#   trunk   a^1 = W_1 [x, y, z] + b_1;  t^l = tanh(a^l);  h^l = t^l + h^{l-2} when l is odd and l >= 3 (a two-layer residual
#           block, ref. [30]), else h^l = t^l;  a^{l+1} = W_{l+1} h^l + b_{l+1};
#   heads   [log k, u] = W_{L+1} h^L + b_{L+1} with W_{L+1} of shape [2][H] (row 0: log k, row 1: u).
# The spatial jet of h^L serves both heads, so the trunk carries 5 channels once; log k uses the first 3 of them.
# Flat packing: as for the plain MLP, with the last layer W [2][H] then b [2].
# ==============================================================================================================
def trunk_param_count(in_dim: int, n_hidden: int, width: int) -> int:
    return width * in_dim + width + (n_hidden - 1) * (width * width + width) + 2 * width + 2


def unpack_trunk_params(theta, in_dim: int, n_hidden: int, width: int):
    theta = np.asarray(theta, dtype=F64)
    assert theta.shape == (trunk_param_count(in_dim, n_hidden, width),), theta.shape
    layers, off, fan_in = [], 0, in_dim
    for l in range(n_hidden + 1):
        fan_out = width if l < n_hidden else 2
        W = theta[off:off + fan_out * fan_in].reshape(fan_out, fan_in); off += fan_out * fan_in
        b = theta[off:off + fan_out]; off += fan_out
        layers.append((W, b)); fan_in = fan_out
    return layers


def _skip_source(l: int, skip: bool):
    """Hidden layer l (1-based) adds h^{l-2} when skips are on and l is odd and >= 3 (reading R8)."""
    return l - 2 if (skip and l >= 3 and l % 2 == 1) else None


def _trunk_forward_one_sample(layers, xy, z_n, C, skip, keep_tape=False):
    """One latent sample at all points xy [P,2]: returns out [2][C][P] (head 0 = log k, head 1 = u) and the tape."""
    W1, b1 = layers[0]
    P, H = xy.shape[0], W1.shape[0]
    L = len(layers) - 1
    x, y = xy[:, 0:1], xy[:, 1:2]
    a = [None] * C
    a[0] = x * W1[:, 0][None, :] + y * W1[:, 1][None, :] + (W1[:, 2:] @ z_n + b1)[None, :]
    if C >= 3:
        a[1] = np.broadcast_to(W1[:, 0], (P, H)).copy(); a[2] = np.broadcast_to(W1[:, 1], (P, H)).copy()
    if C >= 5:
        a[3] = np.zeros((P, H), dtype=F64); a[4] = np.zeros((P, H), dtype=F64)
    hs = [None] * (L + 1)                                   # hs[l] = h^l (list of C arrays), l = 1..L
    tape = []
    for l in range(1, L + 1):
        t = np.tanh(a[0]); s = 1.0 - t * t; q = -2.0 * t * s
        tj = [None] * C                                     # jet of t^l = tanh(a^l)   (O2)
        tj[0] = t
        if C >= 3:
            tj[1] = s * a[1]; tj[2] = s * a[2]
        if C >= 5:
            tj[3] = s * a[3] + q * a[1] * a[1]; tj[4] = s * a[4] + q * a[2] * a[2]
        src = _skip_source(l, skip)
        h = [tj[c] + hs[src][c] for c in range(C)] if src is not None else tj
        hs[l] = h
        if keep_tape:
            tape.append((t, a[1:], h))
        W, b = layers[l]
        a = [h[c] @ W.T for c in range(C)]
        a[0] = a[0] + b[None, :]
    out = np.stack([np.stack([a[c][:, k] for c in range(C)]) for k in range(2)])          # [2][C][P]
    return (out, tape) if keep_tape else out


def trunk_jet_forward_ref(theta, in_dim, n_hidden, width, xy, z, jet_order, skip):
    """out [2][C][n_samples][n_pts]: head 0 = log k, head 1 = u, with their spatial jets."""
    layers = unpack_trunk_params(theta, in_dim, n_hidden, width)
    xy = np.asarray(xy, dtype=F64); z = np.asarray(z, dtype=F64)
    C = N_CHANNELS[jet_order]
    out = np.empty((2, C, z.shape[0], xy.shape[0]), dtype=F64)
    for n in range(z.shape[0]):
        out[:, :, n, :] = _trunk_forward_one_sample(layers, xy, z[n], C, skip)
    return out


def _trunk_backward_one_sample(layers, xy, z_n, tape, o_hat, C, skip, grads):
    """Reverse sweep of the trunk for one sample.  o_hat [2][C][P] = adjoints of the two heads' outputs.
    O4 applies to t^l = tanh(a^l); a skip h^l = t^l + h^{l-2} passes the adjoint of h^l on to h^{l-2} unchanged."""
    L = len(layers) - 1
    W_out, _ = layers[L]
    gWo, gbo = grads[L]
    t_L, _, h_L = tape[L - 1]
    for k in range(2):
        for c in range(C):
            gWo[k] += o_hat[k][c] @ h_L[c]
        gbo[k] += o_hat[k][0].sum()
    h_hat = {L: [o_hat[0][c][:, None] * W_out[0][None, :] + o_hat[1][c][:, None] * W_out[1][None, :] for c in range(C)]}
    for l in range(L, 0, -1):
        t, a_der, _ = tape[l - 1]
        hh = h_hat.pop(l)
        src = _skip_source(l, skip)
        if src is not None:                                 # h^l = t^l + h^{l-2}
            h_hat[src] = [hh[c].copy() for c in range(C)]
        s = 1.0 - t * t; q = -2.0 * t * s; qp = -2.0 * s * (1.0 - 3.0 * t * t)
        a_hat = [None] * C
        val = s * hh[0]
        if C >= 3:
            a_x, a_y = a_der[0], a_der[1]
            val = val + q * (a_x * hh[1] + a_y * hh[2])
            a_hat[1] = s * hh[1]; a_hat[2] = s * hh[2]
        if C >= 5:
            a_xx, a_yy = a_der[2], a_der[3]
            val = val + q * (a_xx * hh[3] + a_yy * hh[4]) + qp * (a_x * a_x * hh[3] + a_y * a_y * hh[4])
            a_hat[1] = a_hat[1] + 2.0 * q * a_x * hh[3]
            a_hat[2] = a_hat[2] + 2.0 * q * a_y * hh[4]
            a_hat[3] = s * hh[3]; a_hat[4] = s * hh[4]
        a_hat[0] = val
        if l >= 2:
            W, _ = layers[l - 1]                            # W_l (layers[] is 0-based)
            gW, gb = grads[l - 1]
            h_prev = tape[l - 2][2]
            for c in range(C):
                gW += a_hat[c].T @ h_prev[c]
            gb += a_hat[0].sum(axis=0)
            back = [a_hat[c] @ W for c in range(C)]
            if (l - 1) in h_hat:
                h_hat[l - 1] = [h_hat[l - 1][c] + back[c] for c in range(C)]
            else:
                h_hat[l - 1] = back
        else:
            gW1, gb1 = grads[0]
            col = a_hat[0].sum(axis=0)
            gW1[:, 0] += (a_hat[0] * xy[:, 0:1]).sum(axis=0)
            gW1[:, 1] += (a_hat[0] * xy[:, 1:2]).sum(axis=0)
            if C >= 3:
                gW1[:, 0] += a_hat[1].sum(axis=0); gW1[:, 1] += a_hat[2].sum(axis=0)
            gW1[:, 2:] += np.outer(col, z_n)
            gb1 += col


def train_step_grads_trunk_ref(gen_shape, disc_shape, theta_G, theta_D, xy_colloc, f, xy_sensors, z, real_snap, eps,
                               gp_lambda=10.0, pde_weight=1.0, skip=True):
    """Oracle of the step with the paper's generator (NEXT-1).  Same losses as train_step_grads_ref; the generator is
    the shared trunk.  Returns g_G, g_D (flat) and losses = [L_D, mean D(fake), mean D(real), GP, L_G, L_pde]."""
    lay_G = unpack_trunk_params(theta_G, *gen_shape); lay_D = unpack_params(theta_D, *disc_shape)
    xy_c = np.asarray(xy_colloc, dtype=F64); xy_s = np.asarray(xy_sensors, dtype=F64)
    f = np.asarray(f, dtype=F64); z = np.asarray(z, dtype=F64)
    real = np.asarray(real_snap, dtype=F64); eps = np.asarray(eps, dtype=F64)
    N, P, S = z.shape[0], xy_c.shape[0], xy_s.shape[0]
    X_fake = np.empty((N, 2 * S), dtype=F64)
    sens_tapes = []
    for n in range(N):
        o, tp = _trunk_forward_one_sample(lay_G, xy_s, z[n], 1, skip, keep_tape=True)
        X_fake[n, :S] = o[0][0]; X_fake[n, S:] = o[1][0]
        sens_tapes.append(tp)
    gD = _zero_grads(lay_D)
    g_fake, D_fake = _disc_forward(lay_D, X_fake)
    g_real, D_real = _disc_forward(lay_D, real)
    _disc_backward(lay_D, g_fake, np.full(N, 1.0 / N), gD)
    _disc_backward(lay_D, g_real, np.full(N, -1.0 / N), gD)
    Xhat = eps[:, None] * real + (1.0 - eps[:, None]) * X_fake
    gp, _ = _gradient_penalty(lay_D, Xhat, gp_lambda, gD)
    L_D = float(D_fake.mean() - D_real.mean() + gp)
    dX = _disc_backward(lay_D, g_fake, np.full(N, -1.0 / N), None)
    gG = _zero_grads(lay_G)
    sum_r2 = 0.0
    for n in range(N):
        o, tp = _trunk_forward_one_sample(lay_G, xy_c, z[n], 5, skip, keep_tape=True)
        r, Y_hat, U_hat = _residual_adjoints(o[0][:3], o[1], f, pde_weight, N * P)
        sum_r2 += float((r * r).sum())
        zero = np.zeros_like(r)
        o_hat = [[Y_hat[0], Y_hat[1], Y_hat[2], zero, zero], [U_hat[c] for c in range(5)]]
        _trunk_backward_one_sample(lay_G, xy_c, z[n], tp, o_hat, 5, skip, gG)
        _trunk_backward_one_sample(lay_G, xy_s, z[n], sens_tapes[n], [[dX[n, :S]], [dX[n, S:]]], 1, skip, gG)
    L_pde = sum_r2 / (N * P)
    L_G = float(-D_fake.mean() + pde_weight * L_pde)
    losses = np.array([L_D, D_fake.mean(), D_real.mean(), gp, L_G, L_pde], dtype=F64)
    return pack_grads(gG), pack_grads(gD), losses


def trunk_generator_loss_ref(gen_shape, disc_shape, theta_G, theta_D, xy_colloc, f, xy_sensors, z, pde_weight=1.0, skip=True):
    """L_G of the shared-trunk generator written as its plain definition (finite-difference pins only)."""
    Jc = trunk_jet_forward_ref(theta_G, *gen_shape, xy_colloc, z, 2, skip)
    _, mean_sq = darcy_residual_ref(Jc[0][:3], Jc[1], f)
    Js = trunk_jet_forward_ref(theta_G, *gen_shape, xy_sensors, z, 0, skip)
    X_fake = np.concatenate([Js[0][0], Js[1][0]], axis=1)
    return float(-disc_forward_ref(theta_D, *disc_shape, X_fake).mean() + pde_weight * mean_sq)


# ==============================================================================================================
# NEXT-2: the paper's snapshot -- "f values at random positions scattered in the domain (we call them
# free sensors) ... concatenate these values and the corresponding spatial coordinates as one fake snapshot";
# "f sensor locations are chosen randomly for each realization".  DESIGN.md reading R9:
#   X_fake[n] = [ Y(s_1..S; z_n), u(s_1..S; z_n), f(p_{n,1..F}; z_n), x(p_{n,1..F}), y(p_{n,1..F}) ]      (2S + 3F entries)
#   f(p; z) = exp(Y) (Y_x u_x + Y_y u_y + u_xx + u_yy) at p: Eq. 1 applied to the generator (the induced network);
#   L_D as before on these snapshots;  L_G = -mean_n D(X_fake[n]) + w_pde mean_{n,p} f(n,p)^2  (the paper's choice is
#   w_pde = 0: the physics reaches the generator through the critic, whose real snapshots carry the data's f, here 0).
# The two-MLP generator of BASELINE.json is kept; the coordinates carry no gradient.
# ==============================================================================================================
def free_snapshot_ref(gen_shape, theta_Y, theta_u, xy_free, xy_sensors, z):
    """X_fake [N][2S + 3F] and the per-sample jets (Yj [3][F], Uj [5][F]) at the free sensors."""
    xy_free = np.asarray(xy_free, dtype=F64); xy_s = np.asarray(xy_sensors, dtype=F64); z = np.asarray(z, dtype=F64)
    N, Fp, S = z.shape[0], xy_free.shape[1], xy_s.shape[0]
    X = np.empty((N, 2 * S + 3 * Fp), dtype=F64)
    jets = []
    for n in range(N):
        Ys = gen_jet_forward_ref(theta_Y, *gen_shape, xy_s, z[n:n + 1], 0)[0, 0]
        Us = gen_jet_forward_ref(theta_u, *gen_shape, xy_s, z[n:n + 1], 0)[0, 0]
        Yj = gen_jet_forward_ref(theta_Y, *gen_shape, xy_free[n], z[n:n + 1], 1)[:, 0]
        Uj = gen_jet_forward_ref(theta_u, *gen_shape, xy_free[n], z[n:n + 1], 2)[:, 0]
        fv = np.exp(Yj[0]) * (Yj[1] * Uj[1] + Yj[2] * Uj[2] + Uj[3] + Uj[4])
        X[n] = np.concatenate([Ys, Us, fv, xy_free[n][:, 0], xy_free[n][:, 1]])
        jets.append((Yj, Uj))
    return X, jets


def free_generator_loss_ref(gen_shape, disc_shape, theta_Y, theta_u, theta_D, xy_free, xy_sensors, z, pde_weight=0.0):
    """L_G of NEXT-2 written as its plain definition (finite-difference pins only)."""
    X, _ = free_snapshot_ref(gen_shape, theta_Y, theta_u, xy_free, xy_sensors, z)
    S, Fp = np.asarray(xy_sensors).shape[0], np.asarray(xy_free).shape[1]
    fv = X[:, 2 * S:2 * S + Fp]
    return float(-disc_forward_ref(theta_D, *disc_shape, X).mean() + pde_weight * np.mean(fv * fv))


def train_step_grads_free_ref(gen_shape, disc_shape, theta_Y, theta_u, theta_D, xy_free, xy_sensors, z, real_snap, eps,
                              gp_lambda=10.0, pde_weight=0.0):
    """Oracle of the step with f at per-sample free sensors fed to the critic.  xy_free [N][F][2]; real_snap [N][2S+3F].
    Returns g_Y, g_u, g_D (flat) and losses = [L_D, mean D(fake), mean D(real), GP, L_G, mean f^2]."""
    lay_Y = unpack_params(theta_Y, *gen_shape); lay_u = unpack_params(theta_u, *gen_shape)
    lay_D = unpack_params(theta_D, *disc_shape)
    xy_free = np.asarray(xy_free, dtype=F64); xy_s = np.asarray(xy_sensors, dtype=F64); z = np.asarray(z, dtype=F64)
    real = np.asarray(real_snap, dtype=F64); eps = np.asarray(eps, dtype=F64)
    N, Fp, S = z.shape[0], xy_free.shape[1], xy_s.shape[0]
    X_fake, _ = free_snapshot_ref(gen_shape, theta_Y, theta_u, xy_free, xy_s, z)
    gD = _zero_grads(lay_D)
    g_fake, D_fake = _disc_forward(lay_D, X_fake)
    g_real, D_real = _disc_forward(lay_D, real)
    _disc_backward(lay_D, g_fake, np.full(N, 1.0 / N), gD)
    _disc_backward(lay_D, g_real, np.full(N, -1.0 / N), gD)
    Xhat = eps[:, None] * real + (1.0 - eps[:, None]) * X_fake
    gp, _ = _gradient_penalty(lay_D, Xhat, gp_lambda, gD)
    L_D = float(D_fake.mean() - D_real.mean() + gp)
    dX = _disc_backward(lay_D, g_fake, np.full(N, -1.0 / N), None)        # dL_G/dX_fake (critic term)
    gY = _zero_grads(lay_Y); gu = _zero_grads(lay_u)
    sum_f2 = 0.0
    for n in range(N):
        Yj, tY = _jet_forward_one_sample(lay_Y, xy_free[n], z[n], 3, keep_tape=True)
        Uj, tU = _jet_forward_one_sample(lay_u, xy_free[n], z[n], 5, keep_tape=True)
        k = np.exp(Yj[0]); D = Yj[1] * Uj[1] + Yj[2] * Uj[2] + Uj[3] + Uj[4]
        fv = k * D
        sum_f2 += float((fv * fv).sum())
        r_hat = dX[n, 2 * S:2 * S + Fp] + 2.0 * pde_weight * fv / (N * Fp)      # dL_G/df(n,p): through the critic (+ the optional penalty)
        Y_hat = np.stack([r_hat * k * D, r_hat * k * Uj[1], r_hat * k * Uj[2]])   # O3 with this r_hat
        U_hat = np.stack([np.zeros_like(fv), r_hat * k * Yj[1], r_hat * k * Yj[2], r_hat * k, r_hat * k])
        _jet_backward_one_sample(lay_Y, xy_free[n], z[n], tY, Y_hat, 3, gY)
        _jet_backward_one_sample(lay_u, xy_free[n], z[n], tU, U_hat, 5, gu)
        _, tYs = _jet_forward_one_sample(lay_Y, xy_s, z[n], 1, keep_tape=True)
        _, tus = _jet_forward_one_sample(lay_u, xy_s, z[n], 1, keep_tape=True)
        _jet_backward_one_sample(lay_Y, xy_s, z[n], tYs, dX[n:n + 1, :S], 1, gY)
        _jet_backward_one_sample(lay_u, xy_s, z[n], tus, dX[n:n + 1, S:2 * S], 1, gu)
    L_f = sum_f2 / (N * Fp)
    L_G = float(-D_fake.mean() + pde_weight * L_f)
    losses = np.array([L_D, D_fake.mean(), D_real.mean(), gp, L_G, L_f], dtype=F64)
    return pack_grads(gY), pack_grads(gu), pack_grads(gD), losses


# ==============================================================================================================
# NEXT-3: hierarchical multi-discriminator loss.  "we partition the whole domain into
# subdomains and assign one discriminator for each subdomain ... each discriminator will only be in charge of all or part of
# the sensors within the assigned subdomain ... The loss of the generator is the weighted average of negative critics from
# all the discriminators ... the weight [is] 1 divided by the product of the number of levels and the number of subdomains
# in this level."  DESIGN.md reading R10:
#   critic k sees X[:, idx_k] (idx_k: d_sub columns of the 2S-entry snapshot: the log k and u entries of its sensors);
#   L_Dk = mean D_k(fake_k) - mean D_k(real_k) + lam mean (||grad D_k(xhat_k)|| - 1)^2 with the shared eps_n, gradient to theta_Dk only;
#   L_G  = sum_k w_k (-mean_n D_k(X_fake[n][idx_k])) + w_pde mean r^2,   w_k = 1 / (levels * subdomains in k's level).
# ==============================================================================================================
def hierarchy_weights(subdomains_per_level):
    """[n_1, n_2, ...] -> w_k for the critics listed level by level: 1 / (number of levels * n_level)."""
    n_levels = len(subdomains_per_level)
    return np.concatenate([np.full(n, 1.0 / (n_levels * n)) for n in subdomains_per_level])


def train_step_grads_hier_ref(gen_shape, disc_shape, theta_Y, theta_u, theta_D_list, subsets, weights, xy_colloc, f, xy_sensors, z,
                              real_snap, eps, gp_lambda=10.0, pde_weight=1.0):
    """Oracle of the step with K critics.  theta_D_list [K][n_disc]; subsets [K][d_sub] (column indices into the 2S-entry
    snapshot); weights [K].  Returns g_Y, g_u, g_D [K][n_disc] and losses = [sum_k L_Dk, sum_k w_k mean D_k(fake),
    sum_k w_k mean D_k(real), sum_k GP_k, L_G, L_pde]."""
    lay_Y = unpack_params(theta_Y, *gen_shape); lay_u = unpack_params(theta_u, *gen_shape)
    xy_c = np.asarray(xy_colloc, dtype=F64); xy_s = np.asarray(xy_sensors, dtype=F64)
    f = np.asarray(f, dtype=F64); z = np.asarray(z, dtype=F64)
    real = np.asarray(real_snap, dtype=F64); eps = np.asarray(eps, dtype=F64)
    subsets = np.asarray(subsets, dtype=np.int64); weights = np.asarray(weights, dtype=F64)
    N, P, S, K = z.shape[0], xy_c.shape[0], xy_s.shape[0], len(theta_D_list)
    X_fake = np.empty((N, 2 * S), dtype=F64)
    sens_tapes = []
    for n in range(N):
        oY, tY = _jet_forward_one_sample(lay_Y, xy_s, z[n], 1, keep_tape=True)
        ou, tu = _jet_forward_one_sample(lay_u, xy_s, z[n], 1, keep_tape=True)
        X_fake[n, :S] = oY[0]; X_fake[n, S:] = ou[0]
        sens_tapes.append((tY, tu))
    dX = np.zeros((N, 2 * S), dtype=F64)                    # dL_G/dX_fake, summed over the critics
    gD_all, sum_LD, wDf, wDr, sum_gp = [], 0.0, 0.0, 0.0, 0.0
    for k in range(K):
        lay_D = unpack_params(theta_D_list[k], *disc_shape)
        idx = subsets[k]
        Xf, Xr = X_fake[:, idx], real[:, idx]
        gD = _zero_grads(lay_D)
        g_fake, D_fake = _disc_forward(lay_D, Xf)
        g_real, D_real = _disc_forward(lay_D, Xr)
        _disc_backward(lay_D, g_fake, np.full(N, 1.0 / N), gD)
        _disc_backward(lay_D, g_real, np.full(N, -1.0 / N), gD)
        gp, _ = _gradient_penalty(lay_D, eps[:, None] * Xr + (1.0 - eps[:, None]) * Xf, gp_lambda, gD)
        gD_all.append(pack_grads(gD))
        sum_LD += float(D_fake.mean() - D_real.mean() + gp); sum_gp += gp
        wDf += weights[k] * float(D_fake.mean()); wDr += weights[k] * float(D_real.mean())
        dXk = _disc_backward(lay_D, g_fake, np.full(N, -weights[k] / N), None)     # d(-w_k mean D_k)/dX_fake[:, idx]
        np.add.at(dX, (slice(None), idx), dXk)
    gY = _zero_grads(lay_Y); gu = _zero_grads(lay_u)
    sum_r2 = 0.0
    for n in range(N):
        Yj, tY = _jet_forward_one_sample(lay_Y, xy_c, z[n], 3, keep_tape=True)
        Uj, tU = _jet_forward_one_sample(lay_u, xy_c, z[n], 5, keep_tape=True)
        r, Y_hat, U_hat = _residual_adjoints(Yj, Uj, f, pde_weight, N * P)
        sum_r2 += float((r * r).sum())
        _jet_backward_one_sample(lay_Y, xy_c, z[n], tY, Y_hat, 3, gY)
        _jet_backward_one_sample(lay_u, xy_c, z[n], tU, U_hat, 5, gu)
        tYs, tus = sens_tapes[n]
        _jet_backward_one_sample(lay_Y, xy_s, z[n], tYs, dX[n:n + 1, :S], 1, gY)
        _jet_backward_one_sample(lay_u, xy_s, z[n], tus, dX[n:n + 1, S:], 1, gu)
    L_pde = sum_r2 / (N * P)
    losses = np.array([sum_LD, wDf, wDr, sum_gp, -wDf + pde_weight * L_pde, L_pde], dtype=F64)
    return pack_grads(gY), pack_grads(gu), np.stack(gD_all), losses
