// NEXT-2 (R9): the paper's snapshot.  Every latent sample has its own F "free
// sensor" points; the induced network f = div(k grad u) is evaluated there (Eq. 1 on the generator's jets) and the critic
// sees  X[n] = [ log k(s_1..S), u(s_1..S), f(p_n,1..F), x(p_n,1..F), y(p_n,1..F) ].  The physics reaches the generator through
// dD/df (plus an optional penalty w_pde mean f^2).  Same kernels as the base step; what changes is the order: the collocation
// forward has to finish before the critic runs, and its reverse sweep starts from the critic's adjoint of f.
#include "ctx.cuh"

namespace pigan {

namespace {

template <typename T>
pigan_status free_step_impl(pigan_ctx* c, const float* thY, const float* thU, const float* thD, const float* xy_free, const float* xy_s, const float* z,
                            const float* real, const float* eps, float loss_scale, float* gY, float* gU, float* gD, float* losses, int* found_inf) {
  const pigan_config& cfg = c->cfg;
  Launcher& L = c->L;
  const NetShape& gs = c->gen; const NetShape& ds = c->disc;
  const int N = cfg.n_samples, F = cfg.n_free, S = cfg.n_sensors, d = ds.in_dim, HD = ds.H;
  const float* th[2] = {thY, thU};
  float* gr[2] = {gY, gU};
  cudaStream_t st = L.stream;
  cudaMemsetAsync(gY, 0, gs.count() * 4, st); cudaMemsetAsync(gU, 0, gs.count() * 4, st); cudaMemsetAsync(gD, 0, ds.count() * 4, st);
  cudaMemsetAsync(c->cw.acc, 0, 8 * sizeof(double), st);
  if (found_inf) cudaMemsetAsync(found_inf, 0, sizeof(int), st);
  for (int n = 0; n < 2; ++n) {
    cudaMemsetAsync(c->net[n].An, 0, (size_t)N * gs.H * 4, st);
    compute_zpart(c, n, th[n], z, N);
    if (cfg.precision != PIGAN_FP32) tc_convert_weights(L, cfg.precision, gs, th[n], c->net[n].w16);
  }
  // ---- sensor rows -> snapshot columns [0, 2S) ----
  const long long srows = (long long)N * S;
  int sc = 0;
  for (long long row0 = 0; row0 < srows; row0 += c->R_ld, ++sc) {
    ChunkGeom g = make_geom(c, row0, srows, S);
    for (int n = 0; n < 2; ++n) {
      gen_forward_chunk<T>(c, n, c->hsens(n, sc), th[n], 1, xy_s, g, c->net[n].o, c->R_ld, /*split=*/true);
      scatter_snapshot(L, c->net[n].o, row0, g.valid, S, d, n * S, c->xfake);
    }
  }
  // ---- free-sensor rows, pass 1: jets -> f = exp(Y)(Y_x u_x + Y_y u_y + u_xx + u_yy) -> snapshot columns [2S, 2S + 3F) ----
  const long long crows = (long long)N * F;
  const bool one_chunk = crows <= c->R_ld;                    // then the activations of pass 1 are still there for the reverse sweep
  for (long long row0 = 0; row0 < crows; row0 += c->R_ld) {
    ChunkGeom g = make_geom(c, row0, crows, F);
    g.per_sample = 1;
    gen_forward_chunk<T>(c, 0, c->hcol(0), thY, 3, xy_free, g, c->net[0].o, c->R_ld);
    gen_forward_chunk<T>(c, 1, c->hcol(1), thU, 5, xy_free, g, c->net[1].o, c->R_ld);
    residual(L, c->net[0].o, c->R_ld, c->net[1].o, c->R_ld, nullptr, row0, g.valid, g.R, F, c->fbuf, c->cw.acc + 3, 0.f, nullptr, nullptr, 0);
    scatter_free(L, c->fbuf, xy_free, row0, g.valid, F, d, 2 * S, c->xfake);
  }
  // ---- critic on the (2S + 3F)-entry snapshots ----
  if (critic_fused_supported(ds)) {
    critic_fused(L, ds, thD, c->xfake, real, eps, N, 1, cfg.gp_lambda, c->cw, gD, c->dX, nullptr);
  } else {
    build_snapshots(L, c->xfake, real, eps, N, d, c->cw.X);
    critic_forward(L, ds, thD, c->cw.X, 3 * N, c->cw.g, c->cw.D);
    reduce_scores(L, c->cw.D, N, c->cw.acc);
    fill_seed(L, c->seed, N);
    const int gstride = 3 * N * HD;
    critic_backward(L, ds, thD, c->cw.X, c->cw.g, 2 * N, gstride, c->seed, gD, c->dX, c->cw.t0, c->cw.t1);
    critic_gp(L, ds, thD, c->cw.X + (size_t)2 * N * d, c->cw.g + (size_t)2 * N * HD, N, gstride, cfg.gp_lambda, c->cw, gD, nullptr);
  }
  // ---- sensor rows, reverse ----
  sc = 0;
  for (long long row0 = 0; row0 < srows; row0 += c->R_ld, ++sc) {
    ChunkGeom g = make_geom(c, row0, srows, S);
    for (int n = 0; n < 2; ++n) {
      cudaMemsetAsync(c->amax + n, 0, 4, st);
      gather_seed(L, c->dX, row0, g.valid, g.R, S, d, n * S, -loss_scale, c->net[n].oh, c->amax + n);
      gen_backward_chunk<T>(c, n, c->hsens(n, sc), th[n], gr[n], 1, xy_s, g);
    }
  }
  // ---- free-sensor rows, pass 2: r_hat = -(1/N) dD/df (+ 2 w_pde f / (N F)), O3 adjoints, reverse sweep ----
  const float seed_scale = (float)(2.0 * cfg.pde_weight / (double)crows * loss_scale);
  for (long long row0 = 0; row0 < crows; row0 += c->R_ld) {
    ChunkGeom g = make_geom(c, row0, crows, F);
    g.per_sample = 1;
    if (!one_chunk) {
      gen_forward_chunk<T>(c, 0, c->hcol(0), thY, 3, xy_free, g, c->net[0].o, c->R_ld);
      gen_forward_chunk<T>(c, 1, c->hcol(1), thU, 5, xy_free, g, c->net[1].o, c->R_ld);
    }
    gather_seed(L, c->dX, row0, g.valid, g.R, F, d, 2 * S, -loss_scale, c->fbuf, nullptr);
    cudaMemsetAsync(c->amax, 0, 8, st);
    residual(L, c->net[0].o, c->R_ld, c->net[1].o, c->R_ld, nullptr, row0, g.valid, g.R, F, nullptr, nullptr, seed_scale, c->net[0].oh, c->net[1].oh,
             c->R_ld, c->amax, c->amax + 1, c->fbuf);
    gen_backward_chunk<T>(c, 0, c->hcol(0), thY, gY, 3, xy_free, g);
    gen_backward_chunk<T>(c, 1, c->hcol(1), thU, gU, 5, xy_free, g);
  }
  for (int n = 0; n < 2; ++n) {
    finalize_first_layer(L, gs, N, c->net[n].An, z, gr[n]);
    unscale_and_check(L, gr[n], gs.count(), 1.f / loss_scale, found_inf);
  }
  unscale_and_check(L, gD, ds.count(), 1.f, found_inf);
  if (losses) write_losses(L, c->cw.acc, N, crows, cfg.gp_lambda, cfg.pde_weight, losses, nullptr, nullptr, 0);
  return finish(c);
}

}  // namespace

pigan_status free_train_step(pigan_ctx* c, const float* thY, const float* thU, const float* thD, const float* xy_free, const float* xy_s, const float* z,
                             const float* real, const float* eps, float loss_scale, float* gY, float* gU, float* gD, float* losses, int* found_inf) {
  if (c->cfg.precision == PIGAN_FP32) return free_step_impl<float>(c, thY, thU, thD, xy_free, xy_s, z, real, eps, loss_scale, gY, gU, gD, losses, found_inf);
  return free_step_impl<__half>(c, thY, thU, thD, xy_free, xy_s, z, real, eps, loss_scale, gY, gU, gD, losses, found_inf);
}

}  // namespace pigan
