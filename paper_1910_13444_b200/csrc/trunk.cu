// NEXT-1 (R7, R8): one step with the paper's own generator -- ONE set of weights,
// separate log k and u outputs in the final layer, residual connections that skip intermediate layers.
//   trunk   h^l = tanh(W_l h^{l-1} + b_l) (+ h^{l-2} when skips are on and l is odd and >= 3), carried as a 5-channel jet;
//   heads   [log k, u] = W_{L+1} h^L + b_{L+1}, W_{L+1} [2][H]; log k uses channels (value, x, y), u all five.
// The hidden layers run on the same kernels as the two-MLP generator (5 channel passes instead of 8).  Layers on the skip
// chain split the fused dgrad into a plain GEMM (raw adjoint planes hhat = W^T ahat) and an elementwise kernel that adds
// the adjoint arriving over the skip, applies O4 to t^l and hands the total on to h^{l-2}; all other layers stay fused.
#include "ctx.cuh"

namespace pigan {

namespace {

inline bool takes_skip(const pigan_ctx* c, int l) { return c->skip && l >= 3 && (l & 1); }                  // h^l = t^l + h^{l-2}
inline bool feeds_skip(const pigan_ctx* c, int l) { return c->skip && l + 2 <= c->gen.L && takes_skip(c, l + 2); }

// (hi, lo) + (hi, lo) -> (hi, lo) for the split sensor forward: the sum is formed in fp32 and split again
template <typename T>
__global__ void __launch_bounds__(256) plane_add_split_kernel(int H, int R, int R_ld, const T* __restrict__ a, const T* __restrict__ b, T* __restrict__ out) {
  const int r = blockIdx.x * 256 + threadIdx.x;
  if (r >= R) return;
  const size_t plane = (size_t)H * R_ld;
  for (int j = blockIdx.y; j < H; j += gridDim.y) {
    const size_t off = (size_t)j * R_ld + r;
    const float sum = (to_f<T>(a[off]) + to_f<T>(b[off])) + (to_f<T>(a[plane + off]) + to_f<T>(b[plane + off]));
    const T hi = from_f<T>(sum);
    out[off] = hi;
    out[plane + off] = from_f<T>(sum - to_f<T>(hi));
  }
}

template <typename T>
void trunk_forward_chunk(pigan_ctx* c, const pigan_ctx::HBuf& hb, const pigan_ctx::HBuf& tb, const float* theta, int C, int C0, const float* xy,
                         const ChunkGeom& g, float* o0, float* o1, long long o_stride, bool split) {
  const NetShape& s = c->gen;
  Launcher& L = c->L;
  const int H = s.H, n = 1;
  const long long pl = (long long)H * g.R_ld;
  const bool f32 = c->cfg.precision == PIGAN_FP32;
  split = split && C == 1 && !f32;
  first_layer_fwd<T>(L, C, s, theta, c->net[n].Zp, xy, g, (T*)hb.at(1), split);
  for (int l = 2; l <= s.L; ++l) {
    char* dst = takes_skip(c, l) ? tb.at(l) : hb.at(l);
    if (f32) {
      sgemm(L, false, false, H, g.R, H, theta + s.W_off(l), H, 0, (const float*)hb.at(l - 1), g.R_ld, pl, c->net[n].apre, g.R_ld, pl, C, false);
      jet_act_fwd_f32(L, C, H, theta + s.b_off(l), g, c->net[n].apre, (float*)dst);
    } else if (split) {
      tc_layer_fwd_split(L, c->cfg.precision, H, g.R, g.R_ld, c->w16(n, l, 0), theta + s.b_off(l), hb.at(l - 1), dst);
    } else {
      tc_layer_fwd(L, c->cfg.precision, C, H, g.R, g.R_ld, c->w16(n, l, 0), theta + s.b_off(l), hb.at(l - 1), dst);
    }
    if (takes_skip(c, l)) {
      if (split) {
        dim3 grid((g.R + 255) / 256, std::min(H, 256));
        plane_add_split_kernel<T><<<grid, 256, 0, L.stream>>>(H, g.R, g.R_ld, (const T*)dst, (const T*)hb.at(l - 2), (T*)hb.at(l));
        L.check("skip_add");
      } else {
        plane_add<T>(L, C, H, g, (const T*)dst, (const T*)hb.at(l - 2), (T*)hb.at(l));
      }
    }
  }
  const float* w_out = theta + s.W_off(s.L + 1); const float* b_out = theta + s.b_off(s.L + 1);
  out_fwd<T>(L, C0, H, w_out, b_out, g, (const T*)hb.at(s.L), o0, o_stride, split);
  out_fwd<T>(L, C, H, w_out + H, b_out + 1, g, (const T*)hb.at(s.L), o1, o_stride, split);
}

// reverse sweep of one chunk; the heads' output adjoints are ohat0 [C0][R_ld] (log k) and ohat1 [C][R_ld] (u)
template <typename T>
void trunk_backward_chunk(pigan_ctx* c, const pigan_ctx::HBuf& hb, const pigan_ctx::HBuf& tb, const float* theta, float* grads, int C, const float* xy,
                          const ChunkGeom& g, const float* ohat0, const float* ohat1) {
  const NetShape& s = c->gen;
  Launcher& L = c->L;
  const int H = s.H, n = 1;
  const long long pl = (long long)H * g.R_ld;
  const bool f32 = c->cfg.precision == PIGAN_FP32;
  const float* amax = f32 ? nullptr : c->amax + 1;
  NetWs& w = c->net[n];
  auto tj = [&](int l) { return takes_skip(c, l) ? tb.at(l) : hb.at(l); };      // the tanh jet t^l that O4 is written in
  int cur = 0;
  top_act_bwd2<T>(L, C, H, g, theta + s.W_off(s.L + 1), ohat0, ohat1, (const T*)hb.at(s.L), (const T*)tj(s.L), (T*)w.ah[cur],
                  takes_skip(c, s.L) ? (T*)w.sk : nullptr, grads + s.b_off(s.L), grads + s.W_off(s.L + 1), grads + s.b_off(s.L + 1), amax);
  for (int l = s.L; l >= 2; --l) {
    const int m = l - 1;                                   // the layer whose pre-activation adjoint this iteration produces
    const bool sk_in = feeds_skip(c, m), sk_out = takes_skip(c, m);
    if (f32) sgemm(L, false, true, H, H, g.R, (const float*)w.ah[cur], g.R_ld, pl, (const float*)hb.at(m), g.R_ld, pl, grads + s.W_off(l), H, 0, C, true);
    else tc_wgrad(L, c->cfg.precision, C, H, g.R, g.R_ld, w.ah[cur], hb.at(m), grads + s.W_off(l), amax);
    if (!sk_in && !sk_out) {
      if (f32) {
        sgemm(L, true, false, H, g.R, H, theta + s.W_off(l), H, 0, (const float*)w.ah[cur], g.R_ld, pl, w.apre, g.R_ld, pl, C, false);
        jet_act_bwd_launch<T>(L, C, H, g, w.apre, nullptr, nullptr, (const T*)hb.at(m), (T*)w.ah[cur ^ 1], grads + s.b_off(m), nullptr, nullptr, amax);
      } else if (m == 1 && tc_first_layer_fusable(H, g)) {
        FirstLayerFuse fl{xy, g.row0, g.npts, s.in_dim, grads, w.An, g.per_sample};
        tc_layer_bwd(L, c->cfg.precision, C, H, g.R, g.R_ld, c->w16(n, l, 1), w.ah[cur], hb.at(m), w.ah[cur ^ 1], grads + s.b_off(m), amax, &fl);
        return;
      } else {
        tc_layer_bwd(L, c->cfg.precision, C, H, g.R, g.R_ld, c->w16(n, l, 1), w.ah[cur], hb.at(m), w.ah[cur ^ 1], grads + s.b_off(m), amax);
      }
    } else {
      // layer m sits on the skip chain: raw adjoint planes, then (+ skip adjoint) -> O4 on t^m -> ahat^m, total handed on
      const T* hh;
      if (f32) {
        sgemm(L, true, false, H, g.R, H, theta + s.W_off(l), H, 0, (const float*)w.ah[cur], g.R_ld, pl, w.apre, g.R_ld, pl, C, false);
        hh = (const T*)w.apre;
      } else {
        tc_layer_fwd(L, c->cfg.precision, C, H, g.R, g.R_ld, c->w16(n, l, 1), nullptr, w.ah[cur], w.hhb, nullptr, /*linear=*/true);
        hh = (const T*)w.hhb;
      }
      skip_adj<T>(L, C, H, g, hh, sk_in ? (const T*)w.sk : nullptr, (const T*)tj(m), (T*)w.ah[cur ^ 1], sk_out ? (T*)w.sk : nullptr,
                  grads + s.b_off(m), amax);
    }
    cur ^= 1;
  }
  first_layer_bwd<T>(L, C, s, xy, g, (const T*)w.ah[cur], grads, w.An, amax);
}

template <typename T>
pigan_status trunk_step_impl(pigan_ctx* c, const float* thG, const float* thD, const float* xy_c, const float* f, const float* xy_s, const float* z,
                             const float* real, const float* eps, float loss_scale, float* gG, float* gD, float* losses, int* found_inf) {
  const pigan_config& cfg = c->cfg;
  Launcher& L = c->L;
  const NetShape& gs = c->gen; const NetShape& ds = c->disc;
  const int N = cfg.n_samples, P = cfg.n_colloc, S = cfg.n_sensors, d = 2 * S, HD = ds.H;
  cudaStream_t st = L.stream;
  cudaMemsetAsync(gG, 0, gs.count() * 4, st); cudaMemsetAsync(gD, 0, ds.count() * 4, st);
  cudaMemsetAsync(c->cw.acc, 0, 8 * sizeof(double), st);
  if (found_inf) cudaMemsetAsync(found_inf, 0, sizeof(int), st);
  cudaMemsetAsync(c->net[1].An, 0, (size_t)N * gs.H * 4, st);
  compute_zpart(c, 1, thG, z, N);
  if (cfg.precision != PIGAN_FP32) tc_convert_weights(L, cfg.precision, gs, thG, c->net[1].w16);
  // ---- sensor rows: ONE value-channel pass gives both halves of the snapshot [log k(s_1..S), u(s_1..S)] ----
  const long long srows = (long long)N * S;
  int sc = 0;
  for (long long row0 = 0; row0 < srows; row0 += c->R_ld, ++sc) {
    ChunkGeom g = make_geom(c, row0, srows, S);
    trunk_forward_chunk<T>(c, c->hsens(1, sc), c->tsens(1, sc), thG, 1, 1, xy_s, g, c->net[0].o, c->net[1].o, c->R_ld, /*split=*/true);
    scatter_snapshot(L, c->net[0].o, row0, g.valid, S, d, 0, c->xfake);
    scatter_snapshot(L, c->net[1].o, row0, g.valid, S, d, S, c->xfake);
  }
  // ---- critic (unchanged) ----
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
  // ---- O7 on the sensor rows: both heads seed the value channel of the one trunk ----
  sc = 0;
  for (long long row0 = 0; row0 < srows; row0 += c->R_ld, ++sc) {
    ChunkGeom g = make_geom(c, row0, srows, S);
    cudaMemsetAsync(c->amax + 1, 0, 4, st);
    gather_seed(L, c->dX, row0, g.valid, g.R, S, d, 0, -loss_scale, c->net[0].oh, c->amax + 1);
    gather_seed(L, c->dX, row0, g.valid, g.R, S, d, S, -loss_scale, c->net[1].oh, c->amax + 1);
    trunk_backward_chunk<T>(c, c->hsens(1, sc), c->tsens(1, sc), thG, gG, 1, xy_s, g, c->net[0].oh, c->net[1].oh);
  }
  // ---- collocation rows: one 5-channel pass, residual, reverse sweep ----
  const long long crows = (long long)N * P;
  const float seed_scale = (float)(2.0 * cfg.pde_weight / (double)crows * loss_scale);
  for (long long row0 = 0; row0 < crows; row0 += c->R_ld) {
    ChunkGeom g = make_geom(c, row0, crows, P);
    trunk_forward_chunk<T>(c, c->hcol(1), c->tcol(1), thG, 5, 3, xy_c, g, c->net[0].o, c->net[1].o, c->R_ld, false);
    cudaMemsetAsync(c->amax + 1, 0, 4, st);
    residual(L, c->net[0].o, c->R_ld, c->net[1].o, c->R_ld, f, row0, g.valid, g.R, P, nullptr, c->cw.acc + 3, seed_scale, c->net[0].oh, c->net[1].oh,
             c->R_ld, c->amax + 1, c->amax + 1);
    trunk_backward_chunk<T>(c, c->hcol(1), c->tcol(1), thG, gG, 5, xy_c, g, c->net[0].oh, c->net[1].oh);
  }
  finalize_first_layer(L, gs, N, c->net[1].An, z, gG);
  unscale_and_check(L, gG, gs.count(), 1.f / loss_scale, found_inf);
  unscale_and_check(L, gD, ds.count(), 1.f, found_inf);
  if (losses) write_losses(L, c->cw.acc, N, crows, cfg.gp_lambda, cfg.pde_weight, losses, nullptr, nullptr, 0);
  return finish(c);
}

template <typename T>
pigan_status trunk_jet_impl(pigan_ctx* c, const float* theta, const float* xy, int n_pts, const float* z, int n_samples, int C, float* out) {
  const long long total = (long long)n_samples * n_pts;
  compute_zpart(c, 1, theta, z, n_samples);
  if (c->cfg.precision != PIGAN_FP32) tc_convert_weights(c->L, c->cfg.precision, c->gen, theta, c->net[1].w16);
  for (long long row0 = 0; row0 < total; row0 += c->R_ld) {
    ChunkGeom g = make_geom(c, row0, total, n_pts);
    trunk_forward_chunk<T>(c, c->hcol(1), c->tcol(1), theta, C, C, xy, g, out + row0, out + (size_t)C * total + row0, total, /*split=*/C == 1);
  }
  return finish(c);
}

}  // namespace

pigan_status trunk_train_step(pigan_ctx* c, const float* thG, const float* thD, const float* xy_c, const float* f, const float* xy_s, const float* z,
                              const float* real, const float* eps, float loss_scale, float* gG, float* gD, float* losses, int* found_inf) {
  if (c->cfg.precision == PIGAN_FP32) return trunk_step_impl<float>(c, thG, thD, xy_c, f, xy_s, z, real, eps, loss_scale, gG, gD, losses, found_inf);
  return trunk_step_impl<__half>(c, thG, thD, xy_c, f, xy_s, z, real, eps, loss_scale, gG, gD, losses, found_inf);
}

pigan_status trunk_jet_forward(pigan_ctx* c, const float* theta, const float* xy, int n_pts, const float* z, int n_samples, int C, float* out) {
  if (c->cfg.precision == PIGAN_FP32) return trunk_jet_impl<float>(c, theta, xy, n_pts, z, n_samples, C, out);
  return trunk_jet_impl<__half>(c, theta, xy, n_pts, z, n_samples, C, out);
}

}  // namespace pigan
