// C-ABI entry points (include/pigan.h) and the host-side orchestration of one step: row-chunking of the N*P
// collocation rows and N*S sensor rows, kernel sequencing on one stream, fp32 accumulation
// of weight gradients across chunks.  Every step of the path runs in this library's kernels; there is no CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "ctx.cuh"

using namespace pigan;

namespace {


template <typename T>
pigan_status jet_forward_impl(pigan_ctx* c, const float* theta, const float* xy, int n_pts, const float* z, int n_samples, int C, float* out) {
  const long long total = (long long)n_samples * n_pts;
  const int n = 1;
  compute_zpart(c, n, theta, z, n_samples);
  if (c->cfg.precision != PIGAN_FP32) tc_convert_weights(c->L, c->cfg.precision, c->gen, theta, c->net[n].w16);
  for (long long row0 = 0; row0 < total; row0 += c->R_ld) {
    ChunkGeom g = make_geom(c, row0, total, n_pts);
    gen_forward_chunk<T>(c, n, c->hcol(n), theta, C, xy, g, out + row0, total, /*split=*/C == 1, /*keep_last=*/false);
  }
  return finish(c);
}

template <typename T>
pigan_status train_step_impl(pigan_ctx* c, const float* thY, const float* thU, const float* thD, const float* xy_c, const float* f,
                             const float* xy_s, const float* z, const float* real, const float* eps, float loss_scale, float* gY,
                             float* gU, float* gD, float* losses, int* found_inf) {
  const pigan_config& cfg = c->cfg;
  Launcher& L = c->L;
  const NetShape& gs = c->gen; const NetShape& ds = c->disc;
  const int N = cfg.n_samples, P = cfg.n_colloc, S = cfg.n_sensors, d = 2 * S, HD = ds.H;
  const float* th[2] = {thY, thU};
  float* gr[2] = {gY, gU};
  cudaStream_t st = L.stream;
  const size_t n_gD = ds.count() * (size_t)std::max(1, c->hier.K);
  const long long srows = (long long)N * S, crows = (long long)N * P;
  // Streams.  The critic stage needs X_fake only and the forward of the collocation rows nothing of the critic's: the critic goes
  // to a side stream beside the forward of the first collocation chunk.  The two generator nets are independent up to the
  // residual: at widths <= 256 (c1 - c3: short kernels, launch chains) net 1's kernels go to a second side stream (measured
  // on B200: c2 step 0.81 -> 0.75 ms, c3 9.3 -> 9.1 ms; at width 512 the two nets' kernels only evict each other's planes from L2).
  // Per-launch profiling keeps everything on the caller's stream (its events time consecutive launches).
  const bool fork = c->side != nullptr && !L.profiling;
  const bool two = fork && c->side2 != nullptr && gs.H <= 256;
  cudaStream_t sn[2] = {st, two ? c->side2 : st};
  int evk = 0;
  auto link = [&](cudaStream_t from, cudaStream_t to) {      // work enqueued on `to` from here on follows what `from` holds now
    if (from == to) return;
    cudaEvent_t e = c->ev_pool[evk++ & 7];
    cudaEventRecord(e, from); cudaStreamWaitEvent(to, e, 0);
  };
  cudaMemsetAsync(gY, 0, gs.count() * 4, st); cudaMemsetAsync(gU, 0, gs.count() * 4, st); cudaMemsetAsync(gD, 0, n_gD * 4, st);
  cudaMemsetAsync(c->cw.acc, 0, 8 * sizeof(double), st);
  if (found_inf) cudaMemsetAsync(found_inf, 0, sizeof(int), st);
  link(st, sn[1]);
  // ---- a1 + a6: z-part, 16-bit weights, sensor evaluation -> X_fake; the (hi) activation planes of every sensor chunk stay in
  //      net[n].hs for the reverse sweep ----
  for (int n = 0; n < 2; ++n) {
    L.stream = sn[n];
    cudaMemsetAsync(c->net[n].An, 0, (size_t)N * gs.H * 4, sn[n]);
    compute_zpart(c, n, th[n], z, N);
    if (cfg.precision != PIGAN_FP32) tc_convert_weights(L, cfg.precision, gs, th[n], c->net[n].w16);
    int sc = 0;
    for (long long row0 = 0; row0 < srows; row0 += c->R_ld, ++sc) {
      NvtxRange nr("pigan:sensor_forward");
      ChunkGeom g = make_geom(c, row0, srows, S);
      gen_forward_chunk<T>(c, n, c->hsens(n, sc), th[n], 1, xy_s, g, c->net[n].o, c->R_ld, /*split=*/true);
      scatter_snapshot(L, c->net[n].o, row0, g.valid, S, d, n * S, c->xfake);
    }
  }
  L.stream = st;
  link(sn[1], st);                                           // X_fake is complete
  // ---- a7-a9: critic losses and gradient; dX rows [0, N) = (1/N) grad_X D(X_fake) ----
  if (fork) { link(st, c->side); L.stream = c->side; }
  nvtxRangePushA("pigan:critic");
  if (c->hier.K > 0) {
    hier_critic_stage(c, thD, real, eps, gD);               // NEXT-3: K critics on column subsets (hier.cu)
  } else if (critic_fused_supported(ds)) {
    // small critic: one kernel for every per-row sweep + the batched weight-gradient GEMMs (critic_fused.cu)
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
  nvtxRangePop();
  // ---- O7 + a10 on the sensor rows: dL_G/dX_fake = -(1/N) grad_X D(X_fake), value channel only ----
  // With their own adjoint set the sensor rows' reverse sweep follows the critic on ITS stream, beside the whole collocation pass.
  const bool sb = two && c->amax_s != nullptr;
  auto sensor_backward = [&](int n, bool own) {
    int sc = 0;
    for (long long row0 = 0; row0 < srows; row0 += c->R_ld, ++sc) {
      NvtxRange nr("pigan:sensor_backward");
      ChunkGeom g = make_geom(c, row0, srows, S);
      float* am = (own ? c->amax_s : c->amax) + n;
      cudaMemsetAsync(am, 0, 4, L.stream);
      gather_seed(L, c->dX, row0, g.valid, g.R, S, d, n * S, -loss_scale, own ? c->net[n].oh_s : c->net[n].oh, am);
      gen_backward_chunk<T>(c, n, c->hsens(n, sc), th[n], gr[n], 1, xy_s, g, own);
    }
  };
  if (sb) {                                                  // net 0 behind the critic on its stream, net 1 beside it on a stream of its own
    link(c->side, c->side3);
    sensor_backward(0, true);
    L.stream = c->side3;
    sensor_backward(1, true);
  }
  L.stream = st;
  const float* thn[2] = {thY, thU};
  const int Cn[2] = {3, 5};
  if (fork) {                                                // forward of the first collocation chunk beside the critic
    NvtxRange nr("pigan:collocation_forward_0");
    ChunkGeom g = make_geom(c, 0, crows, P);
    for (int n = 0; n < 2; ++n) {
      L.stream = sn[n];
      gen_forward_chunk<T>(c, n, c->hcol(n), thn[n], Cn[n], xy_c, g, c->net[n].o, c->R_ld);
    }
    L.stream = st;
    if (!sb) link(c->side, st);                              // the critic's dX
  }
  if (!sb) {
    link(st, sn[1]);
    for (int n = 0; n < 2; ++n) { L.stream = sn[n]; sensor_backward(n, false); }
    L.stream = st;
  }
  // ---- a1-a5, a10 on the collocation rows ----
  const float seed_scale = (float)(2.0 * cfg.pde_weight / (double)crows * loss_scale);
  for (long long row0 = 0; row0 < crows; row0 += c->R_ld) {
    NvtxRange nr("pigan:collocation_chunk");
    ChunkGeom g = make_geom(c, row0, crows, P);
    if (!(fork && row0 == 0)) {                              // the first chunk's forward ran beside the critic
      for (int n = 0; n < 2; ++n) {
        L.stream = sn[n];
        gen_forward_chunk<T>(c, n, c->hcol(n), thn[n], Cn[n], xy_c, g, c->net[n].o, c->R_ld);
      }
      L.stream = st;
    }
    link(sn[1], st);                                         // the residual needs both nets' outputs (and amax[1] is net 1's until here)
    cudaMemsetAsync(c->amax, 0, 8, st);
    residual(L, c->net[0].o, c->R_ld, c->net[1].o, c->R_ld, f, row0, g.valid, g.R, P, nullptr, c->cw.acc + 3, seed_scale, c->net[0].oh,
             c->net[1].oh, c->R_ld, c->amax, c->amax + 1);
    link(st, sn[1]);
    for (int n = 0; n < 2; ++n) {
      L.stream = sn[n];
      gen_backward_chunk<T>(c, n, c->hcol(n), thn[n], gr[n], Cn[n], xy_c, g);
    }
    L.stream = st;
  }
  // ---- finalize: z-part of the first layer, unscale, inf/nan flag, loss scalars ----
  if (sb) { link(c->side, st); link(c->side3, sn[1]); link(c->side3, st); }       // the critic's gradient and the sensor rows' (net 0: side, net 1: side3)
  for (int n = 0; n < 2; ++n) {
    L.stream = sn[n];
    finalize_first_layer(L, gs, N, c->net[n].An, z, gr[n]);
    unscale_and_check(L, gr[n], gs.count(), 1.f / loss_scale, found_inf);
  }
  L.stream = st;
  link(sn[1], st);
  unscale_and_check(L, gD, n_gD, 1.f, found_inf);
  if (losses) {
    if (c->hier.K > 0) hier_write_losses(c, crows, losses);
    else write_losses(L, c->cw.acc, N, crows, cfg.gp_lambda, cfg.pde_weight, losses, nullptr, nullptr, 0);
  }
  return finish(c);
}

bool shape_ok(const pigan_mlp_shape& s) { return s.in_dim >= 1 && s.n_hidden >= 1 && s.width >= 1; }

}  // namespace

// =================================================================================================================
extern "C" {

size_t pigan_param_count(const pigan_mlp_shape* s) {
  if (!s || !shape_ok(*s)) return 0;
  NetShape n{s->in_dim, s->n_hidden, s->width};
  return n.count();
}

size_t pigan_trunk_param_count(const pigan_mlp_shape* s) {
  if (!s || !shape_ok(*s)) return 0;
  NetShape n{s->in_dim, s->n_hidden, s->width};
  n.heads = 2;
  return n.count();
}

const char* pigan_last_error(const pigan_ctx* c) { return c ? c->err.c_str() : "null context"; }
unsigned long long pigan_launch_count(const pigan_ctx* c) { return c ? c->L.count : 0; }

pigan_status pigan_profile_enable(pigan_ctx* c, int enable) {
  if (!c) return PIGAN_ERR_INVALID_ARG;
  DeviceGuard dg(c);
  c->L.profiling = enable != 0;
  if (enable) { c->L.n_rec = 0; c->L.mark("begin"); }
  return PIGAN_OK;
}

pigan_status pigan_profile_report(pigan_ctx* c, char* buf, size_t cap) {
  if (!c || !buf || cap == 0) return PIGAN_ERR_INVALID_ARG;
  DeviceGuard dg(c);
  if (c->L.n_rec == 0) return fail(c, PIGAN_ERR_INVALID_ARG, "profiling was not enabled");
  if (cudaStreamSynchronize(c->L.stream) != cudaSuccess) return fail(c, PIGAN_ERR_CUDA, "stream synchronize failed");
  std::vector<std::pair<std::string, std::pair<unsigned long long, double>>> acc;
  for (size_t i = 1; i < c->L.n_rec; ++i) {
    float ms = 0.f;
    cudaEventElapsedTime(&ms, c->L.events[i - 1], c->L.events[i]);
    const std::string name = c->L.names[i];
    size_t k = 0;
    for (; k < acc.size(); ++k) if (acc[k].first == name) break;
    if (k == acc.size()) acc.push_back({name, {0ull, 0.0}});
    acc[k].second.first += 1; acc[k].second.second += ms;
  }
  std::string js = "{";
  for (size_t k = 0; k < acc.size(); ++k) {
    char tmp[160];
    snprintf(tmp, sizeof tmp, "%s\"%s\": [%llu, %.6f]", k ? ", " : "", acc[k].first.c_str(), acc[k].second.first, acc[k].second.second);
    js += tmp;
  }
  js += "}";
  snprintf(buf, cap, "%s", js.c_str());
  c->L.n_rec = 0;
  if (c->L.profiling) c->L.mark("begin");
  return PIGAN_OK;
}

pigan_status pigan_create(const pigan_config* cfg, void* cuda_stream, pigan_ctx** out) {
  if (out) *out = nullptr;
  if (!cfg || !out) return PIGAN_ERR_INVALID_ARG;
  if (!shape_ok(cfg->gen) || !shape_ok(cfg->disc) || cfg->latent_dim < 1 || cfg->n_samples < 1 || cfg->n_colloc < 1 || cfg->n_sensors < 1)
    return PIGAN_ERR_INVALID_ARG;
  if ((int)cfg->precision < 0 || (int)cfg->precision > 2 || !(cfg->gp_lambda >= 0.f) || cfg->chunk_rows < 0) return PIGAN_ERR_INVALID_ARG;
  if (cfg->gen_variant < 0 || cfg->gen_variant > 2) return PIGAN_ERR_INVALID_ARG;
  if (cfg->n_free < 0 || cfg->n_critics < 0) return PIGAN_ERR_INVALID_ARG;
  if (cfg->gen.in_dim != 2 + cfg->latent_dim) return PIGAN_ERR_SHAPE;
  if (cfg->n_critics == 0 && cfg->disc.in_dim != 2 * cfg->n_sensors + 3 * cfg->n_free) return PIGAN_ERR_SHAPE;
  if (cfg->n_critics > 0 && (cfg->disc.in_dim > 2 * cfg->n_sensors)) return PIGAN_ERR_SHAPE;
  if (cfg->n_critics > 0 && (cfg->n_free > 0 || cfg->gen_variant != PIGAN_GEN_TWO_MLPS)) return PIGAN_ERR_UNSUPPORTED;
  if (cfg->n_free > 0 && cfg->n_colloc != cfg->n_free) return PIGAN_ERR_SHAPE;
  if (cfg->n_free > 0 && cfg->gen_variant != PIGAN_GEN_TWO_MLPS) return PIGAN_ERR_UNSUPPORTED;
  if (cfg->precision == PIGAN_BF16) return PIGAN_ERR_UNSUPPORTED;     // no bf16 datapath (pigan.h); never an alias of another arithmetic
  if (cfg->precision != PIGAN_FP32) {
    std::string why;
    if (!tc_supported(cfg->gen.width, &why)) return PIGAN_ERR_UNSUPPORTED;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return PIGAN_ERR_CUDA; }
  pigan_ctx* c = new (std::nothrow) pigan_ctx();
  if (!c) return PIGAN_ERR_ALLOC;
  c->cfg = *cfg;
  c->gen = NetShape{cfg->gen.in_dim, cfg->gen.n_hidden, cfg->gen.width};
  c->trunk = cfg->gen_variant != PIGAN_GEN_TWO_MLPS;
  c->skip = cfg->gen_variant == PIGAN_GEN_TRUNK_SKIP;
  if (c->trunk) c->gen.heads = 2;
  c->disc = NetShape{cfg->disc.in_dim, cfg->disc.n_hidden, cfg->disc.width};
  c->L.stream = (cudaStream_t)cuda_stream;
  cudaGetDevice(&c->L.device);
  if (cudaDeviceGetAttribute(&c->L.num_sms, cudaDevAttrMultiProcessorCount, c->L.device) != cudaSuccess || c->L.num_sms <= 0) c->L.num_sms = 148;
  {
    bool ok = cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking) == cudaSuccess && cudaStreamCreateWithFlags(&c->side2, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&c->side3, cudaStreamNonBlocking) == cudaSuccess;
    for (int i = 0; ok && i < 8; ++i) ok = cudaEventCreateWithFlags(&c->ev_pool[i], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) {                                               // no side streams: every stage stays on the caller's stream
      cudaGetLastError();
      if (c->side) cudaStreamDestroy(c->side);
      if (c->side2) cudaStreamDestroy(c->side2);
      if (c->side3) cudaStreamDestroy(c->side3);
      c->side = c->side2 = c->side3 = nullptr;
    }
  }
  c->L.one_cta = (cfg->flags & PIGAN_FLAG_ONE_CTA) != 0;
  c->sg.disabled = (cfg->flags & PIGAN_FLAG_NO_GRAPH) != 0;
  c->elem = cfg->precision == PIGAN_FP32 ? 4 : 2;
  const int H = c->gen.H, Lh = c->gen.L, N = cfg->n_samples, S = cfg->n_sensors, d = c->disc.in_dim, HD = c->disc.H, LD = c->disc.L;
  const bool f32 = cfg->precision == PIGAN_FP32;
  // bytes per chunk row over both nets: h (L*C) + adjoint ping-pong (2C) planes [+ fp32 scratch]
  size_t per_row = 0;
  for (int C : {3, 5}) per_row += ((size_t)Lh * C + 2 * C) * H * c->elem + (f32 ? (size_t)C * H * 4 : 0) + 2 * C * 4;
  if (c->skip) per_row += ((size_t)Lh * 5 + 2 * 5) * H * c->elem;           // tanh-jet stash, skip adjoint, raw adjoint planes (net[1])
  // the sensor rows' stash hs (both nets: L x (hi, lo) planes per sensor chunk, kept from the snapshot forward to the reverse sweep;
  // + the tanh-jet stash hts with skips) holds ceil(N S / rows) chunks of `rows` rows: at most (N S + rows) rows' worth
  const size_t sens_row = (size_t)(2 + (c->skip ? 1 : 0)) * Lh * 2 * H * c->elem;
  per_row += sens_row;
  // the sensor rows' own adjoint set at widths <= 256 (value channel: two planes, output adjoint, fp32 scratch), both nets
  if (H <= 256 && !c->trunk && cfg->n_free == 0) per_row += 2 * ((size_t)2 * H * c->elem + 4 + (f32 ? (size_t)H * 4 : 0));
  const long long max_rows = std::max<long long>((long long)N * cfg->n_colloc, (long long)N * S);
  size_t free_b = 0, total_b = 0;
  cudaMemGetInfo(&free_b, &total_b);
  size_t budget = cfg->workspace_bytes ? cfg->workspace_bytes : std::min<size_t>(free_b / 2, (size_t)48 << 30);
  const size_t sens_fixed = (size_t)N * S * sens_row;
  long long rows = budget > sens_fixed ? (long long)((budget - sens_fixed) / per_row) : 0;
  long long cap = 131072;                                  // default chunk rows (sweep on B200: larger chunks amortise launch ramps)
  if (cfg->chunk_rows > 0) cap = std::max(256, cfg->chunk_rows);
  if (!cfg->workspace_bytes) rows = std::min(rows, cap);
  rows = std::min<long long>(rows, (long long)round_up((size_t)max_rows, 256));
  rows = std::max<long long>(rows / 256 * 256, 256);            // workspace_bytes is a hint: never below one 256-row chunk
  c->R_ld = (int)rows;
  c->n_sens_chunks = (int)(((long long)N * S + c->R_ld - 1) / c->R_ld);
  try {
    for (int n = 0; n < 2; ++n) {
      NetWs& w = c->net[n];
      w.Cmax = n == 0 ? 3 : 5;
      const size_t pl = c->plane();
      w.h = c->alloc<char>((size_t)Lh * w.Cmax * pl);
      w.hs = c->alloc<char>((size_t)c->n_sens_chunks * Lh * 2 * pl);
      if (c->skip && n == 1) {
        w.ht = c->alloc<char>((size_t)Lh * w.Cmax * pl);
        w.hts = c->alloc<char>((size_t)c->n_sens_chunks * Lh * 2 * pl);
        w.sk = c->alloc<char>((size_t)w.Cmax * pl);
        w.hhb = c->alloc<char>((size_t)w.Cmax * pl);
      }
      w.ah[0] = c->alloc<char>((size_t)w.Cmax * pl);
      w.ah[1] = c->alloc<char>((size_t)w.Cmax * pl);
      if (f32) w.apre = c->alloc<float>((size_t)w.Cmax * H * c->R_ld);
      w.o = c->alloc<float>((size_t)w.Cmax * c->R_ld);
      w.oh = c->alloc<float>((size_t)w.Cmax * c->R_ld);
      w.Zp = c->alloc<float>((size_t)N * H);
      w.An = c->alloc<float>((size_t)N * H);
      if (!f32) w.w16 = c->alloc<char>((size_t)std::max(Lh - 1, 1) * 2 * H * H * 2);
    }
    const size_t wmax = (size_t)std::max(d, HD);
    CriticWs& cw = c->cw;
    cw.maxB = N;
    cw.X = c->alloc<float>((size_t)3 * N * d);
    cw.g = c->alloc<float>((size_t)LD * 3 * N * HD);
    cw.D = c->alloc<float>((size_t)3 * N);
    cw.t0 = c->alloc<float>((size_t)3 * N * wmax);
    cw.t1 = c->alloc<float>((size_t)3 * N * wmax);
    cw.t2 = c->alloc<float>((size_t)3 * N * wmax);
    cw.gbar = c->alloc<float>((size_t)(LD + 1) * N * wmax);
    cw.abar = c->alloc<float>((size_t)LD * N * HD);
    cw.adjs = c->alloc<float>((size_t)LD * N * HD);
    cw.nu = c->alloc<float>((size_t)N);
    cw.acc = c->alloc<double>(8);
    if (critic_fused_supported(c->disc)) {
      cw.cfA = c->alloc<float>((size_t)LD * 4 * N * HD);
      cw.cfB1 = c->alloc<float>((size_t)4 * N * d);
      cw.cfBh = c->alloc<float>((size_t)LD * 4 * N * HD);
    }
    const int dsnap = cfg->n_critics > 0 ? 2 * S : d;         // width of the generated snapshot
    c->xfake = c->alloc<float>((size_t)N * dsnap);
    c->dX = c->alloc<float>((size_t)2 * N * dsnap);
    if (cfg->n_critics > 0) {
      c->hXf = c->alloc<float>((size_t)N * d); c->hXr = c->alloc<float>((size_t)N * d); c->hdX = c->alloc<float>((size_t)2 * N * d);
      c->htot = c->alloc<double>(4);
    }
    c->seed = c->alloc<float>((size_t)2 * N);
    c->amax = c->alloc<float>(2);
    if (H <= 256 && !c->trunk && cfg->n_free == 0) {          // widths that run the two nets and the critic on three streams (api.cu)
      c->amax_s = c->alloc<float>(2);
      for (int n = 0; n < 2; ++n) {
        NetWs& w = c->net[n];
        w.ah_s[0] = c->alloc<char>(c->plane()); w.ah_s[1] = c->alloc<char>(c->plane());
        w.oh_s = c->alloc<float>((size_t)c->R_ld);
        if (f32) w.apre_s = c->alloc<float>((size_t)H * c->R_ld);
      }
    }
    if (cfg->n_free > 0) c->fbuf = c->alloc<float>((size_t)c->R_ld);
  } catch (const std::bad_alloc&) {
    pigan_destroy(c);
    return PIGAN_ERR_ALLOC;
  }
  *out = c;
  return PIGAN_OK;
}

void pigan_destroy(pigan_ctx* c) {
  if (!c) return;
  DeviceGuard dg(c);
  for (auto& e : c->sg.entries) if (e.exec) cudaGraphExecDestroy(e.exec);
  if (c->sg.cap_stream) cudaStreamDestroy(c->sg.cap_stream);
  if (c->side) cudaStreamDestroy(c->side);
  if (c->side2) cudaStreamDestroy(c->side2);
  if (c->side3) cudaStreamDestroy(c->side3);
  for (cudaEvent_t e : c->ev_pool) if (e) cudaEventDestroy(e);
  for (void* p : c->allocs) cudaFree(p);
  for (cudaEvent_t e : c->L.events) cudaEventDestroy(e);
  delete c;
}

pigan_status pigan_gen_jet_forward(pigan_ctx* c, const float* gen_params, const float* xy, int n_pts, const float* z, int n_samples,
                                   int jet_order, float* out) {
  if (!c) return PIGAN_ERR_INVALID_ARG;
  DeviceGuard dg(c);
  if (jet_order < 0 || jet_order > 2 || n_pts < 0 || n_samples < 0) return fail(c, PIGAN_ERR_INVALID_ARG, "jet_order must be 0..2 and sizes >= 0");
  if (c->trunk) return fail(c, PIGAN_ERR_UNSUPPORTED, "this context holds the shared-trunk generator: call pigan_trunk_jet_forward");
  if (n_pts == 0 || n_samples == 0) return PIGAN_OK;
  if (!gen_params || !xy || !z || !out) return fail(c, PIGAN_ERR_INVALID_ARG, "null pointer");
  if (n_samples > c->cfg.n_samples) return fail(c, PIGAN_ERR_SHAPE, "n_samples exceeds the n_samples of the config");
  const int C = jet_order == 0 ? 1 : jet_order == 1 ? 3 : 5;
  switch (c->cfg.precision) {
    case PIGAN_FP32: return jet_forward_impl<float>(c, gen_params, xy, n_pts, z, n_samples, C, out);
    default: return jet_forward_impl<__half>(c, gen_params, xy, n_pts, z, n_samples, C, out);
  }
}

pigan_status pigan_trunk_jet_forward(pigan_ctx* c, const float* trunk_params, const float* xy, int n_pts, const float* z, int n_samples,
                                     int jet_order, float* out) {
  if (!c) return PIGAN_ERR_INVALID_ARG;
  DeviceGuard dg(c);
  if (jet_order < 0 || jet_order > 2 || n_pts < 0 || n_samples < 0) return fail(c, PIGAN_ERR_INVALID_ARG, "jet_order must be 0..2 and sizes >= 0");
  if (!c->trunk) return fail(c, PIGAN_ERR_UNSUPPORTED, "this context holds the two-MLP generator: call pigan_gen_jet_forward");
  if (n_pts == 0 || n_samples == 0) return PIGAN_OK;
  if (!trunk_params || !xy || !z || !out) return fail(c, PIGAN_ERR_INVALID_ARG, "null pointer");
  if (n_samples > c->cfg.n_samples) return fail(c, PIGAN_ERR_SHAPE, "n_samples exceeds the n_samples of the config");
  return trunk_jet_forward(c, trunk_params, xy, n_pts, z, n_samples, jet_order == 0 ? 1 : jet_order == 1 ? 3 : 5, out);
}

pigan_status pigan_darcy_residual(pigan_ctx* c, const float* logk_jet, const float* u_jet, const float* f, int n_samples, int n_pts,
                                  float* r, float* mean_sq) {
  if (!c) return PIGAN_ERR_INVALID_ARG;
  DeviceGuard dg(c);
  if (n_samples < 0 || n_pts < 0) return fail(c, PIGAN_ERR_INVALID_ARG, "negative size");
  const long long total = (long long)n_samples * n_pts;
  if (total > 0 && (!logk_jet || !u_jet || !f)) return fail(c, PIGAN_ERR_INVALID_ARG, "null pointer");
  cudaMemsetAsync(c->cw.acc, 0, 8 * sizeof(double), c->L.stream);
  for (long long row0 = 0; row0 < total; row0 += (1 << 30)) {
    const int rows = (int)std::min<long long>(1 << 30, total - row0);
    residual(c->L, logk_jet + row0, total, u_jet + row0, total, f, row0, rows, rows, n_pts, r ? r + row0 : nullptr, mean_sq ? c->cw.acc + 3 : nullptr,
             0.f, nullptr, nullptr, 0);
  }
  if (mean_sq) write_losses(c->L, c->cw.acc, 1, 1, 0.f, 0.f, nullptr, nullptr, mean_sq, total);
  return finish(c);
}

pigan_status pigan_disc_forward(pigan_ctx* c, const float* disc_params, const float* snap, int B, float* score) {
  if (!c) return PIGAN_ERR_INVALID_ARG;
  DeviceGuard dg(c);
  if (B < 0) return fail(c, PIGAN_ERR_INVALID_ARG, "negative batch");
  if (B == 0) return PIGAN_OK;
  if (!disc_params || !snap || !score) return fail(c, PIGAN_ERR_INVALID_ARG, "null pointer");
  const int d = c->disc.in_dim, cap = 3 * c->cfg.n_samples;
  for (int b0 = 0; b0 < B; b0 += cap) {
    const int rows = std::min(cap, B - b0);
    critic_forward(c->L, c->disc, disc_params, snap + (size_t)b0 * d, rows, c->cw.g, score + b0);
  }
  return finish(c);
}

pigan_status pigan_gradient_penalty(pigan_ctx* c, const float* disc_params, const float* real, const float* fake, const float* eps, int B,
                                    float* gp, float* grad_norm, float* d_disc_params) {
  if (!c) return PIGAN_ERR_INVALID_ARG;
  DeviceGuard dg(c);
  if (B < 1) return fail(c, PIGAN_ERR_INVALID_ARG, "B must be >= 1");
  if (!disc_params || !real || !fake || !eps) return fail(c, PIGAN_ERR_INVALID_ARG, "null pointer");
  if (B > c->cfg.n_samples) return fail(c, PIGAN_ERR_SHAPE, "B exceeds the n_samples of the config");
  const NetShape& ds = c->disc;
  const int d = ds.in_dim, HD = ds.H;
  cudaStream_t st = c->L.stream;
  cudaMemsetAsync(c->cw.acc, 0, 8 * sizeof(double), st);
  if (d_disc_params) cudaMemsetAsync(d_disc_params, 0, ds.count() * 4, st);
  if (critic_fused_supported(ds)) {
    critic_fused(c->L, ds, disc_params, fake, real, eps, B, 0, c->cfg.gp_lambda, c->cw, d_disc_params, nullptr, grad_norm);
  } else {
    build_snapshots(c->L, fake, real, eps, B, d, c->cw.X);
    float* Xhat = c->cw.X + (size_t)2 * B * d;
    critic_forward(c->L, ds, disc_params, Xhat, B, c->cw.g, c->cw.D);
    critic_gp(c->L, ds, disc_params, Xhat, c->cw.g, B, B * HD, c->cfg.gp_lambda, c->cw, d_disc_params, grad_norm);
  }
  if (gp) write_losses(c->L, c->cw.acc, B, 1, c->cfg.gp_lambda, 0.f, nullptr, gp, nullptr, 0);
  return finish(c);
}

pigan_status pigan_train_step_grads(pigan_ctx* c, const float* logk_params, const float* u_params, const float* disc_params,
                                    const float* xy_colloc, const float* f, const float* xy_sensors, const float* z, const float* real_snap,
                                    const float* eps, float loss_scale, float* g_logk, float* g_u, float* g_disc, float* losses, int* found_inf) {
  if (!c) return PIGAN_ERR_INVALID_ARG;
  DeviceGuard dg(c);
  if (!logk_params || !disc_params || !xy_colloc || (!f && c->cfg.n_free == 0) || !xy_sensors || !z || !real_snap || !eps || !g_logk || !g_disc ||
      (!c->trunk && (!u_params || !g_u)))
    return fail(c, PIGAN_ERR_INVALID_ARG, "null pointer");
  if (!(loss_scale > 0.f) || !std::isfinite(loss_scale)) return fail(c, PIGAN_ERR_INVALID_ARG, "loss_scale must be positive and finite");
  if (c->cfg.n_critics > 0) return fail(c, PIGAN_ERR_UNSUPPORTED, "the context was created with n_critics > 0: call pigan_train_step_grads_hier");
  auto run = [&]() -> pigan_status {
    if (c->cfg.n_free > 0)
      return free_train_step(c, logk_params, u_params, disc_params, xy_colloc, xy_sensors, z, real_snap, eps, loss_scale, g_logk, g_u, g_disc, losses, found_inf);
    if (c->trunk)
      return trunk_train_step(c, logk_params, disc_params, xy_colloc, f, xy_sensors, z, real_snap, eps, loss_scale, g_logk, g_disc, losses, found_inf);
    switch (c->cfg.precision) {
      case PIGAN_FP32: return train_step_impl<float>(c, logk_params, u_params, disc_params, xy_colloc, f, xy_sensors, z, real_snap, eps, loss_scale, g_logk, g_u, g_disc, losses, found_inf);
      default: return train_step_impl<__half>(c, logk_params, u_params, disc_params, xy_colloc, f, xy_sensors, z, real_snap, eps, loss_scale, g_logk, g_u, g_disc, losses, found_inf);
    }
  };
  auto& sg = c->sg;
  if (sg.disabled || c->L.profiling) return run();
  unsigned int ls_bits; memcpy(&ls_bits, &loss_scale, 4);
  const void* ptrs[] = {logk_params, u_params, disc_params, xy_colloc, f, xy_sensors, z, real_snap, eps, g_logk, g_u, g_disc, losses, found_inf};
  std::vector<unsigned long long> key;
  for (const void* q : ptrs) key.push_back((unsigned long long)(uintptr_t)q);
  key.push_back(ls_bits);
  using Entry = pigan_ctx::StepGraph::Entry;
  Entry* ent = nullptr;
  for (Entry& e : sg.entries) if (e.key == key) { ent = &e; break; }
  ++sg.tick;
  if (ent && ent->exec) {                                    // replay
    ent->last_use = sg.tick;
    if (cudaGraphLaunch(ent->exec, c->L.stream) != cudaSuccess) { cudaGetLastError(); return fail(c, PIGAN_ERR_CUDA, "cudaGraphLaunch failed"); }
    c->L.count += ent->launches;
    return PIGAN_OK;
  }
  if (!ent) {                                                // first sight of these arguments: run eagerly (also sets kernel attributes)
    if ((int)sg.entries.size() == pigan_ctx::StepGraph::kMaxGraphs) {      // forget the least recently used argument set
      size_t lru = 0;
      for (size_t k = 1; k < sg.entries.size(); ++k) if (sg.entries[k].last_use < sg.entries[lru].last_use) lru = k;
      if (sg.entries[lru].exec) cudaGraphExecDestroy(sg.entries[lru].exec);
      sg.entries.erase(sg.entries.begin() + lru);
    }
    Entry e; e.key = key; e.last_use = sg.tick;
    sg.entries.push_back(e);
    return run();
  }
  // second call with these arguments: capture on the private stream, then replay on the caller's
  ent->last_use = sg.tick;
  if (!sg.cap_stream && cudaStreamCreateWithFlags(&sg.cap_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); sg.disabled = true; return run(); }
  cudaStream_t user = c->L.stream;
  const unsigned long long count0 = c->L.count;
  if (cudaStreamBeginCapture(sg.cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); sg.disabled = true; return run(); }
  c->L.stream = sg.cap_stream;
  const pigan_status st = run();
  c->L.stream = user;
  cudaGraph_t graph = nullptr;
  const cudaError_t e = cudaStreamEndCapture(sg.cap_stream, &graph);
  const unsigned long long n_launch = c->L.count - count0;
  c->L.count = count0;
  if (st != PIGAN_OK || e != cudaSuccess || !graph || cudaGraphInstantiate(&ent->exec, graph, 0) != cudaSuccess) {
    cudaGetLastError();
    if (graph) cudaGraphDestroy(graph);
    ent->exec = nullptr; sg.disabled = true;                 // capture is not possible here: stay eager for the life of the context
    return run();
  }
  cudaGraphDestroy(graph);
  ent->launches = n_launch;
  if (cudaGraphLaunch(ent->exec, user) != cudaSuccess) { cudaGetLastError(); return fail(c, PIGAN_ERR_CUDA, "cudaGraphLaunch failed"); }
  c->L.count += ent->launches;
  return PIGAN_OK;
}

pigan_status pigan_train_step_grads_hier(pigan_ctx* c, const float* logk_params, const float* u_params, const float* disc_params, const int* subsets,
                                         const float* weights, const float* xy_colloc, const float* f, const float* xy_sensors, const float* z,
                                         const float* real_snap, const float* eps, float loss_scale, float* g_logk, float* g_u, float* g_disc,
                                         float* losses, int* found_inf) {
  if (!c) return PIGAN_ERR_INVALID_ARG;
  DeviceGuard dg(c);
  if (c->cfg.n_critics <= 0) return fail(c, PIGAN_ERR_UNSUPPORTED, "the context was created with n_critics = 0");
  if (!logk_params || !u_params || !disc_params || !subsets || !weights || !xy_colloc || !f || !xy_sensors || !z || !real_snap || !eps || !g_logk ||
      !g_u || !g_disc)
    return fail(c, PIGAN_ERR_INVALID_ARG, "null pointer");
  if (!(loss_scale > 0.f) || !std::isfinite(loss_scale)) return fail(c, PIGAN_ERR_INVALID_ARG, "loss_scale must be positive and finite");
  c->hier.K = c->cfg.n_critics; c->hier.subsets = subsets; c->hier.weights = weights;
  pigan_status st;
  if (c->cfg.precision == PIGAN_FP32)
    st = train_step_impl<float>(c, logk_params, u_params, disc_params, xy_colloc, f, xy_sensors, z, real_snap, eps, loss_scale, g_logk, g_u, g_disc, losses, found_inf);
  else
    st = train_step_impl<__half>(c, logk_params, u_params, disc_params, xy_colloc, f, xy_sensors, z, real_snap, eps, loss_scale, g_logk, g_u, g_disc, losses, found_inf);
  c->hier = pigan_ctx::Hier{};
  return st;
}

pigan_status pigan_adam_update(pigan_ctx* c, float* params, const float* grads, float* m, float* v, size_t n, int step, float lr, float beta1,
                               float beta2, float adam_eps, const int* skip_flag) {
  if (!c) return PIGAN_ERR_INVALID_ARG;
  DeviceGuard dg(c);
  if (n == 0) return PIGAN_OK;
  if (!params || !grads || !m || !v) return fail(c, PIGAN_ERR_INVALID_ARG, "null pointer");
  if (step < 1) return fail(c, PIGAN_ERR_INVALID_ARG, "step is 1-based");
  const float c1 = (float)(1.0 - std::pow((double)beta1, step)), c2 = (float)(1.0 - std::pow((double)beta2, step));
  adam(c->L, params, grads, m, v, n, lr, beta1, beta2, adam_eps, c1, c2, skip_flag);
  return finish(c);
}

}  // extern "C"
