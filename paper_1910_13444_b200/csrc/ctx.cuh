// The context behind the C-ABI (include/pigan.h) and the small host helpers shared by api.cu (BASELINE.json's two-MLP
// generator) and trunk.cu (NEXT-1: the paper's shared-trunk generator).  Not part of the C-ABI.
#pragma once
#include <algorithm>
#include <new>
#include <string>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "common.cuh"

namespace pigan {

struct NetWs {                 // activation workspace of one generator net (planes are [channel][unit][row])
  int Cmax = 0;
  char* h = nullptr;           // L x [Cmax][H][R_ld]      post-activations h^1..h^L
  char* hs = nullptr;          // sensor rows: n_sens_chunks x L x [2][H][R_ld]  (hi, lo) planes of the snapshot forward, kept for the reverse sweep
  char* ah[2] = {nullptr, nullptr};   // adjoint ping-pong, [Cmax][H][R_ld]
  float* apre = nullptr;       // fp32 mode: [Cmax][H][R_ld] pre-activations / hhat scratch
  float* o = nullptr;          // [Cmax][R_ld] outputs of the chunk
  float* oh = nullptr;         // [Cmax][R_ld] output adjoints (seeds)
  float* Zp = nullptr;         // [N][H]  first-layer z-part
  float* An = nullptr;         // [N][H]  per-sample sums of the first-layer value adjoint
  void* w16 = nullptr;         // (L-1) x {W_l, W_l^T} 16-bit copies
  // second adjoint set for the SENSOR rows (value channel only), so that their reverse sweep can run beside the collocation pass
  char* ah_s[2] = {nullptr, nullptr};   // [1][H][R_ld]
  float* oh_s = nullptr;       // [R_ld]
  float* apre_s = nullptr;     // fp32 mode: [1][H][R_ld]
  // NEXT-1, skip connections only (trunk.cu): the tanh jets t^l of the layers that take a skip are kept beside h^l = t^l + h^{l-2}
  char* ht = nullptr;          // L x [Cmax][H][R_ld]
  char* hts = nullptr;         // sensor rows: n_sens_chunks x L x [2][H][R_ld]
  char* sk = nullptr;          // [Cmax][H][R_ld]  adjoint travelling along the skip chain
  char* hhb = nullptr;         // [Cmax][H][R_ld]  raw adjoint planes hhat = W^T ahat of a skip layer (16-bit modes; fp32 mode uses apre)
};

}  // namespace pigan

struct pigan_ctx {
  pigan_config cfg{};
  pigan::NetShape gen{}, disc{};
  pigan::Launcher L;
  std::string err;
  int elem = 4;                // bytes per activation element
  int R_ld = 0;                // rows per chunk (leading dimension of every plane)
  pigan::NetWs net[2];                // 0: G_logk (C <= 3), 1: G_u (C <= 5)
  pigan::CriticWs cw;
  float* xfake = nullptr;      // [N][2S]
  float* dX = nullptr;         // [2N][2S]
  float* seed = nullptr;       // [2N]
  float* amax = nullptr;       // [2] largest output adjoint of the current chunk, per net (block scale of the adjoint planes)
  float* amax_s = nullptr;     // [2] the same for the sensor rows' own adjoint set (null: the sensor rows share net[n].ah / oh)
  std::vector<void*> allocs;
  // CUDA-graph replay of pigan_train_step_grads: the step is hundreds to thousands of launches, launch-latency bound
  // for the small configs.  The first call with a given argument set runs eagerly (it also sets kernel attributes); the second
  // call with that set -- not necessarily the next call -- is captured (on a private stream, so the caller's stream may be the
  // legacy default stream) and replayed from then on.  Up to kMaxGraphs argument sets are remembered (least recently used is
  // dropped), so a caller that alternates between a few sets, e.g. the sequential schedule with two output buffers, replays
  // too.  PIGAN_FLAG_NO_GRAPH disables it.
  struct StepGraph {
    static constexpr int kMaxGraphs = 4;
    struct Entry {
      std::vector<unsigned long long> key;
      cudaGraphExec_t exec = nullptr;                  // null: seen once, not captured yet
      unsigned long long launches = 0, last_use = 0;
    };
    cudaStream_t cap_stream = nullptr;
    std::vector<Entry> entries;
    unsigned long long tick = 0;
    bool disabled = false;
  } sg;

  template <typename T> T* alloc(size_t n) {
    void* p = nullptr;
    if (n == 0) n = 1;
    if (cudaMalloc(&p, n * sizeof(T)) != cudaSuccess) { cudaGetLastError(); throw std::bad_alloc(); }
    allocs.push_back(p);
    return reinterpret_cast<T*>(p);
  }
  // side streams of a step (api.cu): the critic stage beside the first collocation forward; net 1's kernels beside net 0's in one-chunk steps
  cudaStream_t side = nullptr, side2 = nullptr, side3 = nullptr;   // side3: net 1's sensor reverse sweep (beside net 0's on `side`)
  cudaEvent_t ev_pool[8] = {};
  int n_sens_chunks = 1;
  float* fbuf = nullptr;       // NEXT-2: [R_ld] f values of a chunk / the critic's adjoint of them
  // NEXT-3 (hier.cu): K critics on column subsets of the snapshot; set for the duration of pigan_train_step_grads_hier
  struct Hier { int K = 0; const int* subsets = nullptr; const float* weights = nullptr; } hier;
  float* hXf = nullptr; float* hXr = nullptr; float* hdX = nullptr;   // [N][d_sub] gathered fake / real sub-snapshots, one critic's input gradient
  double* htot = nullptr;      // [4] sum_k L_Dk, sum_k w_k mean D_k(fake), sum_k w_k mean D_k(real), sum_k GP_k
  bool trunk = false, skip = false;   // NEXT-1: shared-trunk generator (workspace of net[1]), with skip connections
  size_t plane() const { return (size_t)gen.H * R_ld * elem; }
  // activation stash of one chunk: `planes` planes per layer; l = 1..L
  struct HBuf { char* base; int planes; size_t plane_bytes; char* at(int l) const { return base + (size_t)(l - 1) * planes * plane_bytes; } };
  HBuf hcol(int n) { return HBuf{net[n].h, net[n].Cmax, plane()}; }
  HBuf hsens(int n, int chunk) { return HBuf{net[n].hs + (size_t)chunk * gen.L * 2 * plane(), 2, plane()}; }
  HBuf tcol(int n) { return HBuf{net[n].ht, net[n].Cmax, plane()}; }
  HBuf tsens(int n, int chunk) { return HBuf{net[n].hts + (size_t)chunk * gen.L * 2 * plane(), 2, plane()}; }
  void* w16(int n, int l, int transposed) { return (char*)net[n].w16 + ((size_t)(l - 2) * 2 + transposed) * gen.H * gen.H * 2; }
};

namespace pigan {

// Every entry point runs on the device the context was created on, whatever the caller's current device is.
struct DeviceGuard {
  int prev = -1; bool switched = false;
  explicit DeviceGuard(const pigan_ctx* c) {
    if (!c) return;
    if (cudaGetDevice(&prev) == cudaSuccess && prev != c->L.device) switched = cudaSetDevice(c->L.device) == cudaSuccess;
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

inline pigan_status fail(pigan_ctx* c, pigan_status s, const std::string& msg) {
  if (c) c->err = msg;
  return s;
}

inline pigan_status finish(pigan_ctx* c) {
  if (c->L.err != cudaSuccess) {
    c->err = std::string("CUDA error at ") + c->L.where + ": " + cudaGetErrorString(c->L.err);
    c->L.err = cudaSuccess;
    return PIGAN_ERR_CUDA;
  }
  c->err.clear();
  return PIGAN_OK;
}

// NVTX range per phase of a step (tracing): visible in nsys / ncu --nvtx; a no-op without a tool attached
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
};

inline size_t round_up(size_t a, size_t b) { return (a + b - 1) / b * b; }

inline ChunkGeom make_geom(const pigan_ctx* c, long long row0, long long total, int npts) {
  ChunkGeom g;
  g.row0 = row0;
  g.valid = (int)std::min<long long>(c->R_ld, total - row0);
  g.R = (int)round_up(g.valid, 64);
  g.R_ld = c->R_ld;
  g.npts = npts;
  return g;
}

// Zp[n][j] = sum_k W1[j][2+k] z[n][k]   (a1: once per sample; the bias is added with the xy-part)
inline void compute_zpart(pigan_ctx* c, int n, const float* theta, const float* z, int n_samples) {
  const NetShape& s = c->gen;
  sgemm(c->L, false, true, n_samples, s.H, s.in_dim - 2, z, s.in_dim - 2, 0, theta + 2, s.in_dim, 0, c->net[n].Zp, s.H, 0, 1, false);
}

// ---- one chunk of generator rows, forward ------------------------------------------------------------------------
template <typename T>
void gen_forward_chunk(pigan_ctx* c, int n, const pigan_ctx::HBuf& hb, const float* theta, int C, const float* xy, const ChunkGeom& g, float* o,
                       long long o_stride, bool split = false, bool keep_last = true) {
  const NetShape& s = c->gen;
  Launcher& L = c->L;
  const int H = s.H;
  const long long pl = (long long)H * g.R_ld;
  // split (16-bit modes, value channel only): activations are carried as two 16-bit planes hi + lo, so that the
  // snapshot X_fake the critic sees is accurate to ~2^-17 (the loss values are compared at 1e-3 relative)
  split = split && C == 1 && c->cfg.precision != PIGAN_FP32;
  if (c->cfg.precision == PIGAN_FP32 && gen_fused_f32_supported(s)) {     // narrow fp32 nets: one kernel, no activation planes
    gen_fused_f32_fwd(L, C, s, theta, c->net[n].Zp, xy, g, o, o_stride);
    return;
  }
  if (c->cfg.precision != PIGAN_FP32 && !split && !L.one_cta && tc_fused_fwd_supported(L, s, C, g)) {
    // width 128: the whole forward of the chunk in one kernel, activations stay on the SM between layers (tc_fused_fwd.cu)
    const void* wl[8]; void* hp[8];
    for (int l = 2; l <= s.L; ++l) wl[l - 2] = c->w16(n, l, 0);
    for (int l = 1; l <= s.L; ++l) hp[l - 1] = hb.at(l);
    OutDot od{theta + s.W_off(s.L + 1), theta + s.b_off(s.L + 1), o, o_stride, g.valid};
    cudaMemset2DAsync(o, (size_t)o_stride * 4, 0, (size_t)g.valid * 4, C, L.stream);
    tc_fused_fwd(L, c->cfg.precision, C, s, theta, wl, c->net[n].Zp, xy, g, hp, &od);
    return;
  }
  first_layer_fwd<T>(L, C, s, theta, c->net[n].Zp, xy, g, (T*)hb.at(1), split);
  // the output layer (a4) rides in the epilogue of the last hidden layer where the kernels support it
  const bool fuse_out = c->cfg.precision != PIGAN_FP32 && s.L >= 2 && tc_out_dot_fusable(L, H);
  for (int l = 2; l <= s.L; ++l) {
    if (c->cfg.precision == PIGAN_FP32) {
      // a_c = W_l h_c^{l-1}: M = H, N = rows, K = H, batched over the C channel planes
      sgemm(L, false, false, H, g.R, H, theta + s.W_off(l), H, 0, (const float*)hb.at(l - 1), g.R_ld, pl, c->net[n].apre, g.R_ld, pl, C, false);
      jet_act_fwd_f32(L, C, H, theta + s.b_off(l), g, c->net[n].apre, (float*)hb.at(l));
      continue;
    }
    OutDot od{theta + s.W_off(s.L + 1), theta + s.b_off(s.L + 1), o, o_stride, g.valid};
    const OutDot* odp = (fuse_out && l == s.L) ? &od : nullptr;
    void* h_out = (odp && !keep_last) ? nullptr : hb.at(l);
    if (odp) cudaMemset2DAsync(o, (size_t)o_stride * 4, 0, (size_t)g.valid * 4, C, L.stream);
    if (split) tc_layer_fwd_split(L, c->cfg.precision, H, g.R, g.R_ld, c->w16(n, l, 0), theta + s.b_off(l), hb.at(l - 1), h_out, odp);
    else tc_layer_fwd(L, c->cfg.precision, C, H, g.R, g.R_ld, c->w16(n, l, 0), theta + s.b_off(l), hb.at(l - 1), h_out, odp, false, /*reverse=*/(l & 1) != 0);
  }
  if (!fuse_out) out_fwd<T>(L, C, H, theta + s.W_off(s.L + 1), theta + s.b_off(s.L + 1), g, (const T*)hb.at(s.L), o, o_stride, split);
}

// ---- one chunk of generator rows, reverse sweep; output adjoints are in net[n].oh [C][R_ld] ------------------------
// sens: the adjoint planes, output adjoints and block scale of the sensor rows' own set (pigan_ctx::amax_s != nullptr)
template <typename T>
void gen_backward_chunk(pigan_ctx* c, int n, const pigan_ctx::HBuf& hb, const float* theta, float* grads, int C, const float* xy, const ChunkGeom& g,
                        bool sens = false) {
  const NetShape& s = c->gen;
  Launcher& L = c->L;
  const int H = s.H;
  const long long pl = (long long)H * g.R_ld;
  int cur = 0;
  struct { float* oh; char* ah[2]; float* apre; } w = {c->net[n].oh, {c->net[n].ah[0], c->net[n].ah[1]}, c->net[n].apre};
  if (sens) { w.oh = c->net[n].oh_s; w.ah[0] = c->net[n].ah_s[0]; w.ah[1] = c->net[n].ah_s[1]; w.apre = c->net[n].apre_s; }
  const float* amax = c->cfg.precision == PIGAN_FP32 ? nullptr : (sens ? c->amax_s : c->amax) + n;
  if (c->cfg.precision == PIGAN_FP32 && gen_fused_f32_supported(s)) {     // recomputes the forward of every row (gen_fused_f32.cu)
    gen_fused_f32_bwd(L, C, s, theta, c->net[n].Zp, xy, g, w.oh, grads, c->net[n].An);
    return;
  }
  jet_act_bwd_launch<T>(L, C, H, g, nullptr, theta + s.W_off(s.L + 1), w.oh, (const T*)hb.at(s.L),
                        (T*)w.ah[cur], grads + s.b_off(s.L),
                        grads + s.W_off(s.L + 1), grads + s.b_off(s.L + 1), amax);
  for (int l = s.L; l >= 2; --l) {
    if (c->cfg.precision == PIGAN_FP32) {
      // W_hat_l += sum_c ahat_c h_c^{l-1 T}: M = H, N = H, K = rows
      sgemm(L, false, true, H, H, g.R, (const float*)w.ah[cur], g.R_ld, pl, (const float*)hb.at(l - 1), g.R_ld, pl, grads + s.W_off(l), H, 0, C, true);
      // hhat_c^{l-1} = W_l^T ahat_c: M = H (in), N = rows, K = H (out); A stored [K][M]
      sgemm(L, true, false, H, g.R, H, theta + s.W_off(l), H, 0, (const float*)w.ah[cur], g.R_ld, pl, w.apre, g.R_ld, pl, C, false);
      jet_act_bwd_launch<T>(L, C, H, g, w.apre, nullptr, nullptr, (const T*)hb.at(l - 1),
                            (T*)w.ah[cur ^ 1], grads + s.b_off(l - 1), nullptr, nullptr, amax);
    } else if (tc_fused_bwd_supported(L, H, C)) {
      // widths 128 / 256: wgrad and dgrad of the layer in one kernel (ahat^l and h^{l-1} are read from HBM once)
      if (l == 2 && tc_first_layer_fusable(H, g)) {
        FirstLayerFuse fl{xy, g.row0, g.npts, s.in_dim, grads, c->net[n].An, g.per_sample};
        tc_fused_bwd(L, c->cfg.precision, C, H, g.R, g.R_ld, c->w16(n, l, 1), w.ah[cur], hb.at(l - 1), nullptr, grads + s.W_off(l),
                      grads + s.b_off(l - 1), amax, &fl);
        return;
      }
      tc_fused_bwd(L, c->cfg.precision, C, H, g.R, g.R_ld, c->w16(n, l, 1), w.ah[cur], hb.at(l - 1), w.ah[cur ^ 1],
                    grads + s.W_off(l), grads + s.b_off(l - 1), amax, nullptr);
    } else {
      tc_wgrad(L, c->cfg.precision, C, H, g.R, g.R_ld, w.ah[cur], hb.at(l - 1), grads + s.W_off(l), amax);
      if (l == 2 && tc_first_layer_fusable(H, g)) {
        // the adjoint of the first tanh layer is reduced inside the dgrad epilogue (ahat^1 is never written)
        FirstLayerFuse fl{xy, g.row0, g.npts, s.in_dim, grads, c->net[n].An, g.per_sample};
        tc_layer_bwd(L, c->cfg.precision, C, H, g.R, g.R_ld, c->w16(n, l, 1), w.ah[cur], hb.at(l - 1),
                     w.ah[cur ^ 1], grads + s.b_off(l - 1), amax, &fl);
        return;
      }
      tc_layer_bwd(L, c->cfg.precision, C, H, g.R, g.R_ld, c->w16(n, l, 1), w.ah[cur], hb.at(l - 1),
                   w.ah[cur ^ 1], grads + s.b_off(l - 1), amax);
    }
    cur ^= 1;
  }
  first_layer_bwd<T>(L, C, s, xy, g, (const T*)w.ah[cur], grads, c->net[n].An, amax);
}

// NEXT-1 (trunk.cu)
pigan_status trunk_train_step(pigan_ctx* c, const float* thG, const float* thD, const float* xy_c, const float* f, const float* xy_s, const float* z,
                              const float* real, const float* eps, float loss_scale, float* gG, float* gD, float* losses, int* found_inf);
pigan_status trunk_jet_forward(pigan_ctx* c, const float* theta, const float* xy, int n_pts, const float* z, int n_samples, int C, float* out);
// NEXT-3 (hier.cu): the critic stage with K critics (fills gD [K][count] and c->dX [N][2S]) and its loss scalars
void hier_critic_stage(pigan_ctx* c, const float* thD, const float* real, const float* eps, float* gD);
void hier_write_losses(pigan_ctx* c, long long NP, float* losses);
// NEXT-2 (free.cu): f at per-sample free sensors fed to the critic
pigan_status free_train_step(pigan_ctx* c, const float* thY, const float* thU, const float* thD, const float* xy_free, const float* xy_s, const float* z,
                             const float* real, const float* eps, float loss_scale, float* gY, float* gU, float* gD, float* losses, int* found_inf);

}  // namespace pigan
