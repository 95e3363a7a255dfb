// The context behind the C-ABI (include/pigan.h) and the small host helpers shared by api.cu (BASELINE.json's two-MLP
// generator) and trunk.cu (NEXT-1: the paper's shared-trunk generator).  Not part of the C-ABI.
#pragma once
#include <algorithm>
#include <new>
#include <string>
#include <vector>

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
  std::vector<void*> allocs;
  // CUDA-graph replay of pigan_train_step_grads: the step is hundreds to thousands of launches, launch-latency bound
  // for the small configs.  A call whose arguments repeat the previous call's is captured once (on a private stream,
  // so the caller's stream may be the legacy default stream) and replayed from then on.  PIGAN_FLAG_NO_GRAPH disables it.
  struct StepGraph {
    cudaStream_t cap_stream = nullptr;
    cudaGraphExec_t exec = nullptr;
    std::vector<unsigned long long> key, last_key;
    unsigned long long launches = 0;
    bool disabled = false;
  } sg;

  template <typename T> T* alloc(size_t n) {
    void* p = nullptr;
    if (n == 0) n = 1;
    if (cudaMalloc(&p, n * sizeof(T)) != cudaSuccess) { cudaGetLastError(); throw std::bad_alloc(); }
    allocs.push_back(p);
    return reinterpret_cast<T*>(p);
  }
  int n_sens_chunks = 1;
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

// NEXT-1 (trunk.cu)
pigan_status trunk_train_step(pigan_ctx* c, const float* thG, const float* thD, const float* xy_c, const float* f, const float* xy_s, const float* z,
                              const float* real, const float* eps, float loss_scale, float* gG, float* gD, float* losses, int* found_inf);
pigan_status trunk_jet_forward(pigan_ctx* c, const float* theta, const float* xy, int n_pts, const float* z, int n_samples, int C, float* out);

}  // namespace pigan
