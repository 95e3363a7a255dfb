// fp32 mode, narrow generators (H = 32 or 64; config c1): the whole generator pass of a row in ONE kernel.
// SURVEY.md 8(a) a2-a4 (forward) and a10 (reverse sweep) run layer by layer as ~20 tiny launches per net and chunk in
// fp32 mode (SGEMM + elementwise), which at c1's 1024 rows is pure launch latency.  Here a WARP owns a row: lane j holds
// unit j (and j + 32 for H = 64) of every jet channel in registers, the H x H weights of all hidden layers sit in shared
// memory (W^T for the forward product, W for the transposed one, both read conflict-free), a layer's matrix-vector products
// broadcast the previous layer's activations lane by lane with warp shuffles, and the reductions over units (output dot)
// are warp-shuffle sums.  The reverse kernel recomputes the forward of its row (no activation planes exist in this path),
// keeps the per-layer jets and adjoints in per-warp shared-memory stashes; the CTA then accumulates the weight gradients of its
// 8 rows cooperatively in registers and flushes them with one fp32 atomic per entry and CTA.
#include "common.cuh"

namespace pigan {

namespace {

constexpr int kGfWarps = 8;
constexpr int kGfThreads = kGfWarps * 32;

__device__ __forceinline__ float gf_wsum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

struct GfSmem {            // offsets in floats into the dynamic shared memory
  int WT, W, gW, gb, stash, total;
};
__host__ __device__ inline GfSmem gf_layout(int L, int H, int C, bool bwd) {
  GfSmem m;
  const int hl = (L - 1) * H * H;
  m.WT = 0;
  m.W = m.WT + hl;
  m.gW = m.W + (bwd ? hl : 0);                               // reverse kernel: the adjoint stash [warp][l][c][unit]
  m.gb = m.gW;
  m.stash = m.gW + (bwd ? kGfWarps * L * C * H : 0);         // the jet stash
  m.total = m.stash + (bwd ? kGfWarps * L * C * H : 0);
  return m;
}

// a_c <- W_l h_c (+ b_l on the value channel): lane j accumulates unit j; h_c[k] arrives by shuffle, W^T[k][j] from smem
template <int UPL, int C>
__device__ __forceinline__ void gf_layer_matvec(const float* __restrict__ WT, const float* __restrict__ bias, int H, int lane, const float (*h)[UPL],
                                                float (*a)[UPL]) {
#pragma unroll
  for (int c = 0; c < C; ++c)
#pragma unroll
    for (int u = 0; u < UPL; ++u) a[c][u] = (c == 0) ? bias[lane + 32 * u] : 0.f;
#pragma unroll
  for (int ku = 0; ku < UPL; ++ku) {
#pragma unroll 16
    for (int kl = 0; kl < 32; ++kl) {
      float w[UPL];
#pragma unroll
      for (int u = 0; u < UPL; ++u) w[u] = WT[(ku * 32 + kl) * H + lane + 32 * u];
#pragma unroll
      for (int c = 0; c < C; ++c) {
        const float hv = __shfl_sync(0xffffffffu, h[c][ku], kl);
#pragma unroll
        for (int u = 0; u < UPL; ++u) a[c][u] = fmaf(w[u], hv, a[c][u]);
      }
    }
  }
}

template <int UPL, int C>
__device__ __forceinline__ void gf_act(float (*a)[UPL], float (*h)[UPL]) {
#pragma unroll
  for (int u = 0; u < UPL; ++u) {
    float av[5], hv[5];
#pragma unroll
    for (int c = 0; c < C; ++c) av[c] = a[c][u];
    jet_act_fwd<C>(tanhf(av[0]), av, hv);
#pragma unroll
    for (int c = 0; c < C; ++c) h[c][u] = hv[c];
  }
}

// first layer of the row (n, p): a = Zp[n] + b1 + W1[:,0] x + W1[:,1] y; a_x = W1[:,0], a_y = W1[:,1], a_xx = a_yy = 0
template <int UPL, int C>
__device__ __forceinline__ void gf_first(const NetShape& s, const float* __restrict__ theta, const float* __restrict__ Zp, int n, float x, float y, int lane,
                                         float (*h)[UPL]) {
  float a[C][UPL];
#pragma unroll
  for (int u = 0; u < UPL; ++u) {
    const int j = lane + 32 * u;
    const float wx = theta[(size_t)j * s.in_dim], wy = theta[(size_t)j * s.in_dim + 1];
    a[0][u] = Zp[(size_t)n * s.H + j] + theta[s.b_off(1) + j] + wx * x + wy * y;
    if (C >= 3) { a[1][u] = wx; a[2][u] = wy; }
    if (C >= 5) { a[3][u] = 0.f; a[4][u] = 0.f; }
  }
  gf_act<UPL, C>(a, h);
}

__device__ __forceinline__ void gf_row_geom(const ChunkGeom& g, int r, const float* __restrict__ xy, int& n, float& x, float& y) {
  const long long rg = g.row0 + r;
  n = (int)(rg / g.npts);
  const long long xi = g.per_sample ? rg : rg - (long long)n * g.npts;
  x = xy[2 * xi]; y = xy[2 * xi + 1];
}

template <int UPL, int C>
__global__ void __launch_bounds__(kGfThreads) gen_fused_fwd_kernel(NetShape s, const float* __restrict__ theta, const float* __restrict__ Zp,
                                                                   const float* __restrict__ xy, ChunkGeom g, float* __restrict__ o, long long o_stride) {
  extern __shared__ float sm[];
  const int H = s.H, L = s.L, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const GfSmem m = gf_layout(L, H, C, false);
  for (int l = 2; l <= L; ++l) {                              // W^T of the hidden layers: WT[k][j] = W_l[j][k]
    const float* W = theta + s.W_off(l);
    float* dst = sm + m.WT + (l - 2) * H * H;
    for (int i = threadIdx.x; i < H * H; i += kGfThreads) dst[(i % H) * H + i / H] = W[i];
  }
  __syncthreads();
  float wo[UPL];
#pragma unroll
  for (int u = 0; u < UPL; ++u) wo[u] = theta[s.W_off(L + 1) + lane + 32 * u];
  const float bo = theta[s.b_off(L + 1)];
  for (int r = blockIdx.x * kGfWarps + warp; r < g.valid; r += gridDim.x * kGfWarps) {
    int n; float x, y;
    gf_row_geom(g, r, xy, n, x, y);
    float h[C][UPL], a[C][UPL];
    gf_first<UPL, C>(s, theta, Zp, n, x, y, lane, h);
    for (int l = 2; l <= L; ++l) {
      gf_layer_matvec<UPL, C>(sm + m.WT + (l - 2) * H * H, theta + s.b_off(l), H, lane, h, a);
      gf_act<UPL, C>(a, h);
    }
#pragma unroll
    for (int c = 0; c < C; ++c) {
      float v = 0.f;
#pragma unroll
      for (int u = 0; u < UPL; ++u) v = fmaf(wo[u], h[c][u], v);
      v = gf_wsum(v);
      if (lane == 0) o[(size_t)c * o_stride + r] = v + (c == 0 ? bo : 0.f);
    }
  }
}

// Reverse sweep.  The CTA works on batches of 8 rows (one per warp).  Each warp recomputes the forward of its row (jets of every
// layer -> shared-memory stash), runs the reverse sweep and leaves the pre-activation adjoints ahat^l in a second stash; after a
// barrier the 256 threads of the CTA accumulate the batch's outer products  W_hat_l[j][k] += sum_{rows, c} ahat_c[j] h^{l-1}_c[k]
// into REGISTERS (thread t owns entries t, t + 256, ... of every layer) -- no shared-memory atomics -- and flush them with one
// global fp32 atomic per entry at the end of the kernel.
constexpr int kGfMaxOwn = 48;      // (L - 1) H^2 / 256 entries per thread: H = 64, L = 4

template <int UPL, int C>
__global__ void __launch_bounds__(kGfThreads, 1) gen_fused_bwd_kernel(NetShape s, const float* __restrict__ theta, const float* __restrict__ Zp,
                                                                      const float* __restrict__ xy, ChunkGeom g, const float* __restrict__ ohat,
                                                                      float* __restrict__ grads, float* __restrict__ An) {
  extern __shared__ float sm[];
  constexpr int H = 32 * UPL;
  const int L = s.L, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const GfSmem m = gf_layout(L, H, C, true);
  for (int l = 2; l <= L; ++l) {
    const float* W = theta + s.W_off(l);
    float* wt = sm + m.WT + (l - 2) * H * H;
    float* w = sm + m.W + (l - 2) * H * H;
    for (int i = threadIdx.x; i < H * H; i += kGfThreads) { const float v = W[i]; w[i] = v; wt[(i % H) * H + i / H] = v; }
  }
  __syncthreads();
  float* stash_h = sm + m.stash;                              // [warp][l][c][unit] jets h^l of the batch's rows
  float* stash_a = sm + m.gW;                                 // [warp][l][c][unit] adjoints ahat^l
  float* my_h = stash_h + warp * (L * C * H);
  float* my_a = stash_a + warp * (L * C * H);
  const int n_own = (L - 1) * H * H / kGfThreads;             // weight-gradient entries this thread accumulates
  float gw[kGfMaxOwn];
#pragma unroll
  for (int e = 0; e < kGfMaxOwn; ++e) gw[e] = 0.f;
  float gbias = 0.f;                                          // thread t < L * H owns b_hat_{t / H + 1}[t % H]
  float wo[UPL], g_wo[UPL], g_wx[UPL], g_wy[UPL];
#pragma unroll
  for (int u = 0; u < UPL; ++u) { wo[u] = theta[s.W_off(L + 1) + lane + 32 * u]; g_wo[u] = 0.f; g_wx[u] = 0.f; g_wy[u] = 0.f; }
  float g_bo = 0.f;
  const int n_batches = (g.valid + kGfWarps - 1) / kGfWarps;
  for (int b = blockIdx.x; b < n_batches; b += gridDim.x) {
    const int r = b * kGfWarps + warp;
    if (r < g.valid) {
      int n; float x, y;
      gf_row_geom(g, r, xy, n, x, y);
      float h[C][UPL], a[C][UPL];
      // ---- forward of this row, jets of every layer kept in the stash ----
      gf_first<UPL, C>(s, theta, Zp, n, x, y, lane, h);
      for (int l = 1;; ++l) {
#pragma unroll
        for (int c = 0; c < C; ++c)
#pragma unroll
          for (int u = 0; u < UPL; ++u) my_h[((l - 1) * C + c) * H + lane + 32 * u] = h[c][u];
        if (l == L) break;
        gf_layer_matvec<UPL, C>(sm + m.WT + (l - 1) * H * H, theta + s.b_off(l + 1), H, lane, h, a);
        gf_act<UPL, C>(a, h);
      }
      // ---- reverse: output layer ----
      float oh[C], hh[C][UPL];
#pragma unroll
      for (int c = 0; c < C; ++c) oh[c] = ohat[(size_t)c * g.R_ld + r];
      g_bo += oh[0];
#pragma unroll
      for (int c = 0; c < C; ++c)
#pragma unroll
        for (int u = 0; u < UPL; ++u) { hh[c][u] = wo[u] * oh[c]; g_wo[u] = fmaf(oh[c], h[c][u], g_wo[u]); }
      // ---- reverse: tanh layers L .. 1 ----
      for (int l = L; l >= 1; --l) {
        float aa[C][UPL];
#pragma unroll
        for (int u = 0; u < UPL; ++u) {
          float hj[5], hx[5], av[5];
#pragma unroll
          for (int c = 0; c < C; ++c) { hj[c] = my_h[((l - 1) * C + c) * H + lane + 32 * u]; hx[c] = hh[c][u]; }
          jet_act_bwd<C>(hj, hx, av);
#pragma unroll
          for (int c = 0; c < C; ++c) { aa[c][u] = av[c]; my_a[((l - 1) * C + c) * H + lane + 32 * u] = av[c]; }
        }
        if (l == 1) {
#pragma unroll
          for (int u = 0; u < UPL; ++u) {
            g_wx[u] += aa[0][u] * x + (C >= 3 ? aa[1][u] : 0.f);
            g_wy[u] += aa[0][u] * y + (C >= 3 ? aa[2][u] : 0.f);
            atomicAdd(An + (size_t)n * H + lane + 32 * u, aa[0][u]);
          }
          break;
        }
        // hhat^{l-1}_c[k] = sum_j W_l[j][k] ahat_c[j]: lane k accumulates, ahat_c[j] arrives by shuffle, W_l[j][k] from smem
        const float* Wl = sm + m.W + (l - 2) * H * H;
#pragma unroll
        for (int c = 0; c < C; ++c)
#pragma unroll
          for (int u = 0; u < UPL; ++u) hh[c][u] = 0.f;
#pragma unroll
        for (int ju = 0; ju < UPL; ++ju) {
#pragma unroll 16
          for (int jl = 0; jl < 32; ++jl) {
            float w[UPL];
#pragma unroll
            for (int u = 0; u < UPL; ++u) w[u] = Wl[(ju * 32 + jl) * H + lane + 32 * u];
#pragma unroll
            for (int c = 0; c < C; ++c) {
              const float av = __shfl_sync(0xffffffffu, aa[c][ju], jl);
#pragma unroll
              for (int u = 0; u < UPL; ++u) hh[c][u] = fmaf(w[u], av, hh[c][u]);
            }
          }
        }
      }
    } else {
      for (int i = lane; i < L * C * H; i += 32) { my_a[i] = 0.f; my_h[i] = 0.f; }   // a missing row adds nothing below
    }
    __syncthreads();
    // ---- the batch's weight and bias gradients, cooperatively: thread t owns entries e = t + 256 q of [l][j][k] ----
    for (int q = 0; q < n_own; ++q) {
      const int e = threadIdx.x + q * kGfThreads;
      const int l2 = e / (H * H), jk = e - l2 * (H * H), jj = jk / H, kk = jk - jj * H;    // layer l = l2 + 2
      float acc = 0.f;
#pragma unroll
      for (int w = 0; w < kGfWarps; ++w) {
        const float* ap = stash_a + w * (L * C * H) + (l2 + 1) * C * H + jj;            // ahat^{l}_c[jj]
        const float* hp = stash_h + w * (L * C * H) + l2 * C * H + kk;                  // h^{l-1}_c[kk]
#pragma unroll
        for (int c = 0; c < C; ++c) acc = fmaf(ap[c * H], hp[c * H], acc);
      }
#pragma unroll
      for (int qq = 0; qq < kGfMaxOwn; ++qq) if (qq == q) gw[qq] += acc;
    }
    if (threadIdx.x < L * H) {
      const int l0 = threadIdx.x / H, jj = threadIdx.x - l0 * H;
      float acc = 0.f;
#pragma unroll
      for (int w = 0; w < kGfWarps; ++w) acc += stash_a[w * (L * C * H) + l0 * C * H + jj];
      gbias += acc;
    }
    __syncthreads();
  }
  // ---- flush ----
#pragma unroll
  for (int u = 0; u < UPL; ++u) {
    const int j = lane + 32 * u;
    atomicAdd(grads + s.W_off(L + 1) + j, g_wo[u]);
    atomicAdd(grads + (size_t)j * s.in_dim, g_wx[u]);
    atomicAdd(grads + (size_t)j * s.in_dim + 1, g_wy[u]);
  }
  if (lane == 0) atomicAdd(grads + s.b_off(L + 1), g_bo);     // every lane carries the same sum of ohat_0: one of them adds it
  for (int q = 0; q < n_own; ++q) {
    const int e = threadIdx.x + q * kGfThreads;
    const int l2 = e / (H * H), jk = e - l2 * (H * H);
    float v = 0.f;
#pragma unroll
    for (int qq = 0; qq < kGfMaxOwn; ++qq) if (qq == q) v = gw[qq];
    atomicAdd(grads + s.W_off(l2 + 2) + jk, v);
  }
  if (threadIdx.x < L * H) atomicAdd(grads + s.b_off(threadIdx.x / H + 1) + threadIdx.x % H, gbias);
}

}  // namespace

bool gen_fused_f32_supported(const NetShape& s) {
  if (!(s.H == 32 || s.H == 64) || s.L < 1 || s.heads != 1) return false;
  if ((s.L - 1) * s.H * s.H / kGfThreads > kGfMaxOwn || s.L * s.H > kGfThreads) return false;
  return (size_t)gf_layout(s.L, s.H, 5, true).total * 4 <= 200 * 1024;
}

template <int UPL>
static void gf_launch_fwd(Launcher& L, int C, const NetShape& s, const float* theta, const float* Zp, const float* xy, const ChunkGeom& g, float* o,
                          long long o_stride, int grid, size_t smem) {
  static unsigned long long done[3] = {0, 0, 0};
#define PIGAN_GF(c, i)                                                                                      \
  { ensure_smem_attr(L, gen_fused_fwd_kernel<UPL, c>, 200 * 1024, done[i]);                               \
    gen_fused_fwd_kernel<UPL, c><<<grid, kGfThreads, smem, L.stream>>>(s, theta, Zp, xy, g, o, o_stride); }
  if (C == 1) PIGAN_GF(1, 0) else if (C == 3) PIGAN_GF(3, 1) else PIGAN_GF(5, 2)
#undef PIGAN_GF
}
template <int UPL>
static void gf_launch_bwd(Launcher& L, int C, const NetShape& s, const float* theta, const float* Zp, const float* xy, const ChunkGeom& g,
                          const float* ohat, float* grads, float* An, int grid, size_t smem) {
  static unsigned long long done[3] = {0, 0, 0};
#define PIGAN_GF(c, i)                                                                                      \
  { ensure_smem_attr(L, gen_fused_bwd_kernel<UPL, c>, 200 * 1024, done[i]);                               \
    gen_fused_bwd_kernel<UPL, c><<<grid, kGfThreads, smem, L.stream>>>(s, theta, Zp, xy, g, ohat, grads, An); }
  if (C == 1) PIGAN_GF(1, 0) else if (C == 3) PIGAN_GF(3, 1) else PIGAN_GF(5, 2)
#undef PIGAN_GF
}

void gen_fused_f32_fwd(Launcher& L, int C, const NetShape& s, const float* theta, const float* Zp, const float* xy, const ChunkGeom& g, float* o,
                       long long o_stride) {
  if (g.valid <= 0) return;
  const int grid = std::max(1, std::min((g.valid + kGfWarps - 1) / kGfWarps, 2 * L.num_sms));
  const size_t smem = (size_t)gf_layout(s.L, s.H, C, false).total * 4;
  if (s.H == 32) gf_launch_fwd<1>(L, C, s, theta, Zp, xy, g, o, o_stride, grid, smem);
  else gf_launch_fwd<2>(L, C, s, theta, Zp, xy, g, o, o_stride, grid, smem);
  L.check("gen_fused_fwd");
}

void gen_fused_f32_bwd(Launcher& L, int C, const NetShape& s, const float* theta, const float* Zp, const float* xy, const ChunkGeom& g,
                       const float* ohat, float* grads, float* An) {
  if (g.valid <= 0) return;
  const int grid = std::max(1, std::min((g.valid + kGfWarps - 1) / kGfWarps, L.num_sms));
  const size_t smem = (size_t)gf_layout(s.L, s.H, C, true).total * 4;
  if (s.H == 32) gf_launch_bwd<1>(L, C, s, theta, Zp, xy, g, ohat, grads, An, grid, smem);
  else gf_launch_bwd<2>(L, C, s, theta, Zp, xy, g, ohat, grads, An, grid, smem);
  L.check("gen_fused_bwd");
}

}  // namespace pigan
