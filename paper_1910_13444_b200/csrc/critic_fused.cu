// Fused critic sweeps for small critics: ONE kernel runs, for one latent sample per
// CTA, every per-row sweep of the WGAN-GP critic step -- forward on (fake, real, xhat), the two plain backprops, the
// backward-to-input of the gradient penalty (O5), its norm, and the ascending and descending sweeps of the double
// backward (O6) -- with all per-row vectors in shared memory and warp-level reductions.  What needs a reduction over the
// batch (the weight gradients) is left as two matrices per layer,  V_hat_l = A_l^T B_l,  which one batched SGEMM and one
// column-sum kernel finish.  ~100 launches of the layer-by-layer path become 5.  Used when the critic is small enough for
// every CTA to stream all of its weights (4 passes per CTA); larger critics (c4, c5) keep the layer-by-layer SGEMM path,
// where they are < 0.5 % of the step.
#include "common.cuh"

namespace pigan {

namespace {

constexpr int kCfThreads = 512;       // 16 warps: one CTA per sample, so the loads in flight per SM come from this CTA alone
constexpr int kCfWarps = kCfThreads / 32;
constexpr int kCfMaxIn = 512;      // largest layer input (d = 2S or HD) the fused path takes
constexpr int kCfMaxPer = kCfMaxIn / 32;

__device__ __forceinline__ float wsum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// y_v[j] = sum_i V[j][i] x_v[i] (+ bias[j]) for NV vectors; V is [n_out][n_in] row-major in global, x / y in shared memory.
// A warp owns output unit j (lanes stride over i: coalesced 128-byte reads of the weight row) and reduces by shuffles.
template <int NV>
__device__ __forceinline__ void matvec_rows(const float* __restrict__ V, const float* __restrict__ bias, int n_out, int n_in,
                                            const float* const* x, float* const* y) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  constexpr int U = 4;                                      // output units per warp iteration: U independent row streams in flight
  for (int j0 = warp * U; j0 < n_out; j0 += kCfWarps * U) {
    float acc[U][NV];
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
      for (int v = 0; v < NV; ++v) acc[u][v] = 0.f;
    for (int i = lane; i < n_in; i += 32) {
      float w[U];
#pragma unroll
      for (int u = 0; u < U; ++u) w[u] = (j0 + u < n_out) ? __ldg(V + (size_t)(j0 + u) * n_in + i) : 0.f;
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const float xv = x[v][i];
#pragma unroll
        for (int u = 0; u < U; ++u) acc[u][v] = fmaf(w[u], xv, acc[u][v]);
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
      for (int v = 0; v < NV; ++v) acc[u][v] = wsum(acc[u][v]);
    if (lane == 0) {
#pragma unroll
      for (int u = 0; u < U; ++u) {
        if (j0 + u < n_out) {
          const float b = bias ? bias[j0 + u] : 0.f;
#pragma unroll
          for (int v = 0; v < NV; ++v) y[v][j0 + u] = acc[u][v] + b;
        }
      }
    }
  }
}

// y_v[i] = sum_j V[j][i] x_v[j] (the transposed product) for NV vectors.  Warp w takes the rows j = w, w + kCfWarps, ...; lanes
// cover i (coalesced); the per-warp partial sums per i meet in shared memory.  y must be zero on entry.
template <int NV>
__device__ __forceinline__ void matvec_cols(const float* __restrict__ V, int n_out, int n_in, const float* const* x, float* const* y) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int per = (n_in + 31) / 32;
  float acc[NV][kCfMaxPer];
#pragma unroll
  for (int v = 0; v < NV; ++v)
#pragma unroll
    for (int k = 0; k < kCfMaxPer; ++k) acc[v][k] = 0.f;
#pragma unroll 2
  for (int j = warp; j < n_out; j += kCfWarps) {
    const float* row = V + (size_t)j * n_in;
    float xv[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) xv[v] = x[v][j];
#pragma unroll
    for (int k = 0; k < kCfMaxPer; ++k) {
      if (k < per) {
        const int i = k * 32 + lane;
        const float w = i < n_in ? __ldg(row + i) : 0.f;
#pragma unroll
        for (int v = 0; v < NV; ++v) acc[v][k] = fmaf(w, xv[v], acc[v][k]);
      }
    }
  }
#pragma unroll
  for (int k = 0; k < kCfMaxPer; ++k) {
    if (k < per) {
      const int i = k * 32 + lane;
      if (i < n_in) {
#pragma unroll
        for (int v = 0; v < NV; ++v) atomicAdd(&y[v][i], acc[v][k]);
      }
    }
  }
}

struct CfParams {
  NetShape s;
  const float* theta;
  const float* fake; const float* real; const float* eps;     // [B][d], [B][d], [B]
  int B;
  int plain;                // 1: also the fake / real rows (scores, plain backprops, dX); 0: gradient penalty only
  float lambda;
  float* A;                 // [LD][4B][HD]   rows: ahat_fake | ahat_real | adj_a (descending) | abar
  float* B1;                // [4B][d]        rows: X_fake | X_real | X_hat | adj(gbar^0)
  float* Bh;                // [LD][4B][HD]   slot l-2 (l = 2..LD+1): g_fake^{l-1} | g_real^{l-1} | g_hat^{l-1} | adj(gbar^{l-1})
  float* dX;                // [B][d] = (1/B) grad_X D(X_fake)   (plain only; may be null)
  float* nu; float* grad_norm;   // [B]
  double* acc;              // [0] += D(fake), [1] += D(real), [2] += (nu - 1)^2
  float* score;             // optional [3B] scores (fake | real | xhat), may be null
};

__global__ void __launch_bounds__(kCfThreads) critic_fused_kernel(CfParams p) {
  extern __shared__ float sm[];
  const NetShape& s = p.s;
  const int LD = s.L, HD = s.H, d = s.in_dim, B = p.B;
  const int n = blockIdx.x, tid = threadIdx.x;
  const int wmax = max(d, HD);
  // shared-memory carve-up (floats)
  float* X = sm;                         // [3][d]           fake, real, xhat
  float* g = X + 3 * d;                  // [LD][3][HD]      g^l of the three rows
  float* gbar = g + (size_t)LD * 3 * HD; // [LD][HD]         gbar^l (xhat row), l = 1..LD
  float* adjs = gbar + (size_t)LD * HD;  // [LD][HD]         adj(s^l)
  float* t0 = adjs + (size_t)LD * HD;    // [3][wmax]        running vectors
  float* t1 = t0 + 3 * wmax;             // [3][wmax]
  __shared__ float red[kCfWarps];
  __shared__ float s_nu;

  const float e = p.eps[n];
  for (int i = tid; i < d; i += kCfThreads) {
    const float f = p.fake[(size_t)n * d + i], r = p.real[(size_t)n * d + i];
    const float xh = e * r + (1.f - e) * f;
    X[i] = f; X[d + i] = r; X[2 * d + i] = xh;
    p.B1[((size_t)0 * B + n) * d + i] = f; p.B1[((size_t)1 * B + n) * d + i] = r; p.B1[((size_t)2 * B + n) * d + i] = xh;
  }
  __syncthreads();

  // ---- forward: g^l = tanh(V_l g^{l-1} + c_l) on the three rows (O1) ----
  for (int l = 1; l <= LD; ++l) {
    const int in = l == 1 ? d : HD;
    const float* src = l == 1 ? X : g + (size_t)(l - 2) * 3 * HD;
    float* dst = g + (size_t)(l - 1) * 3 * HD;
    const float* xs[3] = {src, src + in, src + 2 * in};
    float* ys[3] = {dst, dst + HD, dst + 2 * HD};
    matvec_rows<3>(p.theta + s.W_off(l), p.theta + s.b_off(l), HD, in, xs, ys);
    __syncthreads();
    for (int k = tid; k < 3 * HD; k += kCfThreads) {
      const float t = tanhf(dst[k]);
      dst[k] = t;
      const int row = k / HD, j = k - row * HD;
      p.Bh[((size_t)(l - 1) * 4 * B + (size_t)row * B + n) * HD + j] = t;         // B_{l+1} rows: g^l
    }
    __syncthreads();
  }
  // scores D = v_out . g^LD + c_out
  {
    const float* vout = p.theta + s.W_off(LD + 1);
    const float* gl = g + (size_t)(LD - 1) * 3 * HD;
    float a0 = 0.f, a1 = 0.f, a2 = 0.f;
    for (int j = tid; j < HD; j += kCfThreads) { const float w = vout[j]; a0 = fmaf(w, gl[j], a0); a1 = fmaf(w, gl[HD + j], a1); a2 = fmaf(w, gl[2 * HD + j], a2); }
    float part[3] = {a0, a1, a2};
    float tot[3];
    for (int v = 0; v < 3; ++v) {
      float x = wsum(part[v]);
      if ((tid & 31) == 0) red[tid >> 5] = x;
      __syncthreads();
      float t = 0.f;
      for (int w = 0; w < kCfWarps; ++w) t += red[w];
      tot[v] = t + p.theta[s.b_off(LD + 1)];
      __syncthreads();
    }
    if (tid == 0) {
      if (p.plain) { atomicAdd(p.acc + 0, (double)tot[0]); atomicAdd(p.acc + 1, (double)tot[1]); }
      if (p.score) { p.score[n] = tot[0]; p.score[B + n] = tot[1]; p.score[2 * B + n] = tot[2]; }
    }
  }

  // ---- one descending sweep through V_l^T for three vectors at once: the plain backprops of the fake (+1/B) and real
  //      (-1/B) rows (ahat^l = ghat^l * s^l) and the backward-to-input of the penalty on the xhat row (O5: abar^l = gbar^l * s^l) ----
  const float seedf = p.plain ? 1.f / B : 0.f, seedr = p.plain ? -1.f / B : 0.f;
  float* cur = t0; float* nxt = t1;
  {
    const float* vout = p.theta + s.W_off(LD + 1);
    for (int j = tid; j < HD; j += kCfThreads) { const float w = vout[j]; cur[j] = seedf * w; cur[wmax + j] = seedr * w; cur[2 * wmax + j] = w; }
  }
  __syncthreads();
  for (int l = LD; l >= 1; --l) {
    const int in = l == 1 ? d : HD;
    const float* gl = g + (size_t)(l - 1) * 3 * HD;
    for (int j = tid; j < HD; j += kCfThreads) {
      const float gb = cur[2 * wmax + j];
      gbar[(size_t)(l - 1) * HD + j] = gb;
      const float sf = 1.f - gl[j] * gl[j], sr = 1.f - gl[HD + j] * gl[HD + j], sx = 1.f - gl[2 * HD + j] * gl[2 * HD + j];
      const float af = cur[j] * sf, ar = cur[wmax + j] * sr, ab = gb * sx;
      cur[j] = af; cur[wmax + j] = ar; cur[2 * wmax + j] = ab;
      float* Al = p.A + (size_t)(l - 1) * 4 * B * HD;
      Al[((size_t)0 * B + n) * HD + j] = af; Al[((size_t)1 * B + n) * HD + j] = ar; Al[((size_t)3 * B + n) * HD + j] = ab;
    }
    for (int i = tid; i < 3 * wmax; i += kCfThreads) nxt[i] = 0.f;
    __syncthreads();
    const float* xs[3] = {cur, cur + wmax, cur + 2 * wmax};
    float* ys[3] = {nxt, nxt + wmax, nxt + 2 * wmax};
    matvec_cols<3>(p.theta + s.W_off(l), HD, in, xs, ys);
    __syncthreads();
    float* tmp = cur; cur = nxt; nxt = tmp;
  }
  // cur: [0] = (1/B) grad_X D(fake), [2] = G = gbar^0
  if (p.plain && p.dX) for (int i = tid; i < d; i += kCfThreads) p.dX[(size_t)n * d + i] = cur[i];
  {
    float a = 0.f;
    for (int i = tid; i < d; i += kCfThreads) { const float v = cur[2 * wmax + i]; a = fmaf(v, v, a); }
    a = wsum(a);
    if ((tid & 31) == 0) red[tid >> 5] = a;
    __syncthreads();
    if (tid == 0) {
      float t = 0.f;
      for (int w = 0; w < kCfWarps; ++w) t += red[w];
      const float nu = sqrtf(t);
      s_nu = nu;
      p.nu[n] = nu;
      if (p.grad_norm) p.grad_norm[n] = nu;
      atomicAdd(p.acc + 2, (double)(nu - 1.f) * (double)(nu - 1.f));
    }
    __syncthreads();
  }
  // ---- O6 ascending sweep: seed adj(gbar^0) = (lambda / B) 2 (nu - 1) G / nu  (0 when nu == 0, reading G12) ----
  {
    const float nu = s_nu;
    const float k = nu > 0.f ? (p.lambda / B) * 2.f * (nu - 1.f) / nu : 0.f;
    for (int i = tid; i < d; i += kCfThreads) {
      const float v = k * cur[2 * wmax + i];
      nxt[i] = v;
      p.B1[((size_t)3 * B + n) * d + i] = v;
    }
    __syncthreads();
    float* tmp = cur; cur = nxt; nxt = tmp;                  // cur[0..in) = adj(gbar^{l-1})
  }
  for (int l = 1; l <= LD; ++l) {
    const int in = l == 1 ? d : HD;
    const float* xs[1] = {cur};
    float* ys[1] = {nxt};
    matvec_rows<1>(p.theta + s.W_off(l), nullptr, HD, in, xs, ys);          // adj(abar^l) = V_l adj(gbar^{l-1})
    __syncthreads();
    const float* gl = g + (size_t)(l - 1) * 3 * HD + 2 * HD;                 // xhat row
    for (int j = tid; j < HD; j += kCfThreads) {
      const float aab = nxt[j], gx = gl[j];
      adjs[(size_t)(l - 1) * HD + j] = aab * gbar[(size_t)(l - 1) * HD + j];
      const float agb = aab * (1.f - gx * gx);
      nxt[j] = agb;                                                           // adj(gbar^l)
      p.Bh[((size_t)(l - 1) * 4 * B + (size_t)3 * B + n) * HD + j] = agb;     // B_{l+1} row 3: adj(gbar^l)
    }
    __syncthreads();
    float* tmp = cur; cur = nxt; nxt = tmp;
  }
  // ---- O6 descending sweep: adj(g^l) += -2 g^l adj(s^l); adj(a^l) = adj(g^l) s^l; adj(g^{l-1}) = V_l^T adj(a^l) ----
  for (int i = tid; i < wmax; i += kCfThreads) cur[i] = 0.f;
  __syncthreads();
  for (int l = LD; l >= 1; --l) {
    const int in = l == 1 ? d : HD;
    const float* gl = g + (size_t)(l - 1) * 3 * HD + 2 * HD;
    for (int j = tid; j < HD; j += kCfThreads) {
      const float gx = gl[j];
      const float ag = cur[j] - 2.f * gx * adjs[(size_t)(l - 1) * HD + j];
      const float aa = ag * (1.f - gx * gx);
      cur[j] = aa;
      p.A[((size_t)(l - 1) * 4 * B + (size_t)2 * B + n) * HD + j] = aa;
    }
    if (l > 1) for (int i = tid; i < wmax; i += kCfThreads) nxt[i] = 0.f;
    __syncthreads();
    if (l > 1) {
      const float* xs[1] = {cur};
      float* ys[1] = {nxt};
      matvec_cols<1>(p.theta + s.W_off(l), HD, in, xs, ys);
      __syncthreads();
      float* tmp = cur; cur = nxt; nxt = tmp;
    }
  }
}

// bias and output-layer gradients from the per-row matrices:
//   c_hat_l[j] = sum over the first 3B rows of A_l[:, j];  v_hat_out[j] = sum_n (g_fake^LD - g_real^LD) / B + adj(gbar^LD);  c_hat_out = 0
__global__ void __launch_bounds__(256) critic_bias_kernel(NetShape s, int B, int plain, const float* __restrict__ A, const float* __restrict__ Bh,
                                                          float* __restrict__ grads) {
  __shared__ float red[8][33];
  const int LD = s.L, HD = s.H;
  const int l = blockIdx.y + 1;                              // 1..LD: bias of layer l; LD + 1: output layer
  const int c = threadIdx.x & 31, rg = threadIdx.x >> 5, j = blockIdx.x * 32 + c;
  float acc = 0.f;
  if (j < HD) {
    if (l <= LD) {
      const float* Al = A + (size_t)(l - 1) * 4 * B * HD;
      for (int r = rg; r < 3 * B; r += 8) acc += Al[(size_t)r * HD + j];
    } else {
      const float* Bt = Bh + (size_t)(LD - 1) * 4 * B * HD;   // slot of l = LD + 1
      const float w = plain ? 1.f / B : 0.f;
      for (int r = rg; r < B; r += 8)
        acc += w * Bt[(size_t)r * HD + j] - w * Bt[((size_t)B + r) * HD + j] + Bt[((size_t)3 * B + r) * HD + j];
    }
  }
  red[rg][c] = acc;
  __syncthreads();
  if (rg == 0 && j < HD) {
    float t = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) t += red[k][c];
    if (l <= LD) grads[s.b_off(l) + j] = t; else grads[s.W_off(LD + 1) + j] = t;
  }
  if (l == LD + 1 && blockIdx.x == 0 && threadIdx.x == 0) {
    const float w = plain ? 1.f / B : 0.f;
    float sp = 0.f, sn = 0.f;
    for (int r = 0; r < B; ++r) { sp += w; sn += w; }
    grads[s.b_off(LD + 1)] = sp - sn;                        // sum of the output seeds: +1/B and -1/B, B times each
  }
}

size_t cf_smem_bytes(const NetShape& s) {
  const int wmax = std::max(s.in_dim, s.H);
  return ((size_t)3 * s.in_dim + (size_t)s.L * 3 * s.H + (size_t)2 * s.L * s.H + (size_t)6 * wmax) * sizeof(float);
}

}  // namespace

bool critic_fused_supported(const NetShape& s) {
  return s.H <= 256 && s.in_dim <= kCfMaxIn && s.L >= 1 && cf_smem_bytes(s) <= 200 * 1024 && s.H % 4 == 0;
}

// Critic step for small critics.  grads (may be null: no weight gradients) is OVERWRITTEN with
//   plain = 1: d/d theta_D [ mean D(fake) - mean D(real) + GP ];   plain = 0: d GP / d theta_D.
void critic_fused(Launcher& L, const NetShape& s, const float* theta, const float* fake, const float* real, const float* eps, int B, int plain,
                  float lambda, CriticWs& w, float* grads, float* dX, float* grad_norm) {
  CfParams p{};
  p.s = s; p.theta = theta; p.fake = fake; p.real = real; p.eps = eps; p.B = B; p.plain = plain; p.lambda = lambda;
  p.A = w.cfA; p.B1 = w.cfB1; p.Bh = w.cfBh; p.dX = dX; p.nu = w.nu; p.grad_norm = grad_norm; p.acc = w.acc; p.score = w.D;
  const size_t smem = cf_smem_bytes(s);
  static unsigned long long attr_done = 0;
  ensure_smem_attr(L, critic_fused_kernel, 200 * 1024, attr_done);        // the opt-in is per function: ask for the most any critic needs
  critic_fused_kernel<<<B, kCfThreads, smem, L.stream>>>(p);
  L.check("critic_fused");
  if (!grads) return;
  const int HD = s.H, d = s.in_dim, LD = s.L;
  // V_hat_1 = A_1^T B_1 (K = 4B rows);  V_hat_l = A_l^T B_l for l = 2..LD in one batched launch (parameter packing stride)
  sgemm(L, true, false, HD, d, 4 * B, w.cfA, HD, 0, w.cfB1, d, 0, grads + s.W_off(1), d, 0, 1, false);
  if (LD >= 2)
    sgemm(L, true, false, HD, HD, 4 * B, w.cfA + (size_t)4 * B * HD, HD, (long long)4 * B * HD, w.cfBh, HD, (long long)4 * B * HD,
          grads + s.W_off(2), HD, (long long)HD * HD + HD, LD - 1, false);
  dim3 grid((HD + 31) / 32, LD + 1);
  critic_bias_kernel<<<grid, 256, 0, L.stream>>>(s, B, plain, w.cfA, w.cfBh, grads);
  L.check("critic_bias");
}

}  // namespace pigan
