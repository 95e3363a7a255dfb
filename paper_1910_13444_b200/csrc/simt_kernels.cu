// FP32 SIMT kernels of the PI-GAN hot path: everything that is not a 16-bit tensor-core contraction.
// First layer (S8a a1, a2), output dot (a4), Darcy residual (a5), the tanh-jet chain rule and its adjoint in fp32
// mode (a3, a10), first-layer backward, critic (a7-a9, always fp32), Adam (a11).  Activations of the generator
// are feature-major planes [channel][unit][row] so that a thread that owns a unit touches contiguous rows.
#include "common.cuh"

namespace pigan {

static inline int cdiv(long long a, long long b) { return (int)((a + b - 1) / b); }

// =============================================================================================================
// generic batched SGEMM (64x64x32 tiles, 4x4 micro-tiles, register prefetch); used by fp32 mode and by the critic
// =============================================================================================================
template <bool TA, bool TB>
__global__ void __launch_bounds__(256) sgemm_kernel(int M, int N, int K, const float* __restrict__ A, int lda, long long sA,
                                                    const float* __restrict__ B, int ldb, long long sB, float* __restrict__ C,
                                                    int ldc, long long sC, int ksplit, int atomic, float alpha) {
  // 64 x 64 output tile, 32-deep k-steps; the global loads of step k+1 are issued into registers before step k is
  // multiplied, so their latency overlaps the FMAs (the critic's GEMMs are a handful of CTAs with 4-13 k-steps each:
  // latency, not throughput, is what they cost).
  constexpr int BK = 32;
  __shared__ float As[BK][68];
  __shared__ float Bs[BK][68];
  const int batch = blockIdx.z / ksplit, ks = blockIdx.z % ksplit;
  A += (long long)batch * sA; B += (long long)batch * sB; C += (long long)batch * sC;
  int kchunk = (K + ksplit - 1) / ksplit; kchunk = (kchunk + BK - 1) / BK * BK;
  const int k0 = ks * kchunk, k1 = min(K, k0 + kchunk);
  const int m0 = blockIdx.y * 64, n0 = blockIdx.x * 64;
  const int tid = threadIdx.x, tx = tid % 16, ty = tid / 16;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
  float ra[8], rb[8];
  auto fetch = [&](int k) {                                  // this thread's 8 + 8 elements of the (64 x BK) A and (BK x 64) B tiles
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int idx = tid + i * 256;
      int m, kk;
      if (!TA) { m = idx / BK; kk = idx % BK; } else { kk = idx / 64; m = idx % 64; }
      float v = 0.f;
      if (m0 + m < M && k + kk < k1) v = TA ? A[(long long)(k + kk) * lda + m0 + m] : A[(long long)(m0 + m) * lda + k + kk];
      ra[i] = v;
      int n;
      if (!TB) { kk = idx / 64; n = idx % 64; } else { n = idx / BK; kk = idx % BK; }
      v = 0.f;
      if (n0 + n < N && k + kk < k1) v = TB ? B[(long long)(n0 + n) * ldb + k + kk] : B[(long long)(k + kk) * ldb + n0 + n];
      rb[i] = v;
    }
  };
  auto stash = [&]() {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int idx = tid + i * 256;
      if (!TA) As[idx % BK][idx / BK] = ra[i]; else As[idx / 64][idx % 64] = ra[i];
      if (!TB) Bs[idx / 64][idx % 64] = rb[i]; else Bs[idx % BK][idx / BK] = rb[i];
    }
  };
  if (k0 < k1) fetch(k0);
  for (int k = k0; k < k1; k += BK) {
    stash();
    __syncthreads();
    if (k + BK < k1) fetch(k + BK);
#pragma unroll
    for (int kk = 0; kk < BK; ++kk) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = As[kk][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Bs[kk][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int m = m0 + ty * 4 + i;
    if (m >= M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int n = n0 + tx * 4 + j;
      if (n >= N) continue;
      float* p = C + (long long)m * ldc + n;
      if (atomic) atomicAdd(p, alpha * acc[i][j]); else *p = alpha * acc[i][j];
    }
  }
}

void sgemm(Launcher& L, bool TA, bool TB, int M, int N, int K, const float* A, int lda, long long sA, const float* B,
           int ldb, long long sB, float* C, int ldc, long long sC, int batch, bool accumulate, float alpha) {
  if (M <= 0 || N <= 0 || batch <= 0) return;
  const int tiles = cdiv(M, 64) * cdiv(N, 64) * batch;
  int ksplit = 1;
  if (K <= 0) {                                 // empty contraction: result is zero
    if (!accumulate) for (int b = 0; b < batch; ++b) cudaMemset2DAsync(C + b * sC, (size_t)ldc * 4, 0, (size_t)N * 4, M, L.stream);
    return;
  }
  if (tiles < 296 && K >= 256) {                // too few tiles to fill 148 SMs: split the contraction
    ksplit = min(cdiv(592, tiles), K / 128);
    if (ksplit < 1) ksplit = 1;
  } else if (accumulate && tiles < 74 && K >= 64) {
    // the critic's weight-gradient GEMMs (a handful of tiles, K = batch rows): they accumulate with atomics anyway, so
    // splitting the contraction costs nothing and turns 6 serial k-steps per CTA into 1-2
    ksplit = min(cdiv(148, tiles), K / 32);
    if (ksplit < 1) ksplit = 1;
  }
  bool atomic = accumulate;
  if (ksplit > 1 && !accumulate) {
    for (int b = 0; b < batch; ++b) cudaMemset2DAsync(C + b * sC, (size_t)ldc * 4, 0, (size_t)N * 4, M, L.stream);
    atomic = true;
  }
  dim3 grid(cdiv(N, 64), cdiv(M, 64), batch * ksplit);
#define PIGAN_SGEMM(ta, tb) sgemm_kernel<ta, tb><<<grid, 256, 0, L.stream>>>(M, N, K, A, lda, sA, B, ldb, sB, C, ldc, sC, ksplit, atomic ? 1 : 0, alpha)
  if (!TA && !TB) PIGAN_SGEMM(false, false);
  else if (TA && !TB) PIGAN_SGEMM(true, false);
  else if (!TA && TB) PIGAN_SGEMM(false, true);
  else PIGAN_SGEMM(true, true);
#undef PIGAN_SGEMM
  L.check("sgemm");
}

// =============================================================================================================
// generator: first layer (a1 z-part comes from sgemm; a2 here), fp32 math, writes feature-major planes
// =============================================================================================================
// fp32 mode: tanh-jet chain rule applied to the pre-activations written by sgemm
template <int C>
__global__ void __launch_bounds__(128) jet_act_fwd_kernel(int H, const float* __restrict__ bias, ChunkGeom g,
                                                          const float* __restrict__ apre, float* __restrict__ h) {
  const int r = blockIdx.x * 128 + threadIdx.x, j = blockIdx.y;
  if (r >= g.R) return;
  const size_t plane = (size_t)H * g.R_ld, off = (size_t)j * g.R_ld + r;
  float a[5], o[5];
#pragma unroll
  for (int c = 0; c < C; ++c) a[c] = apre[c * plane + off];
  a[0] += bias[j];
  jet_act_fwd<C>(tanhf(a[0]), a, o);
#pragma unroll
  for (int c = 0; c < C; ++c) h[c * plane + off] = o[c];
}

void jet_act_fwd_f32(Launcher& L, int C, int H, const float* bias, const ChunkGeom& g, const float* apre, float* h) {
  dim3 grid(cdiv(g.R, 128), H);
  if (C == 1) jet_act_fwd_kernel<1><<<grid, 128, 0, L.stream>>>(H, bias, g, apre, h);
  else if (C == 3) jet_act_fwd_kernel<3><<<grid, 128, 0, L.stream>>>(H, bias, g, apre, h);
  else jet_act_fwd_kernel<5><<<grid, 128, 0, L.stream>>>(H, bias, g, apre, h);
  L.check("jet_act_fwd");
}

// =============================================================================================================
// Darcy residual (a5, Eq. 1) + adjoint seeds (O3); warp-shuffle + block reduction of sum r^2
// =============================================================================================================
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__global__ void __launch_bounds__(256) residual_kernel(const float* __restrict__ Y, long long ys, const float* __restrict__ U, long long us,
                                                       const float* __restrict__ f, long long row0, int valid, int R, int npts,
                                                       float* __restrict__ r_out, double* __restrict__ sum_sq, float seed_scale,
                                                       float* __restrict__ seedY, float* __restrict__ seedU, int seed_ld,
                                                       float* __restrict__ amaxY, float* __restrict__ amaxU, const float* __restrict__ ext_seed) {
  __shared__ double red[8];
  float my = 0.f, mu = 0.f;
  const int r = blockIdx.x * 256 + threadIdx.x;
  double sq = 0.0;
  if (r < R) {
    float sy[3] = {0.f, 0.f, 0.f}, su[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
    if (r < valid) {
      const int p = (int)((row0 + r) % npts);
      const float y0 = Y[r], yx = Y[ys + r], yy = Y[2 * ys + r];
      const float ux = U[us + r], uy = U[2 * us + r], uxx = U[3 * us + r], uyy = U[4 * us + r];
      const float k = expf(y0);
      const float D = fmaf(yx, ux, fmaf(yy, uy, uxx + uyy));
      const float res = fmaf(k, D, f ? -f[p] : 0.f);
      if (r_out) r_out[r] = res;
      sq = (double)res * (double)res;
      const float rk = (seed_scale * res + (ext_seed ? ext_seed[r] : 0.f)) * k;   // r_hat * k  (loss-scaled in 16-bit modes)
      sy[0] = rk * D; sy[1] = rk * ux; sy[2] = rk * uy;
      su[1] = rk * yx; su[2] = rk * yy; su[3] = rk; su[4] = rk;
      my = fmaxf(fabsf(sy[0]), fmaxf(fabsf(sy[1]), fabsf(sy[2])));
      mu = fmaxf(fabsf(su[1]), fmaxf(fabsf(su[2]), fabsf(su[3])));
    }
    if (seedY) {
#pragma unroll
      for (int c = 0; c < 3; ++c) seedY[(size_t)c * seed_ld + r] = sy[c];
#pragma unroll
      for (int c = 0; c < 5; ++c) seedU[(size_t)c * seed_ld + r] = su[c];
    }
  }
  if (amaxY) {                                               // largest output adjoint of the chunk (positive floats order as ints)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { my = fmaxf(my, __shfl_xor_sync(0xffffffffu, my, o)); mu = fmaxf(mu, __shfl_xor_sync(0xffffffffu, mu, o)); }
    if ((threadIdx.x & 31) == 0) {
      if (!(my <= 3.0e38f)) my = INFINITY;                   // NaN/inf -> inf (flagged downstream through the gradients)
      if (!(mu <= 3.0e38f)) mu = INFINITY;
      atomicMax(reinterpret_cast<int*>(amaxY), __float_as_int(my));
      atomicMax(reinterpret_cast<int*>(amaxU), __float_as_int(mu));
    }
  }
  if (sum_sq) {
    sq = warp_sum_d(sq);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = sq;
    __syncthreads();
    if (threadIdx.x < 8) {
      double v = red[threadIdx.x];
      for (int o = 4; o > 0; o >>= 1) v += __shfl_xor_sync(0xffu, v, o);
      if (threadIdx.x == 0) atomicAdd(sum_sq, v);
    }
  }
}

void residual(Launcher& L, const float* Y, long long y_stride, const float* U, long long u_stride, const float* f, long long row0,
              int valid, int R, int npts, float* r_out, double* sum_sq, float seed_scale, float* seedY, float* seedU, int seed_ld,
              float* amaxY, float* amaxU, const float* ext_seed) {
  if (R <= 0) return;
  residual_kernel<<<cdiv(R, 256), 256, 0, L.stream>>>(Y, y_stride, U, u_stride, f, row0, valid, R, npts, r_out, sum_sq, seed_scale,
                                                      seedY, seedU, seed_ld, amaxY, amaxU, ext_seed);
  L.check("residual");
}

void finalize_first_layer(Launcher& L, const NetShape& s, int N, const float* An, const float* z, float* grads) {
  const int m = s.in_dim - 2;
  // W_hat_1[:, 2:] = An^T z : M = H, N = m, K = N_samples; A stored [K][M]
  // (b_hat_1 = sum_{n,p} a_hat is already reduced by the adjoint kernel of layer 1)
  sgemm(L, true, false, s.H, m, N, An, s.H, 0, z, m, 0, grads + 2, s.in_dim, 0, 1, /*accumulate=*/true);
}

// =============================================================================================================
// gradient post-processing and Adam (a11): vectorised, coalesced elementwise kernels
// =============================================================================================================
__global__ void __launch_bounds__(256) unscale_check_kernel(float* __restrict__ g, size_t n, float inv_scale, int* __restrict__ found_inf) {
  const size_t n4 = n / 4;
  bool bad = false;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
    float4 v = reinterpret_cast<float4*>(g)[i];
    v.x *= inv_scale; v.y *= inv_scale; v.z *= inv_scale; v.w *= inv_scale;
    bad |= !(isfinite(v.x) && isfinite(v.y) && isfinite(v.z) && isfinite(v.w));
    reinterpret_cast<float4*>(g)[i] = v;
  }
  if (blockIdx.x == 0 && threadIdx.x < (n & 3)) {
    float v = g[n4 * 4 + threadIdx.x] * inv_scale;
    bad |= !isfinite(v);
    g[n4 * 4 + threadIdx.x] = v;
  }
  if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0 && found_inf) atomicOr(found_inf, 1);
}

void unscale_and_check(Launcher& L, float* g, size_t n, float inv_scale, int* found_inf) {
  if (n == 0) return;
  const int blocks = (int)std::min<size_t>((n / 4 + 255) / 256 + 1, 148 * 8);
  unscale_check_kernel<<<blocks, 256, 0, L.stream>>>(g, n, inv_scale, found_inf);
  L.check("unscale_check");
}

// 16 B read of p, g, m, v and 12 B... (28 B moved per parameter: 16 read + 12 written); grid = multiple of 148 SMs
__global__ void __launch_bounds__(256) adam_kernel(float* __restrict__ p, const float* __restrict__ g, float* __restrict__ m, float* __restrict__ v,
                                                   size_t n, float lr, float b1, float b2, float eps, float c1, float c2,
                                                   const int* __restrict__ skip) {
  if (skip && *skip) return;
  const size_t n4 = n / 4;
  auto upd = [&](float& pp, float gg, float& mm, float& vv) {
    mm = fmaf(b1, mm, (1.f - b1) * gg);
    vv = fmaf(b2, vv, (1.f - b2) * gg * gg);
    const float mh = mm / c1, vh = vv / c2;
    pp -= lr * mh / (sqrtf(vh) + eps);
  };
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
    float4 P = reinterpret_cast<float4*>(p)[i], M = reinterpret_cast<float4*>(m)[i], V = reinterpret_cast<float4*>(v)[i];
    const float4 G = __ldg(reinterpret_cast<const float4*>(g) + i);
    upd(P.x, G.x, M.x, V.x); upd(P.y, G.y, M.y, V.y); upd(P.z, G.z, M.z, V.z); upd(P.w, G.w, M.w, V.w);
    reinterpret_cast<float4*>(p)[i] = P; reinterpret_cast<float4*>(m)[i] = M; reinterpret_cast<float4*>(v)[i] = V;
  }
  if (blockIdx.x == 0 && threadIdx.x < (n & 3)) {
    const size_t i = n4 * 4 + threadIdx.x;
    float P = p[i], M = m[i], V = v[i];
    upd(P, g[i], M, V);
    p[i] = P; m[i] = M; v[i] = V;
  }
}

void adam(Launcher& L, float* p, const float* g, float* m, float* v, size_t n, float lr, float b1, float b2, float eps, float c1,
          float c2, const int* skip) {
  if (n == 0) return;
  const int blocks = (int)std::min<size_t>((n / 4 + 255) / 256 + 1, 148 * 8);
  adam_kernel<<<blocks, 256, 0, L.stream>>>(p, g, m, v, n, lr, b1, b2, eps, c1, c2, skip);
  L.check("adam");
}

// =============================================================================================================
// critic (a7-a9): fp32, batch-major activations; contractions through sgemm, the rest warp-level elementwise
// =============================================================================================================
__global__ void bias_tanh_kernel(float* __restrict__ a, const float* __restrict__ bias, int rows, int cols) {
  const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (i >= (size_t)rows * cols) return;
  a[i] = tanhf(a[i] + bias[i % cols]);
}
__global__ void bias_add_kernel(float* __restrict__ a, const float* __restrict__ bias, int rows) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < rows) a[i] += bias[0];
}

// g: LD arrays [ld_rows][HD] (layer stride ld_rows*HD); D [rows]
void critic_forward(Launcher& L, const NetShape& s, const float* theta, const float* X, int rows, float* g, float* D) {
  if (rows <= 0) return;
  const float* in = X; int in_dim = s.in_dim;
  for (int l = 1; l <= s.L; ++l) {
    float* out = g + (size_t)(l - 1) * rows * s.H;
    sgemm(L, false, true, rows, s.H, in_dim, in, in_dim, 0, theta + s.W_off(l), in_dim, 0, out, s.H, 0, 1, false);
    bias_tanh_kernel<<<cdiv((size_t)rows * s.H, 256), 256, 0, L.stream>>>(out, theta + s.b_off(l), rows, s.H);
    L.check("bias_tanh");
    in = out; in_dim = s.H;
  }
  sgemm(L, false, true, rows, 1, s.H, in, s.H, 0, theta + s.W_off(s.L + 1), s.H, 0, D, 1, 0, 1, false);
  bias_add_kernel<<<cdiv(rows, 256), 256, 0, L.stream>>>(D, theta + s.b_off(s.L + 1), rows);
  L.check("bias_add");
}

// out = a * (1 - g*g)
__global__ void mul_s_kernel(const float* __restrict__ a, const float* __restrict__ g, float* __restrict__ out, size_t n) {
  const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (i < n) { const float gg = g[i]; out[i] = a[i] * (1.f - gg * gg); }
}
// out[j] += sum_n A[n][j]; block = 32 columns x 8 row groups (the batch is a few hundred rows: a serial loop per column was
// 8 us of dependent-latency per call)
__global__ void __launch_bounds__(256) colsum_acc_kernel(const float* __restrict__ A, int rows, int cols, float* __restrict__ out) {
  __shared__ float red[8][33];
  const int c = threadIdx.x & 31, rg = threadIdx.x >> 5, j = blockIdx.x * 32 + c;
  float s = 0.f;
  if (j < cols)
    for (int n = rg; n < rows; n += 8) s += A[(size_t)n * cols + j];
  red[rg][c] = s;
  __syncthreads();
  if (rg == 0 && j < cols) {
    float t = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) t += red[k][c];
    out[j] += t;
  }
}
// out[b][j] = seed[b] * w[j]
__global__ void outer_kernel(const float* __restrict__ seed, const float* __restrict__ w, int rows, int cols, float* __restrict__ out) {
  const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (i < (size_t)rows * cols) out[i] = seed[i / cols] * w[i % cols];
}

// Ordinary backprop of sum_b seed[b] D(X_b).  g: activations g^1..g^LD of these rows, layer stride g_layer_stride.
void critic_backward(Launcher& L, const NetShape& s, const float* theta, const float* X, const float* g, int rows, int g_layer_stride,
                     const float* seed, float* grads, float* dX, float* t0, float* t1) {
  if (rows <= 0) return;
  const int LD = s.L, HD = s.H;
  const float* gL = g + (size_t)(LD - 1) * g_layer_stride;
  if (grads) {
    // v_hat_out += seed^T g^LD ; c_hat_out += sum seed
    sgemm(L, true, false, 1, HD, rows, seed, 1, 0, gL, HD, 0, grads + s.W_off(LD + 1), HD, 0, 1, true);
    colsum_acc_kernel<<<1, 256, 0, L.stream>>>(seed, rows, 1, grads + s.b_off(LD + 1));
    L.check("colsum_acc");
  }
  float* ghat = t0; float* ahat = t1;
  outer_kernel<<<cdiv((size_t)rows * HD, 256), 256, 0, L.stream>>>(seed, theta + s.W_off(LD + 1), rows, HD, ghat);
  L.check("outer");
  for (int l = LD; l >= 1; --l) {
    const float* gl = g + (size_t)(l - 1) * g_layer_stride;
    const float* gprev = (l > 1) ? g + (size_t)(l - 2) * g_layer_stride : X;
    const int in_dim = (l > 1) ? HD : s.in_dim;
    mul_s_kernel<<<cdiv((size_t)rows * HD, 256), 256, 0, L.stream>>>(ghat, gl, ahat, (size_t)rows * HD);
    L.check("mul_s");
    if (grads) {
      sgemm(L, true, false, HD, in_dim, rows, ahat, HD, 0, gprev, in_dim, 0, grads + s.W_off(l), in_dim, 0, 1, true);
      colsum_acc_kernel<<<cdiv(HD, 32), 256, 0, L.stream>>>(ahat, rows, HD, grads + s.b_off(l));
      L.check("colsum_acc");
    }
    if (l > 1 || dX) {
      float* dst = (l > 1) ? ghat : dX;
      sgemm(L, false, false, rows, in_dim, HD, ahat, HD, 0, theta + s.W_off(l), in_dim, 0, dst, in_dim, 0, 1, false);
    }
  }
}

__global__ void bcast_rows_kernel(const float* __restrict__ w, int rows, int cols, float* __restrict__ out) {
  const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (i < (size_t)rows * cols) out[i] = w[i % cols];
}
// one warp per row: nu = ||G||, accumulate (nu-1)^2, seed = (lambda/B) 2 (nu-1)/nu G  (0 when nu == 0, reading G12)
__global__ void gp_norm_seed_kernel(const float* __restrict__ G, int B, int d, float lambda, float* __restrict__ nu_out,
                                    float* __restrict__ grad_norm, double* __restrict__ acc, float* __restrict__ seed) {
  const int b = blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32, lane = threadIdx.x & 31;
  if (b >= B) return;
  float s = 0.f;
  for (int j = lane; j < d; j += 32) { const float v = G[(size_t)b * d + j]; s = fmaf(v, v, s); }
  s = warp_sum(s);
  const float nu = sqrtf(s);
  if (lane == 0) {
    nu_out[b] = nu;
    if (grad_norm) grad_norm[b] = nu;
    atomicAdd(acc, (double)(nu - 1.f) * (double)(nu - 1.f));
  }
  if (seed) {
    const float k = nu > 0.f ? (lambda / B) * 2.f * (nu - 1.f) / nu : 0.f;
    for (int j = lane; j < d; j += 32) seed[(size_t)b * d + j] = k * G[(size_t)b * d + j];
  }
}
// ascending sweep elementwise: adj_s = adj_abar * gbar ; adj_gbar = adj_abar * s
__global__ void gp_ascend_kernel(const float* __restrict__ adj_abar, const float* __restrict__ gbar, const float* __restrict__ g,
                                 float* __restrict__ adj_s, float* __restrict__ adj_gbar, size_t n) {
  const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (i < n) { const float a = adj_abar[i], gg = g[i]; adj_s[i] = a * gbar[i]; adj_gbar[i] = a * (1.f - gg * gg); }
}
// descending sweep elementwise: adj_g += -2 g adj_s ; adj_a = adj_g * s
__global__ void gp_descend_kernel(float* __restrict__ adj_g, const float* __restrict__ g, const float* __restrict__ adj_s,
                                  float* __restrict__ adj_a, size_t n, int first) {
  const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (i < n) {
    const float gg = g[i];
    const float ag = (first ? 0.f : adj_g[i]) - 2.f * gg * adj_s[i];
    adj_a[i] = ag * (1.f - gg * gg);
  }
}

// O5 + O6.  g: activations g^1..g^LD of the xhat rows.
void critic_gp(Launcher& L, const NetShape& s, const float* theta, const float* Xhat, const float* g, int B, int g_layer_stride,
               float lambda, CriticWs& w, float* grads, float* grad_norm) {
  const int LD = s.L, HD = s.H, d = s.in_dim;
  const size_t wmax = (size_t)std::max(d, HD);
  auto gbar = [&](int l) { return w.gbar + (size_t)l * w.maxB * wmax; };
  auto abar = [&](int l) { return w.abar + (size_t)(l - 1) * w.maxB * HD; };
  auto adjs = [&](int l) { return w.adjs + (size_t)(l - 1) * w.maxB * HD; };
  auto gl = [&](int l) { return g + (size_t)(l - 1) * g_layer_stride; };
  const int nb = cdiv((size_t)B * HD, 256);
  // O5 backward-to-input
  bcast_rows_kernel<<<nb, 256, 0, L.stream>>>(theta + s.W_off(LD + 1), B, HD, gbar(LD));
  L.check("bcast_rows");
  for (int l = LD; l >= 1; --l) {
    const int in_dim = (l > 1) ? HD : d;
    mul_s_kernel<<<nb, 256, 0, L.stream>>>(gbar(l), gl(l), abar(l), (size_t)B * HD);
    L.check("mul_s");
    sgemm(L, false, false, B, in_dim, HD, abar(l), HD, 0, theta + s.W_off(l), in_dim, 0, gbar(l - 1), in_dim, 0, 1, false);
  }
  float* seed = grads ? w.t0 : nullptr;                       // adj(gbar^0), [B][d]
  gp_norm_seed_kernel<<<cdiv(B, 8), 256, 0, L.stream>>>(gbar(0), B, d, lambda, w.nu, grad_norm, w.acc + 2, seed);
  L.check("gp_norm_seed");
  if (!grads) return;
  // O6 ascending sweep
  float* adj_gbar = w.t0; float* adj_abar = w.t1; float* spare = w.t2;
  for (int l = 1; l <= LD; ++l) {
    const int in_dim = (l > 1) ? HD : d;
    // adj(abar^l) = adj(gbar^{l-1}) V_l^T
    sgemm(L, false, true, B, HD, in_dim, adj_gbar, in_dim, 0, theta + s.W_off(l), in_dim, 0, adj_abar, HD, 0, 1, false);
    // V_hat_l += abar^l^T adj(gbar^{l-1})
    sgemm(L, true, false, HD, in_dim, B, abar(l), HD, 0, adj_gbar, in_dim, 0, grads + s.W_off(l), in_dim, 0, 1, true);
    gp_ascend_kernel<<<nb, 256, 0, L.stream>>>(adj_abar, gbar(l), gl(l), adjs(l), spare, (size_t)B * HD);
    L.check("gp_ascend");
    std::swap(adj_gbar, spare);                               // adj(gbar^l) now lives in adj_gbar
  }
  // v_hat_out += sum_b adj(gbar^LD)
  colsum_acc_kernel<<<cdiv(HD, 32), 256, 0, L.stream>>>(adj_gbar, B, HD, grads + s.W_off(LD + 1));
  L.check("colsum_acc");
  // O6 descending sweep (adj_g in adj_gbar's buffer is free now: reuse t-buffers)
  float* adj_g = adj_gbar; float* adj_a = adj_abar;
  for (int l = LD; l >= 1; --l) {
    const int in_dim = (l > 1) ? HD : d;
    const float* gprev = (l > 1) ? gl(l - 1) : Xhat;
    gp_descend_kernel<<<nb, 256, 0, L.stream>>>(adj_g, gl(l), adjs(l), adj_a, (size_t)B * HD, l == LD ? 1 : 0);
    L.check("gp_descend");
    sgemm(L, true, false, HD, in_dim, B, adj_a, HD, 0, gprev, in_dim, 0, grads + s.W_off(l), in_dim, 0, 1, true);
    colsum_acc_kernel<<<cdiv(HD, 32), 256, 0, L.stream>>>(adj_a, B, HD, grads + s.b_off(l));
    L.check("colsum_acc");
    if (l > 1) sgemm(L, false, false, B, HD, HD, adj_a, HD, 0, theta + s.W_off(l), HD, 0, adj_g, HD, 0, 1, false);
  }
}

// X = [fake; real; eps*real + (1-eps)*fake]
__global__ void build_snapshots_kernel(const float* __restrict__ fake, const float* __restrict__ real, const float* __restrict__ eps, int B,
                                       int d, float* __restrict__ X) {
  const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (i >= (size_t)B * d) return;
  const float f = fake[i], r = real[i], e = eps[i / d];
  X[i] = f; X[(size_t)B * d + i] = r; X[2 * (size_t)B * d + i] = e * r + (1.f - e) * f;
}
void build_snapshots(Launcher& L, const float* fake, const float* real, const float* eps, int B, int d, float* X) {
  build_snapshots_kernel<<<cdiv((size_t)B * d, 256), 256, 0, L.stream>>>(fake, real, eps, B, d, X);
  L.check("build_snapshots");
}
// seed[0..B) = +1/B (fake rows), seed[B..2B) = -1/B (real rows)
__global__ void fill_seed_kernel(float* seed, int B) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < 2 * B) seed[i] = (i < B ? 1.f : -1.f) / B;
}
void fill_seed(Launcher& L, float* seed, int B) {
  fill_seed_kernel<<<cdiv(2 * B, 256), 256, 0, L.stream>>>(seed, B);
  L.check("fill_seed");
}
// acc[0] = sum D[0..B), acc[1] = sum D[B..2B)
__global__ void reduce_scores_kernel(const float* __restrict__ D, int B, double* __restrict__ acc) {
  double s = 0.0;
  const float* p = D + (size_t)blockIdx.x * B;
  for (int i = threadIdx.x; i < B; i += 32) s += p[i];
  s = warp_sum_d(s);
  if (threadIdx.x == 0) acc[blockIdx.x] = s;
}
void reduce_scores(Launcher& L, const float* D, int B, double* acc) {
  reduce_scores_kernel<<<2, 32, 0, L.stream>>>(D, B, acc);
  L.check("reduce_scores");
}
// losses[6] = {L_D, mean D(fake), mean D(real), GP, L_G, L_pde}; gp_out / meansq_out serve the single-op entry points
__global__ void write_losses_kernel(const double* __restrict__ acc, int N, long long NP, float lambda, float w_pde, float* losses,
                                    float* gp_out, float* meansq_out, long long meansq_count) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const double gp = N > 0 ? lambda * acc[2] / N : 0.0;
  if (gp_out) *gp_out = (float)gp;
  if (meansq_out) *meansq_out = (float)(meansq_count > 0 ? acc[3] / meansq_count : 0.0);
  if (losses) {
    const double df = acc[0] / N, dr = acc[1] / N, lp = acc[3] / NP;
    losses[0] = (float)(df - dr + gp); losses[1] = (float)df; losses[2] = (float)dr; losses[3] = (float)gp;
    losses[4] = (float)(-df + w_pde * lp); losses[5] = (float)lp;
  }
}
void write_losses(Launcher& L, const double* acc, int N, long long NP, float lambda, float w_pde, float* losses, float* gp_out,
                  float* meansq_out, long long meansq_count) {
  write_losses_kernel<<<1, 32, 0, L.stream>>>(acc, N, NP, lambda, w_pde, losses, gp_out, meansq_out, meansq_count);
  L.check("write_losses");
}

// sensor rows r = (n, s) <-> snapshot entries X[n][col0 + s]  (log k and u at the sensors, concatenated)
__global__ void scatter_snapshot_kernel(const float* __restrict__ o, long long row0, int valid, int S, int d, int col0, float* __restrict__ X) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= valid) return;
  const long long rg = row0 + r;
  X[(rg / S) * d + col0 + (rg % S)] = o[r];
}
void scatter_snapshot(Launcher& L, const float* o, long long row0, int valid, int S, int d, int col0, float* X) {
  if (valid <= 0) return;
  scatter_snapshot_kernel<<<cdiv(valid, 256), 256, 0, L.stream>>>(o, row0, valid, S, d, col0, X);
  L.check("scatter_snapshot");
}
__global__ void scatter_free_kernel(const float* __restrict__ fvals, const float* __restrict__ xy, long long row0, int valid, int F, int d, int col0,
                                    float* __restrict__ X) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= valid) return;
  const long long rg = row0 + r;
  float* row = X + (rg / F) * d + col0 + (rg % F);
  row[0] = fvals[r]; row[F] = xy[2 * rg]; row[2 * F] = xy[2 * rg + 1];
}
void scatter_free(Launcher& L, const float* fvals, const float* xy_free, long long row0, int valid, int F, int d, int col0, float* X) {
  if (valid <= 0) return;
  scatter_free_kernel<<<cdiv(valid, 256), 256, 0, L.stream>>>(fvals, xy_free, row0, valid, F, d, col0, X);
  L.check("scatter_snapshot");
}
__global__ void gather_seed_kernel(const float* __restrict__ dX, long long row0, int valid, int R, int S, int d, int col0, float alpha,
                                   float* __restrict__ seed, float* __restrict__ amax) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  float v = 0.f;
  if (r < R) {
    const long long rg = row0 + r;
    v = r < valid ? alpha * dX[(rg / S) * d + col0 + (rg % S)] : 0.f;
    seed[r] = v;
  }
  if (amax) {
    float m = fabsf(v);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) { if (!(m <= 3.0e38f)) m = INFINITY; atomicMax(reinterpret_cast<int*>(amax), __float_as_int(m)); }
  }
}
void gather_seed(Launcher& L, const float* dX, long long row0, int valid, int R, int S, int d, int col0, float alpha, float* seed, float* amax) {
  if (R <= 0) return;
  gather_seed_kernel<<<cdiv(R, 256), 256, 0, L.stream>>>(dX, row0, valid, R, S, d, col0, alpha, seed, amax);
  L.check("gather_seed");
}

}  // namespace pigan
