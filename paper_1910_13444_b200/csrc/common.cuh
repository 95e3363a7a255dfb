// Internal declarations shared by the translation units of libpigan.so (not part of the C-ABI).
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

#include "pigan.h"

namespace pigan {

// ---- flat parameter packing (include/pigan.h): W_l [out][in] then b_l [out], l = 1..L+1 ----------------------
struct NetShape {
  int in_dim, L, H;
  int heads = 1;                                                 // outputs of the last layer: 1 (plain MLP) or 2 (shared trunk: log k, u)
  __host__ __device__ size_t first_size() const { return (size_t)H * in_dim + H; }
  __host__ __device__ size_t W_off(int l) const {              // l is 1-based
    if (l == 1) return 0;
    return first_size() + (size_t)(l - 2) * ((size_t)H * H + H);
  }
  __host__ __device__ size_t b_off(int l) const {
    if (l == 1) return (size_t)H * in_dim;
    if (l <= L) return W_off(l) + (size_t)H * H;
    return W_off(l) + (size_t)heads * H;                       // output layer: w_out [heads][H], then b_out [heads]
  }
  __host__ __device__ size_t count() const { return first_size() + (size_t)(L - 1) * ((size_t)H * H + H) + (size_t)heads * (H + 1); }
};

template <typename T> __device__ __forceinline__ float to_f(T v);
template <> __device__ __forceinline__ float to_f<float>(float v) { return v; }
template <> __device__ __forceinline__ float to_f<__half>(__half v) { return __half2float(v); }
template <typename T> __device__ __forceinline__ T from_f(float v);
template <> __device__ __forceinline__ float from_f<float>(float v) { return v; }
template <> __device__ __forceinline__ __half from_f<__half>(float v) { return __float2half_rn(v); }

// ---- the tanh jet chain rule and its adjoint (O4); C = 1, 3 or 5 channels ------------------
// forward: a[0] already holds the value pre-activation (bias added); a[1..] the derivative pre-activations.
template <int C>
__device__ __forceinline__ void jet_act_fwd(float t, const float* a, float* h) {
  const float s = 1.f - t * t;
  h[0] = t;
  if (C >= 3) { h[1] = s * a[1]; h[2] = s * a[2]; }
  if (C >= 5) {
    const float q = -2.f * t * s;
    h[3] = fmaf(s, a[3], q * a[1] * a[1]);
    h[4] = fmaf(s, a[4], q * a[2] * a[2]);
  }
}
// adjoint, written in the layer's OUTPUT jet h = (t, h_x, h_y, h_xx, h_yy) -- no pre-activation derivatives are kept.
// With s = 1 - t^2, q = -2ts, q' = -2s(1 - 3t^2) and h_x = s a_x, h_xx = s a_xx + q a_x^2, O4 becomes
//   q a_x = -2t h_x,   q a_xx + q' a_x^2 = -2t h_xx - 2 h_x^2   (substitute s a_xx = h_xx - q a_x^2), so
//   ahat_xx = s hhat_xx;  ahat_x = s hhat_x - 4t h_x hhat_xx;
//   ahat = s hhat - 2t (h_x hhat_x + h_y hhat_y + h_xx hhat_xx + h_yy hhat_yy) - 2 (h_x^2 hhat_xx + h_y^2 hhat_yy).
// hh = adjoints of h_c; aa = adjoints of a_c.
template <int C>
__device__ __forceinline__ void jet_act_bwd(const float* h, const float* hh, float* aa) {
  const float t = h[0], s = 1.f - t * t;
  float v = s * hh[0];
  if (C >= 3) {
    const float m2t = -2.f * t;
    v = fmaf(m2t, fmaf(h[1], hh[1], h[2] * hh[2]), v);
    aa[1] = s * hh[1];
    aa[2] = s * hh[2];
    if (C >= 5) {
      v = fmaf(m2t, fmaf(h[3], hh[3], h[4] * hh[4]), v);
      v = fmaf(-2.f, fmaf(h[1] * h[1], hh[3], h[2] * h[2] * hh[4]), v);
      aa[1] = fmaf(2.f * m2t * h[1], hh[3], aa[1]);
      aa[2] = fmaf(2.f * m2t * h[2], hh[4], aa[2]);
      aa[3] = s * hh[3];
      aa[4] = s * hh[4];
    }
  }
  aa[0] = v;
}

// ---- block scaling of the 16-bit adjoint planes -----------------------------------------------------------------
// The output adjoints of a chunk are multiplied by 2^(8-e), e = exponent of their largest magnitude (amax = m 2^e,
// m in [0.5, 1)), so that the adjoint planes sit in the middle of the fp16 range whatever 1/(N P) and loss_scale are;
// every reduction of adjoints into an fp32 gradient multiplies by the exact inverse.  amax == nullptr (fp32 mode): 1.
__device__ __forceinline__ int adj_exponent(const float* amax) {
  if (!amax) return 8;
  const float a = *amax;
  if (!(a > 0.f) || !isfinite(a)) return 8;
  int e;
  frexpf(a, &e);
  return min(max(e, -100), 100);
}
__device__ __forceinline__ float adj_scale(const float* amax) { return ldexpf(1.f, 8 - adj_exponent(amax)); }
__device__ __forceinline__ float adj_inv_scale(const float* amax) { return ldexpf(1.f, adj_exponent(amax) - 8); }

// ---- launch bookkeeping -------------------------------------------------------------------------------------
struct Launcher {
  cudaStream_t stream = nullptr;
  int device = 0;              // the CUDA device the owning context was created on
  int num_sms = 148;           // multiprocessors of that device
  bool one_cta = false;        // PIGAN_FLAG_ONE_CTA: never take the CTA-pair kernels
  unsigned long long count = 0;
  cudaError_t err = cudaSuccess;
  const char* where = "";
  // optional per-launch CUDA-event trace (pigan_profile_*): one event after every launch on the launch stream;
  // the duration of launch i is event_i - event_{i-1} (the stream is kept busy, so gaps are launch latency only).
  bool profiling = false;
  std::vector<cudaEvent_t> events;
  std::vector<const char*> names;
  size_t n_rec = 0;
  void check(const char* w) {
    ++count;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess && err == cudaSuccess) { err = e; where = w; }
    if (profiling) mark(w);
  }
  void mark(const char* w) {
    if (n_rec == events.size()) { cudaEvent_t ev; cudaEventCreate(&ev); events.push_back(ev); names.push_back(w); }
    names[n_rec] = w;
    cudaEventRecord(events[n_rec++], stream);
  }
};

// cudaFuncAttributeMaxDynamicSharedMemorySize is per (function, device): remember which devices were opted in
template <typename K>
inline void ensure_smem_attr(const Launcher& L, K kern, int bytes, unsigned long long& done_mask) {
  const unsigned long long bit = 1ull << (L.device & 63);
  if (!(done_mask & bit)) { cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes); done_mask |= bit; }
}

// ---- SIMT kernels (simt_kernels.cu) ---------------------------------------------------------------------------
// C[M x N] (ldc) = or += alpha * op(A)[M x K] op(B)[K x N], batched (batch index adds sA/sB/sC), fp32.
//   TA: A stored [K][M] (lda) else [M][K];  TB: B stored [N][K] (ldb) else [K][N].
//   accumulate: atomicAdd into C (C must be initialised) -- also used when the K range is split.
void sgemm(Launcher& L, bool TA, bool TB, int M, int N, int K, const float* A, int lda, long long sA, const float* B,
           int ldb, long long sB, float* C, int ldc, long long sC, int batch, bool accumulate, float alpha = 1.f);

struct ChunkGeom {          // one chunk of generator rows r = row0 .. row0+valid-1 ; row -> (n, p) = (r / npts, r % npts)
  long long row0;           // first global row of the chunk
  int valid;                // rows of the chunk that exist (<= R)
  int R;                    // rows computed (valid rounded up to the row tile)
  int R_ld;                 // leading dimension (rows) of every plane
  int npts;                 // points per latent sample
  int per_sample = 0;       // NEXT-2: every sample has its own points, xy is [n][npts][2] (row r reads xy[r]); else xy is [npts][2] shared
};

template <typename T>
void first_layer_fwd(Launcher& L, int C, const NetShape& s, const float* theta, const float* Zp, const float* xy,
                     const ChunkGeom& g, T* h1, bool split = false);   // split: C = 1, writes planes (hi, lo)
void jet_act_fwd_f32(Launcher& L, int C, int H, const float* bias, const ChunkGeom& g, const float* apre, float* h);
template <typename T>
void out_fwd(Launcher& L, int C, int H, const float* w_out, const float* b_out, const ChunkGeom& g, const T* hL,
             float* o, long long o_plane_stride, bool split = false);          // split: C = 1, sums planes (hi, lo)
// f may be null (target 0); ext_seed (may be null) [R]: an additional adjoint of r per row, already loss-scaled (NEXT-2: -dD/df / N)
void residual(Launcher& L, const float* Y, long long y_stride, const float* U, long long u_stride, const float* f,
              long long row0, int valid, int R, int npts, float* r_out, double* sum_sq, float seed_scale, float* seedY,
              float* seedU, int seed_ld, float* amaxY = nullptr, float* amaxU = nullptr, const float* ext_seed = nullptr);
// NEXT-2: X[n][col0 + p] = fvals[(n, p)], X[n][col0 + F + p] = x, X[n][col0 + 2F + p] = y for the chunk's rows
void scatter_free(Launcher& L, const float* fvals, const float* xy_free, long long row0, int valid, int F, int d, int col0, float* X);
// adjoint of one tanh layer: hh_c = (hhat planes) or (w_out[j] * ohat_c[r]) ; writes ahat planes, accumulates
// b_hat_l[j] += sum_r ahat_0 (and for the output layer w_hat_out[j], b_hat_out).
template <typename T>
void jet_act_bwd_launch(Launcher& L, int C, int H, const ChunkGeom& g, const float* hhat /*or null*/,
                        const float* w_out, const float* ohat /*[C][R_ld] when hhat null*/, const T* h /*[C][H][R_ld]*/, T* ahat,
                        float* g_bias, float* g_wout, float* g_bout, const float* amax);
template <typename T>
void first_layer_bwd(Launcher& L, int C, const NetShape& s, const float* xy, const ChunkGeom& g, const T* ahat,
                     float* gW1 /* flat grads base of this net */, float* An /*[N][H]*/, const float* amax);
void finalize_first_layer(Launcher& L, const NetShape& s, int N, const float* An, const float* z, float* grads);
// fp32 mode, H = 32 / 64 (gen_fused_f32.cu): the whole generator pass of a chunk in one kernel (a warp per row)
bool gen_fused_f32_supported(const NetShape& s);
void gen_fused_f32_fwd(Launcher& L, int C, const NetShape& s, const float* theta, const float* Zp, const float* xy, const ChunkGeom& g, float* o,
                       long long o_stride);
void gen_fused_f32_bwd(Launcher& L, int C, const NetShape& s, const float* theta, const float* Zp, const float* xy, const ChunkGeom& g,
                       const float* ohat /*[C][R_ld]*/, float* grads, float* An);
// NEXT-1 (shared trunk, two heads, skip connections): see gen_kernels.cu
template <typename T>
void top_act_bwd2(Launcher& L, int C, int H, const ChunkGeom& g, const float* w_out /*[2][H]*/, const float* ohat0, const float* ohat1, const T* h,
                  const T* tjet, T* ahat, T* sk_out, float* g_bias, float* g_wout /*[2][H]*/, float* g_bout /*[2]*/, const float* amax);
template <typename T> void plane_add(Launcher& L, int C, int H, const ChunkGeom& g, const T* a, const T* b, T* out);
template <typename T>
void skip_adj(Launcher& L, int C, int H, const ChunkGeom& g, const T* hh, const T* sk_in, const T* tjet, T* ahat, T* sk_out, float* g_bias, const float* amax);
void unscale_and_check(Launcher& L, float* g, size_t n, float inv_scale, int* found_inf);
void adam(Launcher& L, float* p, const float* g, float* m, float* v, size_t n, float lr, float b1, float b2, float eps,
          float c1, float c2, const int* skip);

// critic (always fp32; activations are batch-major [rows][width])
struct CriticWs {
  float* X = nullptr;       // [3B][d]   fake, real, xhat
  float* g = nullptr;       // (LD) x [3B][HD]   g^1..g^LD
  float* D = nullptr;       // [3B]
  float* t0 = nullptr;      // scratch [3B][max(d,HD)]
  float* t1 = nullptr;      // scratch [3B][max(d,HD)]
  float* t2 = nullptr;      // scratch [3B][max(d,HD)]
  float* gbar = nullptr;    // (LD+1) x [B][max(d,HD)]  gbar^0..gbar^LD  (gp)
  float* abar = nullptr;    // (LD) x [B][HD]           abar^1..abar^LD
  float* adjs = nullptr;    // (LD) x [B][HD]           adj(s^l)
  float* nu = nullptr;      // [B]
  double* acc = nullptr;    // [8] accumulators: 0 sum D fake, 1 sum D real, 2 sum (nu-1)^2, 3 sum r^2
  int maxB = 0;
  // fused path (critic_fused.cu): per-row factors of the weight gradients, V_hat_l = A_l^T B_l
  float* cfA = nullptr;     // [LD][4B][HD]
  float* cfB1 = nullptr;    // [4B][d]
  float* cfBh = nullptr;    // [LD][4B][HD]
};
bool critic_fused_supported(const NetShape& s);
void critic_fused(Launcher& L, const NetShape& s, const float* theta, const float* fake, const float* real, const float* eps, int B, int plain,
                  float lambda, CriticWs& w, float* grads, float* dX, float* grad_norm);
void critic_forward(Launcher& L, const NetShape& s, const float* theta, const float* X, int rows, float* g, float* D);
// plain backprop of sum_b seed[b] D(X_b) over `rows` rows starting at activations g; accumulates into grads if non-null;
// writes d/dX into dX if non-null.
void critic_backward(Launcher& L, const NetShape& s, const float* theta, const float* X, const float* g, int rows,
                     int ld_rows, const float* seed, float* grads, float* dX, float* t0, float* t1);
void critic_gp(Launcher& L, const NetShape& s, const float* theta, const float* Xhat, const float* g /*of xhat rows*/,
               int B, int g_layer_stride, float lambda, CriticWs& w, float* grads /*may be null*/, float* grad_norm);
void build_snapshots(Launcher& L, const float* fake, const float* real, const float* eps, int B, int d, float* X);
void fill_seed(Launcher& L, float* seed, int B);
void scatter_snapshot(Launcher& L, const float* o, long long row0, int valid, int S, int d, int col0, float* X);
void gather_seed(Launcher& L, const float* dX, long long row0, int valid, int R, int S, int d, int col0, float alpha, float* seed, float* amax);
void reduce_scores(Launcher& L, const float* D, int B, double* acc);
void write_losses(Launcher& L, const double* acc, int N, long long NP, float lambda, float w_pde, float* losses, float* gp_out,
                  float* meansq_out, long long meansq_count);

// ---- tensor-core kernels (tc_kernels.cu), 16-bit modes -------------------------------------------------------
struct TcPlan;   // opaque: tensor maps + 16-bit weight copies for one (net, chunk buffer set)
bool tc_supported(int H, std::string* why);
// Converts W_l (l = 2..L) of one net to 16-bit: w16[(l-2)*2+0] = W_l [out][in], w16[(l-2)*2+1] = W_l^T [in][out].
void tc_convert_weights(Launcher& L, int precision, const NetShape& s, const float* theta, void* w16);
// Output layer (a4) fused into the epilogue of the LAST hidden layer's forward: o_c[r] += sum_j w_out[j] h^L_c[j][r]
// (+ b_out on the value channel).  o must be zero on entry; h_out may then be nullptr (forward-only callers).
struct OutDot { const float* w_out; const float* b_out; float* o; long long o_stride; int valid; };
bool tc_out_dot_fusable(const Launcher& L, int H);
// hidden layer l forward: h_in [C][H][R_ld] -> h_out [C][H][R_ld]   (fused tanh-jet epilogue)
// linear: plain GEMM out_c = W in_c (no bias, no tanh) -- the raw adjoint planes hhat = W^T ahat of a skip layer (NEXT-1)
// reverse: sweep the row tiles last-to-first (CTA-pair kernels; alternating it layer by layer keeps a layer's first reads in L2)
void tc_layer_fwd(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* w16_l, const float* bias,
                  const void* h_in, void* h_out, const OutDot* od = nullptr, bool linear = false, bool reverse = false);
void tc_layer_fwd_split(Launcher& L, int precision, int H, int R, int R_ld, const void* w16_l, const float* bias, const void* h_in, void* h_out,
                        const OutDot* od = nullptr);
// dgrad of layer l with the adjoint of layer l-1's tanh fused: ahat_in (layer l) -> ahat_out (layer l-1)
struct FirstLayerFuse;
void tc_layer_bwd(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* w16T_l, const void* ahat_in,
                  const void* h_prev /*[C][H][R_ld]*/, void* ahat_out, float* g_bias_prev, const float* amax,
                  const FirstLayerFuse* fl = nullptr);
// wgrad of layer l: gW [H][H] += sum_c ahat_c h_prev_c^T   (fp32 atomics)
void tc_wgrad(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* ahat, const void* h_prev, float* gW, const float* amax);


// first-layer backward fused into the dgrad of layer 2 (CTA-pair kernels only): the adjoint planes ahat^1 are reduced
// in the epilogue into W_hat_1[:, 0:2], An and b_hat_1 and never written.  Valid when npts % 64 == 0 and R == valid.
struct FirstLayerFuse {
  const float* xy; long long row0; int npts; int in_dim; float* gW1; float* An; int per_sample = 0;
};
bool tc_first_layer_fusable(int H, const ChunkGeom& g);

// ---- the same four on CTA pairs (tc2_kernels.cu, cta_group::2), taken when tc2_supported(H) ---------------------
bool tc2_supported(const Launcher& L, int H);
void tc2_layer_fwd(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* w16_l, const float* bias,
                   const void* h_in, void* h_out, const OutDot* od, bool linear, bool reverse);
void tc2_layer_fwd_split(Launcher& L, int precision, int H, int R, int R_ld, const void* w16_l, const float* bias, const void* h_in, void* h_out,
                         const OutDot* od);
void tc2_layer_bwd(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* w16T_l, const void* ahat_in,
                   const void* h_prev, void* ahat_out, float* g_bias_prev, const float* amax, const FirstLayerFuse* fl);
void tc2_wgrad(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* ahat, const void* h_prev, float* gW, const float* amax);

// ---- width 128: first layer and every hidden layer of a chunk's forward in ONE kernel (tc_fused_fwd.cu) -----------------
// h[l - 1] receives the planes of h^l (l = 1 .. L); w16[l - 2] is the 16-bit copy of W_l.  Collocation rows only (C = 3, 5).
bool tc_fused_fwd_supported(const Launcher& L, const NetShape& s, int C, const ChunkGeom& g);
// od (may be null): the output layer rides in the last layer's epilogue (od->o zeroed by the caller; every row of the chunk is valid)
void tc_fused_fwd(Launcher& L, int precision, int C, const NetShape& s, const float* theta, const void* const* w16, const float* Zp,
                  const float* xy, const ChunkGeom& g, void* const* h, const OutDot* od);

// ---- widths 128 / 256: wgrad and dgrad (+ adjoint epilogue) of one layer in ONE kernel ---------------------------------
// (tc_fused_bwd.cu: width 128 on one CTA; tc2_fused_bwd.cu: width 256 on CTA pairs)
// gW (W_hat_l) += sum_c ahat_c h_prev_c^T and ahat_out = J^T (W_l^T ahat_in), b_hat_{l-1} += ...; the planes ahat_in and h_prev
// cross HBM once instead of twice.  fl != nullptr: layer 2 with the first-layer reduction (no ahat_out).
bool tc_fused_bwd_supported(const Launcher& L, int H, int C);
void tc_fused_bwd(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* w16T_l, const void* ahat_in, const void* h_prev,
                  void* ahat_out, float* gW, float* g_bias_prev, const float* amax, const FirstLayerFuse* fl);
bool tc2_fused_bwd_supported(const Launcher& L, int H, int C);
void tc2_fused_bwd(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* w16T_l, const void* ahat_in, const void* h_prev,
                   void* ahat_out, float* gW, float* g_bias_prev, const float* amax, const FirstLayerFuse* fl);

}  // namespace pigan
