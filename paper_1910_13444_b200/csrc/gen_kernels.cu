// Generator-side SIMT kernels (HBM-bound): first layer (S8a a1/a2), output dot (a4), adjoint of a tanh layer in SIMT form
// (top layer in every mode, all layers in fp32 mode; O4), first-layer backward.  Planes are [channel][unit][row]; every
// thread owns 8 consecutive rows of one unit, so all plane accesses are 16-byte (16-bit modes) or 32-byte (fp32) vectors
// and a warp touches 512 contiguous bytes per plane.
#include "common.cuh"

namespace pigan {

static inline int cdiv(long long a, long long b) { return (int)((a + b - 1) / b); }

template <typename T> __device__ __forceinline__ void load8(const T* p, float* v);
template <> __device__ __forceinline__ void load8<float>(const float* p, float* v) {
  const float4 a = *reinterpret_cast<const float4*>(p), b = *reinterpret_cast<const float4*>(p + 4);
  v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
}
template <> __device__ __forceinline__ void load8<__half>(const __half* p, float* v) {
  const uint4 u = *reinterpret_cast<const uint4*>(p);
  const __half2* h = reinterpret_cast<const __half2*>(&u);
#pragma unroll
  for (int i = 0; i < 4; ++i) { const float2 f = __half22float2(h[i]); v[2 * i] = f.x; v[2 * i + 1] = f.y; }
}
template <typename T> __device__ __forceinline__ void store8(T* p, const float* v);
template <> __device__ __forceinline__ void store8<float>(float* p, const float* v) {
  *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
  *reinterpret_cast<float4*>(p + 4) = make_float4(v[4], v[5], v[6], v[7]);
}
template <> __device__ __forceinline__ void store8<__half>(__half* p, const float* v) {
  uint4 u;
  __half2* h = reinterpret_cast<__half2*>(&u);
#pragma unroll
  for (int i = 0; i < 4; ++i) h[i] = __floats2half2_rn(v[2 * i], v[2 * i + 1]);
  *reinterpret_cast<uint4*>(p) = u;
}

__device__ __forceinline__ float tanh_approx(float x) {
  float y;
  asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float warp_sum_f(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
// sums `v` over the 256 threads of the block; result valid in thread 0
__device__ __forceinline__ float block_sum_256(float v, float* red /*[8]*/) {
  v = warp_sum_f(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  float s = 0.f;
  if (threadIdx.x == 0) for (int w = 0; w < 8; ++w) s += red[w];
  return s;
}

// =============================================================================================================
// first layer: a = Zp[n] + b1 + W1[:,0] x + W1[:,1] y ; a_x = W1[:,0], a_y = W1[:,1], a_xx = a_yy = 0 ; tanh jet.  fp32 math.
// block = 256 rows x 32 units: lane -> 8 rows, warp w -> units w, w+8, w+16, w+24 of the block's group
// =============================================================================================================
template <typename T, int C, bool SPLIT>
__global__ void __launch_bounds__(256) first_layer_fwd_kernel(NetShape s, const float* __restrict__ theta, const float* __restrict__ Zp,
                                                              const float* __restrict__ xy, ChunkGeom g, T* __restrict__ h1) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int r0 = blockIdx.x * 256 + lane * 8;
  if (r0 >= g.R) return;
  float x[8], y[8]; int n[8];
  {
    // one 64-bit division per thread; the 8 rows then step through (n, p) incrementally.  Padded rows repeat the
    // last valid row (finite values).
    const long long rg0 = g.row0 + min(r0, g.valid - 1);
    int nn = (int)(rg0 / g.npts), p = (int)(rg0 - (long long)nn * g.npts);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      n[i] = nn;
      const float2 q = *reinterpret_cast<const float2*>(xy + 2 * (g.per_sample ? (long long)nn * g.npts + p : (long long)p));
      x[i] = q.x; y[i] = q.y;
      if (r0 + i + 1 < g.valid) { if (++p == g.npts) { p = 0; ++nn; } }
    }
  }
  const bool one_sample = n[0] == n[7];
  const float* W1 = theta; const float* b1 = theta + s.b_off(1);
  const size_t plane = (size_t)s.H * g.R_ld;
  for (int j = blockIdx.y * 32 + warp; j < min(s.H, blockIdx.y * 32 + 32); j += 8) {
    const float wx = W1[(size_t)j * s.in_dim], wy = W1[(size_t)j * s.in_dim + 1], bj = b1[j];
    const float z0 = Zp[(size_t)n[0] * s.H + j];
    float o[C][8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const float zp = one_sample ? z0 : Zp[(size_t)n[i] * s.H + j];
      const float a0 = zp + bj + wx * x[i] + wy * y[i];
      float a[5] = {a0, wx, wy, 0.f, 0.f}, h[5];
      // 16-bit planes round t to 2^-11 anyway: tanh.approx there (R4); fp32 mode and the split snapshot path stay exact
      jet_act_fwd<C>((sizeof(T) == 2 && !SPLIT) ? tanh_approx(a0) : tanhf(a0), a, h);
#pragma unroll
      for (int c = 0; c < C; ++c) o[c][i] = h[c];
    }
#pragma unroll
    for (int c = 0; c < C; ++c) store8<T>(h1 + c * plane + (size_t)j * g.R_ld + r0, o[c]);
    if (SPLIT) {                                             // second plane: what the 16-bit rounding of t dropped
      float lo[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) lo[i] = o[0][i] - to_f<T>(from_f<T>(o[0][i]));
      store8<T>(h1 + plane + (size_t)j * g.R_ld + r0, lo);
    }
  }
}

template <typename T>
void first_layer_fwd(Launcher& L, int C, const NetShape& s, const float* theta, const float* Zp, const float* xy, const ChunkGeom& g, T* h1, bool split) {
  if (g.R <= 0) return;
  dim3 grid(cdiv(g.R, 256), cdiv(s.H, 32));
  if (split) first_layer_fwd_kernel<T, 1, true><<<grid, 256, 0, L.stream>>>(s, theta, Zp, xy, g, h1);
  else if (C == 1) first_layer_fwd_kernel<T, 1, false><<<grid, 256, 0, L.stream>>>(s, theta, Zp, xy, g, h1);
  else if (C == 3) first_layer_fwd_kernel<T, 3, false><<<grid, 256, 0, L.stream>>>(s, theta, Zp, xy, g, h1);
  else first_layer_fwd_kernel<T, 5, false><<<grid, 256, 0, L.stream>>>(s, theta, Zp, xy, g, h1);
  L.check("first_layer_fwd");
}
template void first_layer_fwd<float>(Launcher&, int, const NetShape&, const float*, const float*, const float*, const ChunkGeom&, float*, bool);
template void first_layer_fwd<__half>(Launcher&, int, const NetShape&, const float*, const float*, const float*, const ChunkGeom&, __half*, bool);

// =============================================================================================================
// output layer (a4): o_c[r] = w_out . h_c[:, r] (+ b_out on the value channel)
// block = 256 rows x (H / gridDim.y) units; warp w strides over the block's units; cross-warp sum in smem; one
// atomicAdd per (channel, row) per block (o is zeroed by the launcher)
// =============================================================================================================
template <typename T, int C, bool SPLIT>
__global__ void __launch_bounds__(256) out_fwd_kernel(int H, const float* __restrict__ w_out, const float* __restrict__ b_out, ChunkGeom g,
                                                      const T* __restrict__ hL, float* __restrict__ o, long long o_stride) {
  __shared__ float red[8][C][256];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int seg = blockIdx.x * 256, r0 = seg + lane * 8;
  const int per = (H + gridDim.y - 1) / gridDim.y, jb = blockIdx.y * per, je = min(H, jb + per);
  const size_t plane = (size_t)H * g.R_ld;
  float acc[C][8];
#pragma unroll
  for (int c = 0; c < C; ++c)
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[c][i] = 0.f;
  if (r0 < g.R) {
#pragma unroll 2
    for (int j = jb + warp; j < je; j += 8) {
      const float w = __ldg(w_out + j);
#pragma unroll
      for (int c = 0; c < C; ++c) {
        float v[8];
        load8<T>(hL + c * plane + (size_t)j * g.R_ld + r0, v);
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[c][i] = fmaf(w, v[i], acc[c][i]);
      }
    }
  }
#pragma unroll
  for (int c = 0; c < C; ++c)
#pragma unroll
    for (int i = 0; i < 8; ++i) red[warp][c][lane * 8 + i] = acc[c][i];
  __syncthreads();
  const int r = seg + threadIdx.x;
  if (r < g.valid) {
    if (SPLIT) {                                             // planes (hi, lo) of one value channel
      float sum = 0.f;
#pragma unroll
      for (int w = 0; w < 8; ++w) sum += red[w][0][threadIdx.x] + red[w][C - 1][threadIdx.x];
      if (blockIdx.y == 0) sum += b_out[0];
      atomicAdd(o + r, sum);
    } else {
#pragma unroll
      for (int c = 0; c < C; ++c) {
        float sum = 0.f;
#pragma unroll
        for (int w = 0; w < 8; ++w) sum += red[w][c][threadIdx.x];
        if (c == 0 && blockIdx.y == 0) sum += b_out[0];
        atomicAdd(o + c * o_stride + r, sum);
      }
    }
  }
}

template <typename T>
void out_fwd(Launcher& L, int C, int H, const float* w_out, const float* b_out, const ChunkGeom& g, const T* hL, float* o, long long o_plane_stride,
             bool split) {
  if (g.valid <= 0) return;
  cudaMemset2DAsync(o, (size_t)o_plane_stride * 4, 0, (size_t)g.valid * 4, split ? 1 : C, L.stream);
  const int rb = cdiv(g.R, 256);
  int jsplit = std::max(1, std::min(cdiv(600, rb), H / 8));
  dim3 grid(rb, jsplit);
  if (split) out_fwd_kernel<T, 2, true><<<grid, 256, 0, L.stream>>>(H, w_out, b_out, g, hL, o, o_plane_stride);
  else if (C == 1) out_fwd_kernel<T, 1, false><<<grid, 256, 0, L.stream>>>(H, w_out, b_out, g, hL, o, o_plane_stride);
  else if (C == 3) out_fwd_kernel<T, 3, false><<<grid, 256, 0, L.stream>>>(H, w_out, b_out, g, hL, o, o_plane_stride);
  else out_fwd_kernel<T, 5, false><<<grid, 256, 0, L.stream>>>(H, w_out, b_out, g, hL, o, o_plane_stride);
  L.check("out_fwd");
}
template void out_fwd<float>(Launcher&, int, int, const float*, const float*, const ChunkGeom&, const float*, float*, long long, bool);
template void out_fwd<__half>(Launcher&, int, int, const float*, const float*, const ChunkGeom&, const __half*, float*, long long, bool);

// =============================================================================================================
// adjoint of one tanh layer (O4), SIMT form.  block = one unit x 2048 rows (8 rows per thread).
//   hh_c = hhat_c[j][r] (fp32 planes from sgemm) or w_out[j] * ohat_c[r] (output layer).
//   writes ahat planes; b_hat_l[j] += sum_r ahat_0 ; output layer also w_hat_out[j] += sum_{c,r} ohat_c h_c, b_hat_out += sum ohat_0
// =============================================================================================================
template <typename T, int C>
__global__ void __launch_bounds__(256) jet_act_bwd_kernel(int H, ChunkGeom g, const float* __restrict__ hhat, const float* __restrict__ w_out,
                                                          const float* __restrict__ ohat, const T* __restrict__ h, T* __restrict__ ahat,
                                                          float* __restrict__ g_bias, float* __restrict__ g_wout, float* __restrict__ g_bout,
                                                          const float* __restrict__ amax) {
  __shared__ float red[8];
  const int j = blockIdx.y;
  const size_t plane = (size_t)H * g.R_ld;
  const float sc = adj_scale(amax), inv_sc = adj_inv_scale(amax);     // block scale of the adjoint planes (1 in fp32 mode)
  const float wj = w_out ? w_out[j] * sc : 0.f;
  float s_bias = 0.f, s_wout = 0.f, s_bout = 0.f;
  const int r0 = blockIdx.x * 2048 + threadIdx.x * 8;
  if (r0 < g.R) {
    const size_t off = (size_t)j * g.R_ld + r0;
    float hv[C][8], hh[C][8], o[C][8];
#pragma unroll
    for (int c = 0; c < C; ++c) load8<T>(h + c * plane + off, hv[c]);
    if (hhat) {
#pragma unroll
      for (int c = 0; c < C; ++c) load8<float>(hhat + c * plane + off, hh[c]);
    } else {
#pragma unroll
      for (int c = 0; c < C; ++c) {
        float ov[8];
        load8<float>(ohat + (size_t)c * g.R_ld + r0, ov);
#pragma unroll
        for (int i = 0; i < 8; ++i) { hh[c][i] = wj * ov[i]; s_wout = fmaf(ov[i], hv[c][i], s_wout); if (c == 0) s_bout += ov[i]; }
      }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      float hx[5], hj[5], aa[5];
#pragma unroll
      for (int c = 0; c < C; ++c) { hx[c] = hh[c][i]; hj[c] = hv[c][i]; }
      jet_act_bwd<C>(hj, hx, aa);
      s_bias += aa[0];
#pragma unroll
      for (int c = 0; c < C; ++c) o[c][i] = aa[c];
    }
#pragma unroll
    for (int c = 0; c < C; ++c) store8<T>(ahat + c * plane + off, o[c]);
  }
  float v = block_sum_256(s_bias, red);
  if (threadIdx.x == 0) atomicAdd(g_bias + j, v * inv_sc);
  if (g_wout) { v = block_sum_256(s_wout, red); if (threadIdx.x == 0) atomicAdd(g_wout + j, v); }
  if (g_bout && j == 0) { v = block_sum_256(s_bout, red); if (threadIdx.x == 0) atomicAdd(g_bout, v); }
}


// Output-layer form of the same adjoint (hh_c = w_out[j] * ohat_c[r]): a block owns 2048 rows x kTopUnits units and keeps
// the C x 8 output adjoints of its rows in registers across the unit loop, so per unit it only streams the h planes in
// and the ahat planes out (the generic kernel above re-read ohat for every unit: 3x the bytes through L2).
constexpr int kTopUnits = 16;
template <typename T, int C>
__global__ void __launch_bounds__(256) top_act_bwd_kernel(int H, ChunkGeom g, const float* __restrict__ w_out, const float* __restrict__ ohat,
                                                          const T* __restrict__ h, T* __restrict__ ahat, float* __restrict__ g_bias,
                                                          float* __restrict__ g_wout, float* __restrict__ g_bout, const float* __restrict__ amax) {
  __shared__ float red[kTopUnits][2];
  __shared__ float red8[8];
  const int lane = threadIdx.x & 31;
  const int jb = blockIdx.y * kTopUnits, je = min(H, jb + kTopUnits);
  const size_t plane = (size_t)H * g.R_ld;
  const float sc = adj_scale(amax), inv_sc = adj_inv_scale(amax);
  if (threadIdx.x < kTopUnits * 2) (&red[0][0])[threadIdx.x] = 0.f;
  __syncthreads();
  const int r0 = blockIdx.x * 2048 + threadIdx.x * 8;
  const bool active = r0 < g.R;
  float ov[C][8];
  float s_bout = 0.f;
#pragma unroll
  for (int c = 0; c < C; ++c) {
    if (active) load8<float>(ohat + (size_t)c * g.R_ld + r0, ov[c]);
    else {
#pragma unroll
      for (int i = 0; i < 8; ++i) ov[c][i] = 0.f;
    }
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) s_bout += ov[0][i];
  for (int j = jb; j < je; ++j) {
    float s_bias = 0.f, s_wout = 0.f;
    if (active) {
      const float wj = w_out[j] * sc;
      const size_t off = (size_t)j * g.R_ld + r0;
      float hv[C][8], o[C][8];
#pragma unroll
      for (int c = 0; c < C; ++c) load8<T>(h + c * plane + off, hv[c]);
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        float hx[5], hj[5], aa[5];
#pragma unroll
        for (int c = 0; c < C; ++c) { hx[c] = wj * ov[c][i]; hj[c] = hv[c][i]; s_wout = fmaf(ov[c][i], hv[c][i], s_wout); }
        jet_act_bwd<C>(hj, hx, aa);
        s_bias += aa[0];
#pragma unroll
        for (int c = 0; c < C; ++c) o[c][i] = aa[c];
      }
#pragma unroll
      for (int c = 0; c < C; ++c) store8<T>(ahat + c * plane + off, o[c]);
    }
    s_bias = warp_sum_f(s_bias); s_wout = warp_sum_f(s_wout);
    if (lane == 0) { atomicAdd(&red[j - jb][0], s_bias); atomicAdd(&red[j - jb][1], s_wout); }
  }
  __syncthreads();
  if (threadIdx.x < je - jb) {
    atomicAdd(g_bias + jb + threadIdx.x, red[threadIdx.x][0] * inv_sc);
    atomicAdd(g_wout + jb + threadIdx.x, red[threadIdx.x][1]);
  }
  if (blockIdx.y == 0) { const float v = block_sum_256(s_bout, red8); if (threadIdx.x == 0) atomicAdd(g_bout, v); }
}

template <typename T>
void jet_act_bwd_launch(Launcher& L, int C, int H, const ChunkGeom& g, const float* hhat, const float* w_out, const float* ohat, const T* h,
                        T* ahat, float* g_bias, float* g_wout, float* g_bout, const float* amax) {
  if (g.R <= 0) return;
  if (!hhat) {
    dim3 tgrid(cdiv(g.R, 2048), cdiv(H, kTopUnits));
#define PIGAN_TOP(c) top_act_bwd_kernel<T, c><<<tgrid, 256, 0, L.stream>>>(H, g, w_out, ohat, h, ahat, g_bias, g_wout, g_bout, amax)
    if (C == 1) PIGAN_TOP(1); else if (C == 3) PIGAN_TOP(3); else PIGAN_TOP(5);
#undef PIGAN_TOP
    L.check("jet_act_bwd");
    return;
  }
  dim3 grid(cdiv(g.R, 2048), H);
#define PIGAN_BWD(c) jet_act_bwd_kernel<T, c><<<grid, 256, 0, L.stream>>>(H, g, hhat, w_out, ohat, h, ahat, g_bias, g_wout, g_bout, amax)
  if (C == 1) PIGAN_BWD(1); else if (C == 3) PIGAN_BWD(3); else PIGAN_BWD(5);
#undef PIGAN_BWD
  L.check("jet_act_bwd");
}
template void jet_act_bwd_launch<float>(Launcher&, int, int, const ChunkGeom&, const float*, const float*, const float*, const float*, float*, float*, float*, float*, const float*);
template void jet_act_bwd_launch<__half>(Launcher&, int, int, const ChunkGeom&, const float*, const float*, const float*, const __half*, __half*, float*, float*, float*, const float*);

// =============================================================================================================
// first-layer backward (O4 'First layer'): W_hat_1[:,0] += sum (ahat x + ahat_x), W_hat_1[:,1] += sum (ahat y + ahat_y),
// An[n][j] += sum_{p in chunk} ahat[j][(n,p)]  (the z-part GEMM and b_hat_1 use An / the layer-1 adjoint reduction).
// block = one unit x 2048 rows
// =============================================================================================================
template <typename T, int C>
__global__ void __launch_bounds__(256) first_layer_bwd_kernel(NetShape s, const float* __restrict__ xy, ChunkGeom g, const T* __restrict__ ahat,
                                                              float* __restrict__ gW1, float* __restrict__ An, const float* __restrict__ amax) {
  __shared__ float red[8];
  const int j = blockIdx.y;
  const size_t plane = (size_t)s.H * g.R_ld;
  const float inv_sc = adj_inv_scale(amax);
  const int b0 = blockIdx.x * 2048, r0 = b0 + threadIdx.x * 8;
  const int n_first = (int)((g.row0 + b0) / g.npts), n_last = (int)((g.row0 + min(b0 + 2047, g.valid - 1)) / g.npts);
  const bool uniform = n_first == n_last;                   // the whole block lies inside one latent sample
  float sx = 0.f, sy = 0.f, sa = 0.f;
  if (r0 < g.valid) {
    const size_t off = (size_t)j * g.R_ld + r0;
    float a0[8], ax[8], ay[8];
    load8<T>(ahat + off, a0);
    if (C >= 3) { load8<T>(ahat + plane + off, ax); load8<T>(ahat + 2 * plane + off, ay); }
    int run_n = -1; float run = 0.f;
    // one 64-bit division per thread; the 8 rows then step through (n, p) incrementally
    const long long rg0 = g.row0 + r0;
    int n = (int)(rg0 / g.npts), p = (int)(rg0 - (long long)n * g.npts);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      if (r0 + i < g.valid) {
        const float2 q = *reinterpret_cast<const float2*>(xy + 2 * (g.per_sample ? (long long)n * g.npts + p : (long long)p));
        sx = fmaf(a0[i], q.x, sx); sy = fmaf(a0[i], q.y, sy);
        if (C >= 3) { sx += ax[i]; sy += ay[i]; }
        if (uniform) sa += a0[i];
        else {
          if (n != run_n) { if (run_n >= 0) atomicAdd(An + (size_t)run_n * s.H + j, run * inv_sc); run_n = n; run = 0.f; }
          run += a0[i];
        }
        if (++p == g.npts) { p = 0; ++n; }
      }
    }
    if (!uniform && run_n >= 0) atomicAdd(An + (size_t)run_n * s.H + j, run * inv_sc);
  }
  float v = block_sum_256(sx, red);
  if (threadIdx.x == 0) atomicAdd(gW1 + (size_t)j * s.in_dim, v * inv_sc);
  v = block_sum_256(sy, red);
  if (threadIdx.x == 0) atomicAdd(gW1 + (size_t)j * s.in_dim + 1, v * inv_sc);
  if (uniform) { v = block_sum_256(sa, red); if (threadIdx.x == 0) atomicAdd(An + (size_t)n_first * s.H + j, v * inv_sc); }
}

template <typename T>
void first_layer_bwd(Launcher& L, int C, const NetShape& s, const float* xy, const ChunkGeom& g, const T* ahat, float* gW1, float* An, const float* amax) {
  if (g.valid <= 0) return;
  dim3 grid(cdiv(g.valid, 2048), s.H);
  if (C == 1) first_layer_bwd_kernel<T, 1><<<grid, 256, 0, L.stream>>>(s, xy, g, ahat, gW1, An, amax);
  else if (C == 3) first_layer_bwd_kernel<T, 3><<<grid, 256, 0, L.stream>>>(s, xy, g, ahat, gW1, An, amax);
  else first_layer_bwd_kernel<T, 5><<<grid, 256, 0, L.stream>>>(s, xy, g, ahat, gW1, An, amax);
  L.check("first_layer_bwd");
}
template void first_layer_bwd<float>(Launcher&, int, const NetShape&, const float*, const ChunkGeom&, const float*, float*, float*, const float*);
template void first_layer_bwd<__half>(Launcher&, int, const NetShape&, const float*, const ChunkGeom&, const __half*, float*, float*, const float*);



// =============================================================================================================
// NEXT-1: shared-trunk generator with two output heads and skip connections.
// The trunk reuses the layer kernels; what is new is elementwise and lives here:
//   top_act_bwd2   adjoint of the last tanh layer seeded by BOTH heads: hhat_c = w_k[j] Yhat_c[r] + w_u[j] uhat_c[r]
//   plane_add      h^l = t^l + h^{l-2}                                   (skip connection, forward)
//   skip_adj       hhat_total = hhat + skip adjoint; ahat = J^T hhat_total (O4 on t^l); hands hhat_total on to h^{l-2}
// =============================================================================================================
template <typename T, int C>
__global__ void __launch_bounds__(256) top_act_bwd2_kernel(int H, ChunkGeom g, const float* __restrict__ w_out /*[2][H]*/,
                                                           const float* __restrict__ ohat0 /*[C0][R_ld]*/, const float* __restrict__ ohat1 /*[C][R_ld]*/,
                                                           const T* __restrict__ h, const T* __restrict__ tjet, T* __restrict__ ahat,
                                                           T* __restrict__ sk_out, float* __restrict__ g_bias, float* __restrict__ g_wout /*[2][H]*/,
                                                           float* __restrict__ g_bout /*[2]*/, const float* __restrict__ amax) {
  constexpr int C0 = C >= 3 ? 3 : 1;                          // log k carries (value, x, y); its xx, yy adjoints are zero (O3)
  __shared__ float red[kTopUnits][3];
  __shared__ float red8[8];
  const int lane = threadIdx.x & 31;
  const int jb = blockIdx.y * kTopUnits, je = min(H, jb + kTopUnits);
  const size_t plane = (size_t)H * g.R_ld;
  const float sc = adj_scale(amax), inv_sc = adj_inv_scale(amax);
  if (threadIdx.x < kTopUnits * 3) (&red[0][0])[threadIdx.x] = 0.f;
  __syncthreads();
  const int r0 = blockIdx.x * 2048 + threadIdx.x * 8;
  const bool active = r0 < g.R;
  float o0[C0][8], o1[C][8];
#pragma unroll
  for (int c = 0; c < C; ++c) {
    if (active) { load8<float>(ohat1 + (size_t)c * g.R_ld + r0, o1[c]); if (c < C0) load8<float>(ohat0 + (size_t)c * g.R_ld + r0, o0[c]); }
    else {
#pragma unroll
      for (int i = 0; i < 8; ++i) { o1[c][i] = 0.f; if (c < C0) o0[c][i] = 0.f; }
    }
  }
  float sb0 = 0.f, sb1 = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) { sb0 += o0[0][i]; sb1 += o1[0][i]; }
  for (int j = jb; j < je; ++j) {
    float s_bias = 0.f, s_w0 = 0.f, s_w1 = 0.f;
    if (active) {
      const float w0 = w_out[j] * sc, w1 = w_out[H + j] * sc;
      const size_t off = (size_t)j * g.R_ld + r0;
      float hv[C][8], tv[C][8], o[C][8], hh[C][8];
#pragma unroll
      for (int c = 0; c < C; ++c) { load8<T>(h + c * plane + off, hv[c]); load8<T>(tjet + c * plane + off, tv[c]); }
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        float hx[5], hj[5], aa[5];
#pragma unroll
        for (int c = 0; c < C; ++c) {
          hx[c] = w1 * o1[c][i]; s_w1 = fmaf(o1[c][i], hv[c][i], s_w1);
          if (c < C0) { hx[c] = fmaf(w0, o0[c][i], hx[c]); s_w0 = fmaf(o0[c][i], hv[c][i], s_w0); }
          hj[c] = tv[c][i]; hh[c][i] = hx[c];
        }
        jet_act_bwd<C>(hj, hx, aa);
        s_bias += aa[0];
#pragma unroll
        for (int c = 0; c < C; ++c) o[c][i] = aa[c];
      }
#pragma unroll
      for (int c = 0; c < C; ++c) { store8<T>(ahat + c * plane + off, o[c]); if (sk_out) store8<T>(sk_out + c * plane + off, hh[c]); }
    }
    s_bias = warp_sum_f(s_bias); s_w0 = warp_sum_f(s_w0); s_w1 = warp_sum_f(s_w1);
    if (lane == 0) { atomicAdd(&red[j - jb][0], s_bias); atomicAdd(&red[j - jb][1], s_w0); atomicAdd(&red[j - jb][2], s_w1); }
  }
  __syncthreads();
  if (threadIdx.x < je - jb) {
    atomicAdd(g_bias + jb + threadIdx.x, red[threadIdx.x][0] * inv_sc);
    atomicAdd(g_wout + jb + threadIdx.x, red[threadIdx.x][1]);
    atomicAdd(g_wout + H + jb + threadIdx.x, red[threadIdx.x][2]);
  }
  if (blockIdx.y == 0) {
    float v = block_sum_256(sb0, red8); if (threadIdx.x == 0) atomicAdd(g_bout, v);
    v = block_sum_256(sb1, red8); if (threadIdx.x == 0) atomicAdd(g_bout + 1, v);
  }
}

template <typename T>
void top_act_bwd2(Launcher& L, int C, int H, const ChunkGeom& g, const float* w_out, const float* ohat0, const float* ohat1, const T* h,
                  const T* tjet, T* ahat, T* sk_out, float* g_bias, float* g_wout, float* g_bout, const float* amax) {
  if (g.R <= 0) return;
  dim3 grid(cdiv(g.R, 2048), cdiv(H, kTopUnits));
#define PIGAN_TOP2(c) top_act_bwd2_kernel<T, c><<<grid, 256, 0, L.stream>>>(H, g, w_out, ohat0, ohat1, h, tjet, ahat, sk_out, g_bias, g_wout, g_bout, amax)
  if (C == 1) PIGAN_TOP2(1); else if (C == 3) PIGAN_TOP2(3); else PIGAN_TOP2(5);
#undef PIGAN_TOP2
  L.check("jet_act_bwd");
}
template void top_act_bwd2<float>(Launcher&, int, int, const ChunkGeom&, const float*, const float*, const float*, const float*, const float*, float*, float*, float*, float*, float*, const float*);
template void top_act_bwd2<__half>(Launcher&, int, int, const ChunkGeom&, const float*, const float*, const float*, const __half*, const __half*, __half*, __half*, float*, float*, float*, const float*);

// out_c = a_c + b_c on C planes [C][H][R_ld] (rows < R)
template <typename T>
__global__ void __launch_bounds__(256) plane_add_kernel(int n_planes_rows /* C*H */, int R, int R_ld, const T* __restrict__ a, const T* __restrict__ b,
                                                        T* __restrict__ out) {
  const int r0 = blockIdx.x * 2048 + threadIdx.x * 8;
  if (r0 >= R) return;
  for (int pj = blockIdx.y; pj < n_planes_rows; pj += gridDim.y) {
    const size_t off = (size_t)pj * R_ld + r0;
    float x[8], y[8];
    load8<T>(a + off, x); load8<T>(b + off, y);
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] += y[i];
    store8<T>(out + off, x);
  }
}
template <typename T>
void plane_add(Launcher& L, int C, int H, const ChunkGeom& g, const T* a, const T* b, T* out) {
  if (g.R <= 0) return;
  dim3 grid(cdiv(g.R, 2048), std::min(C * H, 1024));
  plane_add_kernel<T><<<grid, 256, 0, L.stream>>>(C * H, g.R, g.R_ld, a, b, out);
  L.check("skip_add");
}
template void plane_add<float>(Launcher&, int, int, const ChunkGeom&, const float*, const float*, float*);
template void plane_add<__half>(Launcher&, int, int, const ChunkGeom&, const __half*, const __half*, __half*);

// skip layers, reverse: total = hh (+ sk_in); sk_out = total (if the layer itself takes a skip); ahat = J^T(tjet) total; b_hat += sum ahat_0
template <typename T, int C>
__global__ void __launch_bounds__(256) skip_adj_kernel(int H, ChunkGeom g, const T* __restrict__ hh, const T* __restrict__ sk_in, const T* __restrict__ tjet,
                                                       T* __restrict__ ahat, T* __restrict__ sk_out, float* __restrict__ g_bias,
                                                       const float* __restrict__ amax) {
  __shared__ float red[8];
  const int j = blockIdx.y;
  const size_t plane = (size_t)H * g.R_ld;
  const float inv_sc = adj_inv_scale(amax);
  float s_bias = 0.f;
  const int r0 = blockIdx.x * 2048 + threadIdx.x * 8;
  if (r0 < g.R) {
    const size_t off = (size_t)j * g.R_ld + r0;
    float tv[C][8], tot[C][8], o[C][8];
#pragma unroll
    for (int c = 0; c < C; ++c) {
      load8<T>(tjet + c * plane + off, tv[c]);
      load8<T>(hh + c * plane + off, tot[c]);
      if (sk_in) {
        float s[8];
        load8<T>(sk_in + c * plane + off, s);
#pragma unroll
        for (int i = 0; i < 8; ++i) tot[c][i] += s[i];
      }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      float hx[5], hj[5], aa[5];
#pragma unroll
      for (int c = 0; c < C; ++c) { hx[c] = tot[c][i]; hj[c] = tv[c][i]; }
      jet_act_bwd<C>(hj, hx, aa);
      s_bias += aa[0];
#pragma unroll
      for (int c = 0; c < C; ++c) o[c][i] = aa[c];
    }
#pragma unroll
    for (int c = 0; c < C; ++c) { store8<T>(ahat + c * plane + off, o[c]); if (sk_out) store8<T>(sk_out + c * plane + off, tot[c]); }
  }
  const float v = block_sum_256(s_bias, red);
  if (threadIdx.x == 0) atomicAdd(g_bias + j, v * inv_sc);
}
template <typename T>
void skip_adj(Launcher& L, int C, int H, const ChunkGeom& g, const T* hh, const T* sk_in, const T* tjet, T* ahat, T* sk_out, float* g_bias, const float* amax) {
  if (g.R <= 0) return;
  dim3 grid(cdiv(g.R, 2048), H);
  if (C == 1) skip_adj_kernel<T, 1><<<grid, 256, 0, L.stream>>>(H, g, hh, sk_in, tjet, ahat, sk_out, g_bias, amax);
  else if (C == 3) skip_adj_kernel<T, 3><<<grid, 256, 0, L.stream>>>(H, g, hh, sk_in, tjet, ahat, sk_out, g_bias, amax);
  else skip_adj_kernel<T, 5><<<grid, 256, 0, L.stream>>>(H, g, hh, sk_in, tjet, ahat, sk_out, g_bias, amax);
  L.check("skip_adj");
}
template void skip_adj<float>(Launcher&, int, int, const ChunkGeom&, const float*, const float*, const float*, float*, float*, float*, const float*);
template void skip_adj<__half>(Launcher&, int, int, const ChunkGeom&, const __half*, const __half*, const __half*, __half*, __half*, float*, const float*);

}  // namespace pigan
