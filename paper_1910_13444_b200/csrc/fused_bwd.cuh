// Shared by the two fused reverse-sweep kernels (tc2_fused_bwd.cu: width 256 on CTA pairs; tc_fused_bwd.cu: width 128 on one
// CTA): parameters and the epilogue of one warp.  Both kernels tile the rows by 32, hold the previous layer's output jet
// h^{l-1} of the CTA's 128 in units as an "H box" in shared memory ([channel][unit][32 rows], planes of 8 KB, 64-byte
// swizzle: the operand layout of the weight-gradient MMA), and give epilogue warp (q, hs) the units [32 q, 32 q + 32)
// (TMEM lanes) x rows [16 hs, 16 hs + 16) of the tile.
#pragma once
#include "tc_ptx.cuh"

namespace pigan {

constexpr int kFRows = 32;                   // rows of a tile
constexpr int kFEpiWarps = 8;
constexpr int kFThreads = (4 + kFEpiWarps) * 32;

struct FusedParams {
  int H;                 // width (128: one CTA, 256: CTA pair)
  int n_tiles;           // R / 32
  float* gW;             // W_hat_l [H][H] fp32, += (scaled back by the block scale of the adjoint planes)
  float* g_bias;         // b_hat_{l-1} [H]
  void* out;             // MODE 1: ahat^{l-1} planes [C][H][R_ld]
  int R_ld;
  const float* amax;     // block-scale source of the adjoint planes
  // MODE 3 (layer 2: the adjoint of the FIRST tanh layer is reduced here and never written; npts % 32 == 0)
  const float* xy; long long row0; int npts, in_dim, per_sample;
  float* gW1; float* An;
};

// One epilogue warp, one tile.  hh = this lane's D1 values (hhat^{l-1} of its unit, 16 rows per channel); box = the H box.
// Applies O4 written in the output jet (jet_act_bwd); MODE 1: writes ahat^{l-1} in place into the box and copies it out
// (two lanes cover the 32 contiguous bytes -- one sector -- of one unit's 16 rows; every lane pulls its share into registers,
// orders its generic-proxy accesses before the next TMA write of the box with fence.proxy.async, and only then issues the
// global stores); MODE 3: reduces the first-layer gradients.  The caller arrives on the box's free barrier afterwards.
template <typename T, int C, int MODE>
__device__ __forceinline__ void fused_epi_tile(const FusedParams& p, const float (&hh)[C][16], uint8_t* box, int q, int hs, int lane,
                                               int unit0 /*global unit of box unit 0*/, int row0 /*chunk row of this warp's first row*/,
                                               float inv_amax, float& bias_tot, float& sx, float& sy) {
  const int ul = q * 32 + lane;
  const uint32_t swz = (uint32_t)((lane >> 1) & 3);          // 64B swizzle: 16-byte chunk ^= (unit >> 1) & 3
  uint8_t* my_row = box + ul * 64;
  float bias_acc = 0.f;
  const long long grow = p.row0 + row0;                      // MODE 3: global row of this warp's first row
  const float2* xyp = MODE == 3 ? reinterpret_cast<const float2*>(p.xy) + (p.per_sample ? grow : grow % p.npts) : nullptr;
#pragma unroll
  for (int hf = 0; hf < 2; ++hf) {
    const uint32_t off = (((uint32_t)(hs * 2 + hf)) ^ swz) << 4;
    float hp[C][8], o[C][8];
#pragma unroll
    for (int c = 0; c < C; ++c) unpack8<T>(lds128(my_row + c * 8192 + off), hp[c]);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      float hx[5], hj[5], aa[5];
#pragma unroll
      for (int c = 0; c < C; ++c) { hx[c] = hh[c][hf * 8 + i]; hj[c] = hp[c][i]; }
      jet_act_bwd<C>(hj, hx, aa);
      bias_acc += aa[0];
      if (MODE == 3) {
        const float2 pt = __ldg(xyp + hf * 8 + i);           // same address in every lane: one broadcast load
        sx = fmaf(aa[0], pt.x, sx); sy = fmaf(aa[0], pt.y, sy);
        if (C >= 3) { sx += aa[1]; sy += aa[2]; }
      }
#pragma unroll
      for (int c = 0; c < C; ++c) o[c][i] = aa[c];
    }
    if (MODE == 1) {
#pragma unroll
      for (int c = 0; c < C; ++c) sts128(my_row + c * 8192 + off, pack8<T>(o[c]));
    }
  }
  bias_tot += bias_acc;
  if (MODE == 1) {
    __syncwarp();
    T* gout = reinterpret_cast<T*>(p.out);
    const int half = lane & 1, uu = lane >> 1;
    uint4 v[C][2];
#pragma unroll
    for (int c = 0; c < C; ++c)
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int u = q * 32 + j * 16 + uu;
        v[c][j] = lds128(box + c * 8192 + u * 64 + ((((uint32_t)(hs * 2 + half)) ^ (uint32_t)((u >> 1) & 3)) << 4));
      }
    fence_proxy_async();
#pragma unroll
    for (int c = 0; c < C; ++c)
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int u = unit0 + q * 32 + j * 16 + uu;
        *reinterpret_cast<uint4*>(gout + ((size_t)c * p.H + u) * p.R_ld + row0 + half * 8) = v[c][j];
      }
  } else {
    fence_proxy_async();                                     // generic reads of the H box before the next TMA write
    atomicAdd(p.An + (size_t)(grow / p.npts) * p.H + unit0 + ul, bias_acc * inv_amax);
  }
}

// accumulator columns [0, ncols) of this lane's TMEM row -> dst[0 .. ncols) += (fp32 vector reductions)
__device__ __forceinline__ void fused_drain(uint32_t taddr, float* dst, int ncols, float scale) {
#pragma unroll 2
  for (int n = 0; n < ncols; n += 8) {
    float v[8];
    tmem_ld8(taddr + n, v);
    tmem_ld_wait();
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] *= scale;
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst + n), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]) : "memory");
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst + n + 4), "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7]) : "memory");
  }
}

}  // namespace pigan
