// Reverse sweep of ONE hidden layer of width 128 in ONE kernel on one CTA: the
// dgrad GEMM with the adjoint of the previous tanh in its epilogue AND the weight-gradient GEMM of the same layer, as
// tc2_fused_bwd.cu does for width 256 on CTA pairs.  One CTA holds everything, so the adjoint tile is loaded once and
// serves both GEMMs from the same shared-memory bytes:
//   box AT = ahat^l [channel][128 out units][32 rows] (planes of 8 KB, 64-byte swizzle), box H = h^{l-1} likewise.
//   MMA1 (dgrad)  D1[128 in units][(channel, row)] = W^T[128 x 128] . AT      A = W^T, K-major SW128, resident (32 KB);
//                 B = AT read MN-major (contraction over its units, N = 32 rows of each channel).
//   MMA2 (wgrad)  D2[128 out units][128 in units] += sum_{c, row} AT_c[out][row] H_c[in][row]
//                 A = AT read K-major (contraction over its rows), B = H, K-major.  D2 stays in TMEM over all tiles.
//   Epilogue: fused_epi_tile (fused_bwd.cuh).
// c2 (65536 rows per pass) is launch-chain bound: this halves the tensor-core launches of the reverse sweep and reads the
// adjoint and jet planes once instead of twice.
#include "fused_bwd.cuh"

namespace pigan {

constexpr int kF1WBytes = 2 * 128 * 64 * 2;  // resident W^T: 2 k-blocks of 128 units x 64 contraction elements
constexpr uint32_t kF1D1Col = 128;           // D2 = columns [0, 128), D1 = [128, 128 + 32 C)

template <int C> struct Fused1Cfg {
  static constexpr int kSlot = C * 8192;
  static constexpr int kNA = C == 5 ? 2 : C == 3 ? 3 : 4;      // AT boxes in flight
  static constexpr int kNH = C == 5 ? 2 : 4;                   // H boxes in flight (held until the epilogue has copied its tile out)
  static constexpr int kSmem = kF1WBytes + (kNA + kNH) * kSlot + 1024 /*align*/ + 256 /*barriers*/;
  static_assert(kSmem <= 232448, "shared memory budget");
};

template <typename T, int C, int MODE>
__global__ void __launch_bounds__(kFThreads, 1)
fused_bwd128_kernel(const __grid_constant__ CUtensorMap tmW,     // W_l^T [128 in][128 out] 16-bit, box 64 x 128, SW128
                    const __grid_constant__ CUtensorMap tmA,     // ahat^l planes, box 32 rows x 128 units x C, SW64
                    const __grid_constant__ CUtensorMap tmH,     // h^{l-1} planes, box 32 rows x 128 units x C, SW64
                    FusedParams p) {
  using Cfg = Fused1Cfg<C>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sW = smem;
  uint8_t* sA = sW + kF1WBytes;
  uint8_t* sH = sA + Cfg::kNA * Cfg::kSlot;
  uint64_t* bars = reinterpret_cast<uint64_t*>(sH + Cfg::kNH * Cfg::kSlot);
  uint64_t* wfull = bars;                       // [1]
  uint64_t* fullA = wfull + 1;                  // [kNA]
  uint64_t* emptyA = fullA + Cfg::kNA;          // [kNA]  2 arrivals: MMA1 and MMA2 of the tile have read the box
  uint64_t* fullH = emptyA + Cfg::kNA;          // [kNH]
  uint64_t* hfree = fullH + Cfg::kNH;           // [kNH]  8 arrivals: the epilogue warps have copied the tile out
  uint64_t* m2done = hfree + Cfg::kNH;          // [kNH]  MMA2 has read H box it % kNH (it runs at most kNH - 1 tiles ahead of the epilogue)
  uint64_t* tfull = m2done + Cfg::kNH;          // [1]    D1 of the tile is complete
  uint64_t* tempty = tfull + 1;                 // [1]    8 arrivals: D1 is in the epilogue warps' registers
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 1);

  const int warp = uniform_warp_idx(), lane = threadIdx.x & 31;
  const int cta = blockIdx.x, n_ctas = gridDim.x;

  if (warp == 0 && lane == 0) { prefetch_tmap(&tmW); prefetch_tmap(&tmA); prefetch_tmap(&tmH); }
  if (warp == 1 && lane == 0) {
    mbar_init(wfull, 1);
    for (int i = 0; i < Cfg::kNA; ++i) { mbar_init(fullA + i, 1); mbar_init(emptyA + i, 2); }
    for (int i = 0; i < Cfg::kNH; ++i) { mbar_init(fullH + i, 1); mbar_init(hfree + i, kFEpiWarps); mbar_init(m2done + i, 1); }
    mbar_init(tfull, 1); mbar_init(tempty, kFEpiWarps);
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot, 0);

  if (warp == 0) {
    // ===================== TMA producer: two load streams, each gated by its own consumers (see tc2_fused_bwd.cu) ==========
    if (elect_one()) {
      mbar_expect_tx(wfull, kF1WBytes);
      tma_load_2d(sW, &tmW, wfull, 0, 0);
      tma_load_2d(sW + kF1WBytes / 2, &tmW, wfull, 64, 0);
    }
    __syncwarp();
    const int n_my = (p.n_tiles - cta + n_ctas - 1) / n_ctas;
    int itA = 0, itH = 0;
    uint32_t spins = 0;
    while (itA < n_my || itH < n_my) {
      bool progress = false;
      if (itH < n_my) {
        const int s = itH % Cfg::kNH; const uint32_t ph = (uint32_t)(itH / Cfg::kNH) & 1;
        if (__all_sync(0xffffffffu, mbar_test_wait(hfree + s, ph ^ 1))) {
          if (elect_one()) {
            mbar_expect_tx(fullH + s, Cfg::kSlot);
            tma_load_3d(sH + s * Cfg::kSlot, &tmH, fullH + s, (cta + itH * n_ctas) * kFRows, 0, 0);
          }
          __syncwarp();
          ++itH; progress = true;
        }
      }
      if (itA < n_my) {
        const int s = itA % Cfg::kNA; const uint32_t ph = (uint32_t)(itA / Cfg::kNA) & 1;
        if (__all_sync(0xffffffffu, mbar_test_wait(emptyA + s, ph ^ 1))) {
          if (elect_one()) {
            mbar_expect_tx(fullA + s, Cfg::kSlot);
            tma_load_3d(sA + s * Cfg::kSlot, &tmA, fullA + s, (cta + itA * n_ctas) * kFRows, 0, 0);
          }
          __syncwarp();
          ++itA; progress = true;
        }
      }
      if (progress) spins = 0;
      else if (++spins > (1u << 26)) { if (lane == 0) printf("pigan: fused_bwd128 producer timed out (block %d)\n", (int)blockIdx.x); __trap(); }
    }
  } else if (warp == 1) {
    // ===================== MMA1 issuer: D1 = W^T ahat^l (contraction over the 128 out units, 8 k-steps) =====================
    constexpr uint32_t idesc1 = umma_idesc(Fmt<T>::umma, 0, 1, 128, 32 * C);
    const uint32_t d1 = tmem_base + kF1D1Col;
    const uint32_t aW = smem_u32(sW);
    mbar_wait(wfull, 0);
    int it = 0;
    for (int t = cta; t < p.n_tiles; t += n_ctas, ++it) {
      const int s = it % Cfg::kNA; const uint32_t ph = (uint32_t)(it / Cfg::kNA) & 1;
      mbar_wait(fullA + s, ph);
      mbar_wait(tempty, (uint32_t)(it & 1) ^ 1);            // the epilogue holds D1 of the previous tile in registers
      tc_fence_after();
      const uint32_t bA = smem_u32(sA + s * Cfg::kSlot);
      if (elect_one()) {
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
          // A: k-block ks / 4 (16 KB each), +32 B per 16 elements inside the 128-byte swizzle span
          // B (MN-major SW64): 32-row chunks (channels) 8 KB apart (LBO), 8-unit groups 512 B apart (SBO), 16 units = +1 KB
          tc_mma(d1, umma_desc_sw128(aW + (ks >> 2) * (kF1WBytes / 2) + (ks & 3) * 32, 16, 1024), umma_desc_sw64(bA + ks * 1024, 8192, 512), idesc1,
                 ks ? 1u : 0u);
        }
        tc_commit(emptyA + s);
        tc_commit(tfull);
      }
      __syncwarp();
    }
  } else if (warp == 3) {
    // ===================== MMA2 issuer: D2 += ahat^l h^{l-1 T} (contraction over the tile's 32 rows of every channel) ==========
    constexpr uint32_t idesc2 = umma_idesc(Fmt<T>::umma, 0, 0, 128, 128);
    const uint32_t d2 = tmem_base;
    int it = 0;
    for (int t = cta; t < p.n_tiles; t += n_ctas, ++it) {
      const int sa = it % Cfg::kNA; const uint32_t pa = (uint32_t)(it / Cfg::kNA) & 1;
      const int sh = it % Cfg::kNH; const uint32_t phh = (uint32_t)(it / Cfg::kNH) & 1;
      mbar_wait(fullA + sa, pa);
      mbar_wait(fullH + sh, phh);
      tc_fence_after();
      const uint32_t aA = smem_u32(sA + sa * Cfg::kSlot), bH = smem_u32(sH + sh * Cfg::kSlot);
      if (elect_one()) {
#pragma unroll
        for (int c = 0; c < C; ++c)
#pragma unroll
          for (int k = 0; k < 2; ++k)
            tc_mma(d2, umma_desc_sw64(aA + c * 8192 + k * 32, 16, 512), umma_desc_sw64(bH + c * 8192 + k * 32, 16, 512), idesc2, (it | c | k) ? 1u : 0u);
        tc_commit(emptyA + sa);
        tc_commit(m2done + sh);
      }
      __syncwarp();
    }
  } else if (warp >= 4) {
    // ===================== epilogue: warp (q, hs) owns TMEM lanes / in units [32 q, 32 q + 32) x rows [16 hs, 16 hs + 16) =====
    const int e = warp - 4, q = e & 3, hs = e >> 2;
    const int unit = q * 32 + lane;
    const uint32_t lane_base = tmem_base + ((uint32_t)(q * 32) << 16);
    const uint32_t tD1 = lane_base + kF1D1Col + hs * 16;     // D1 columns: [channel][32 rows]
    const float inv_amax = adj_inv_scale(p.amax);
    float bias_tot = 0.f, sx = 0.f, sy = 0.f;
    int it = 0;
    for (int t = cta; t < p.n_tiles; t += n_ctas, ++it) {
      const int sh = it % Cfg::kNH;
      const int row0 = t * kFRows + hs * 16;
      mbar_wait(tfull, (uint32_t)(it & 1));
      tc_fence_after();
      float hh[C][16];
#pragma unroll
      for (int c = 0; c < C; ++c) { tmem_ld8(tD1 + c * 32, hh[c]); tmem_ld8(tD1 + c * 32 + 8, hh[c] + 8); }
      tmem_ld_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(tempty);
      // MMA2 of this tile reads the H box this warp is about to overwrite in place
      mbar_wait(m2done + sh, (uint32_t)(it / Cfg::kNH) & 1);
      fused_epi_tile<T, C, MODE>(p, hh, sH + sh * Cfg::kSlot, q, hs, lane, 0, row0, inv_amax, bias_tot, sx, sy);
      __syncwarp();
      if (lane == 0) mbar_arrive(hfree + sh);
    }
    atomicAdd(p.g_bias + unit, bias_tot * inv_amax);
    if (MODE == 3) {
      atomicAdd(p.gW1 + (size_t)unit * p.in_dim, sx * inv_amax);
      atomicAdd(p.gW1 + (size_t)unit * p.in_dim + 1, sy * inv_amax);
    }
    // ---- D2 -> W_hat_l: every MMA of this CTA has retired (the last m2done) ----
    {
      const int last = it - 1;
      mbar_wait(m2done + last % Cfg::kNH, (uint32_t)(last / Cfg::kNH) & 1);
      tc_fence_after();
      fused_drain(lane_base + hs * 64, p.gW + (size_t)unit * 128 + hs * 64, 64, inv_amax);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) { tc_fence_after(); tmem_dealloc(tmem_base, 512); }
}

// =============================================================================================================
// host side
// =============================================================================================================
template <int C, int MODE>
static void launch_fused1(Launcher& L, const CUtensorMap& w, const CUtensorMap& a, const CUtensorMap& h, const FusedParams& p) {
  using Cfg = Fused1Cfg<C>;
  static unsigned long long attr_done = 0;
  auto kern = fused_bwd128_kernel<__half, C, MODE>;
  ensure_smem_attr(L, kern, Cfg::kSmem, attr_done);
  const int ctas = std::min(p.n_tiles, L.num_sms);
  kern<<<ctas, kFThreads, Cfg::kSmem, L.stream>>>(w, a, h, p);
  L.check("jet_layer_bwd_wgrad");
}

bool tc_fused_bwd_supported(const Launcher& L, int H, int C) {
  if (C != 1 && C != 3 && C != 5) return false;
  return H == 128 || tc2_fused_bwd_supported(L, H, C);
}

void tc_fused_bwd(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* w16T_l, const void* ahat_in, const void* h_prev,
                  void* ahat_out, float* gW, float* g_bias_prev, const float* amax, const FirstLayerFuse* fl) {
  if (R <= 0) return;
  if (H != 128) { tc2_fused_bwd(L, precision, C, H, R, R_ld, w16T_l, ahat_in, h_prev, ahat_out, gW, g_bias_prev, amax, fl); return; }
  CUtensorMap w, a, h;
  bool ok = weight_map(L, &w, precision, w16T_l, H) && plane_map(L, &a, precision, ahat_in, H, R_ld, C, 32, 128, C, CU_TENSOR_MAP_SWIZZLE_64B) &&
            plane_map(L, &h, precision, h_prev, H, R_ld, C, 32, 128, C, CU_TENSOR_MAP_SWIZZLE_64B);
  if (!ok) return;
  FusedParams p{};
  p.H = H; p.n_tiles = R / kFRows; p.gW = gW; p.g_bias = g_bias_prev; p.out = ahat_out; p.R_ld = R_ld; p.amax = amax;
  if (fl) {
    p.xy = fl->xy; p.row0 = fl->row0; p.npts = fl->npts; p.in_dim = fl->in_dim; p.gW1 = fl->gW1; p.An = fl->An; p.per_sample = fl->per_sample;
    if (C == 1) launch_fused1<1, 3>(L, w, a, h, p); else if (C == 3) launch_fused1<3, 3>(L, w, a, h, p); else launch_fused1<5, 3>(L, w, a, h, p);
    return;
  }
  if (C == 1) launch_fused1<1, 1>(L, w, a, h, p); else if (C == 3) launch_fused1<3, 1>(L, w, a, h, p); else launch_fused1<5, 1>(L, w, a, h, p);
}

}  // namespace pigan
