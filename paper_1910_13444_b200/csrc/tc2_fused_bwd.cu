// Reverse sweep of ONE hidden layer of width 256 in ONE kernel on CTA pairs:
// the dgrad GEMM with the adjoint of the previous tanh in its epilogue AND the weight-gradient GEMM of the same layer.
// Both read the adjoint planes ahat^l and the output jet h^{l-1}; layer by layer (tc2_kernels.cu) those planes cross
// HBM twice (5 C plane passes per layer: dgrad reads 2 C and writes C, wgrad reads 2 C), here once (3 C).  At width 256
// the layer is HBM-bound, so the plane passes are what the step pays for.
//
// Per tile of 32 rows (persistent, one CTA pair per tile, tiles strided over the pairs):
//   MMA1 (dgrad)  D1[256 in units][(channel, row)] = W^T[256 x 256] . ahat^l          A = W^T, K-major SW128, RESIDENT in
//                 shared memory for the whole launch (CTA r holds in units [128 r, 128 r + 128): 64 KB);
//                 B = ahat^l planes, MN-major SW32: CTA r supplies rows [16 r, 16 r + 16) of the tile for all 256 units
//                 and C channels (box "M1"); N = 32 C, accumulator columns [CTA half][channel][16 rows].
//   MMA2 (wgrad)  D2[256 out units][256 in units] += sum_{c, row} ahat^l_c[out][row] h^{l-1}_c[in][row]
//                 A = ahat^l, K-major SW64: CTA r supplies out units [128 r, +128) for all 32 rows (box "A2");
//                 B = h^{l-1}, K-major SW64: CTA r supplies in units [128 r, +128) for all 32 rows (box "H").
//                 D2 stays in TMEM (256 columns) over ALL tiles of the pair and is added to W_hat_l once, at the end.
//   The two GEMMs split the adjoint tile differently between the CTAs (MMA1 contracts over units and splits rows, MMA2
//   contracts over rows and splits units), and one descriptor addresses the same offset in both CTAs, so each CTA
//   loads the whole 256 x 32 adjoint tile (once as M1, once as A2; the second read is an L2 hit).
//   Epilogue (8 warps per CTA, warp (q, hs) = units [32 q, +32) x rows [16 hs, +16)): pulls its D1 columns into
//   registers and releases D1 at once, reads h^{l-1} from the H box (the same bytes MMA2 contracts), applies O4 written in
//   the output jet (jet_act_bwd), writes ahat^{l-1} in place into the H box and copies it out with 16-byte global stores
//   (MODE 1), or reduces the first-layer gradients and writes nothing (MODE 3).  b_hat_{l-1} is kept in registers over
//   all tiles.
#include "fused_bwd.cuh"

namespace pigan {

constexpr int kFWBytes = 4 * 128 * 64 * 2;   // resident W^T half: 4 k-blocks of 128 units x 64 contraction elements
constexpr uint32_t kFD1Col = 256;            // D2 = columns [0, 256), D1 = [256, 256 + 32 C)

template <int C> struct FusedCfg {
  static constexpr int kSlot = C * 8192;                       // every box is C planes of 8 KB
  static constexpr int kNH = C == 1 ? 4 : C == 3 ? 3 : 2;                   // H boxes in flight (held until the epilogue has copied its tile out)
  static constexpr int kNA = C == 1 ? 2 : 1;                   // A2 boxes
  static constexpr int kNM = C == 5 ? 1 : 2;                   // M1 boxes (C = 5: 64 KB of W^T + 4 boxes of 40 KB fill the 227 KB)
  static constexpr int kSmem = kFWBytes + (kNH + kNA + kNM) * kSlot + 1024 /*align*/ + 256 /*barriers*/;
  static_assert(kSmem <= 232448, "shared memory budget");
};

// [61,64) layout 6 = SWIZZLE_32B (MN-major atoms of 16 elements x 8 contraction rows = 256 B)
__device__ __forceinline__ uint64_t umma_desc_sw32(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16) | ((uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32) |
         (1ull << 46) | (6ull << 61);
}

template <typename T, int C, int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kFThreads, 1)
fused_bwd256_kernel(const __grid_constant__ CUtensorMap tmW,     // W_l^T [256 in][256 out] 16-bit, box 64 x 128, SW128
                    const __grid_constant__ CUtensorMap tmA2,    // ahat^l planes, box 32 rows x 128 units x C, SW64
                    const __grid_constant__ CUtensorMap tmH,     // h^{l-1} planes, box 32 rows x 128 units x C, SW64
                    const __grid_constant__ CUtensorMap tmM1,    // ahat^l planes, box 16 rows x 256 units x C, SW32
                    FusedParams p) {
  using Cfg = FusedCfg<C>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sW = smem;
  uint8_t* sH = sW + kFWBytes;
  uint8_t* sA2 = sH + Cfg::kNH * Cfg::kSlot;
  uint8_t* sM1 = sA2 + Cfg::kNA * Cfg::kSlot;
  uint64_t* bars = reinterpret_cast<uint64_t*>(sM1 + Cfg::kNM * Cfg::kSlot);
  uint64_t* wfull = bars;                       // [1]    leader's: the resident W^T halves of both CTAs have landed
  uint64_t* fullH = wfull + 1;                  // [kNH]  leader's
  uint64_t* hfree = fullH + Cfg::kNH;           // [kNH]  per CTA, 8 arrivals: the epilogue warps have copied the tile out
  uint64_t* fullA2 = hfree + Cfg::kNH;          // [kNA]  leader's
  uint64_t* emptyA2 = fullA2 + Cfg::kNA;        // [kNA]  per CTA (commit)
  uint64_t* fullM1 = emptyA2 + Cfg::kNA;        // [kNM]  leader's
  uint64_t* emptyM1 = fullM1 + Cfg::kNM;        // [kNM]  per CTA (commit)
  uint64_t* tfull = emptyM1 + Cfg::kNM;         // [1]    per CTA (commit): D1 of the tile is complete
  uint64_t* tempty = tfull + 1;                 // [1]    leader's, 16 arrivals: D1 is in the epilogue warps' registers
  uint64_t* m2done = tempty + 1;                // [kNH]  per CTA (commit): MMA2 has read H box it % kNH (it runs at most kNH - 1 tiles ahead of the epilogue)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(m2done + Cfg::kNH);

  const int warp = uniform_warp_idx(), lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int cluster_id = blockIdx.x >> 1, n_clusters = gridDim.x >> 1;

  if (warp == 0 && lane == 0) { prefetch_tmap(&tmW); prefetch_tmap(&tmA2); prefetch_tmap(&tmH); prefetch_tmap(&tmM1); }
  if (warp == 1 && lane == 0) {
    mbar_init(wfull, 1);
    for (int i = 0; i < Cfg::kNH; ++i) { mbar_init(fullH + i, 1); mbar_init(hfree + i, kFEpiWarps); }
    for (int i = 0; i < Cfg::kNA; ++i) { mbar_init(fullA2 + i, 1); mbar_init(emptyA2 + i, 1); }
    for (int i = 0; i < Cfg::kNM; ++i) { mbar_init(fullM1 + i, 1); mbar_init(emptyM1 + i, 1); }
    mbar_init(tfull, 1); mbar_init(tempty, 2 * kFEpiWarps);
    for (int i = 0; i < Cfg::kNH; ++i) mbar_init(m2done + i, 1);
    fence_barrier_init();
  }
  if (warp == 2) tmem2_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot, 0);

  if (warp == 0) {
    // ===================== TMA producer (both CTAs) =====================
    if (elect_one()) {
      if (rank == 0) mbar_expect_tx(wfull, 2 * kFWBytes);
      const uint32_t wb = mapa_u32(wfull, 0);
#pragma unroll
      for (int kb = 0; kb < 4; ++kb) tma2_load_2d(sW + kb * (kFWBytes / 4), &tmW, wb, kb * 64, (int)rank * 128);
    }
    __syncwarp();
    // Three load streams (M1, A2, H), each gated by its own consumer: MMA1 / MMA2 retiring the previous use of the slot, the
    // epilogue having copied the tile kNH back out.  The warp polls the three gates and issues whichever load may go, so a
    // stream never queues behind another one's gate (in program order H waited behind M1 and A2: measured, the epilogue
    // warps then sat 46 % of their time waiting for operands).
    const int n_my = (p.n_tiles - cluster_id + n_clusters - 1) / n_clusters;
    int itM = 0, itA = 0, itH = 0;
    uint32_t spins = 0;
    while (itM < n_my || itA < n_my || itH < n_my) {
      bool progress = false;
      if (itH < n_my) {
        const int s = itH % Cfg::kNH; const uint32_t ph = (uint32_t)(itH / Cfg::kNH) & 1;
        if (__all_sync(0xffffffffu, mbar_test_wait(hfree + s, ph ^ 1))) {
          if (elect_one()) {
            if (rank == 0) mbar_expect_tx(fullH + s, 2 * Cfg::kSlot);
            tma2_load_3d(sH + s * Cfg::kSlot, &tmH, mapa_u32(fullH + s, 0), (cluster_id + itH * n_clusters) * kFRows, (int)rank * 128, 0);
          }
          __syncwarp();
          ++itH; progress = true;
        }
      }
      if (itM < n_my) {
        const int s = itM % Cfg::kNM; const uint32_t ph = (uint32_t)(itM / Cfg::kNM) & 1;
        if (__all_sync(0xffffffffu, mbar_test_wait(emptyM1 + s, ph ^ 1))) {
          if (elect_one()) {
            if (rank == 0) mbar_expect_tx(fullM1 + s, 2 * Cfg::kSlot);
            tma2_load_3d(sM1 + s * Cfg::kSlot, &tmM1, mapa_u32(fullM1 + s, 0), (cluster_id + itM * n_clusters) * kFRows + (int)rank * 16, 0, 0);
          }
          __syncwarp();
          ++itM; progress = true;
        }
      }
      if (itA < n_my) {
        const int s = itA % Cfg::kNA; const uint32_t ph = (uint32_t)(itA / Cfg::kNA) & 1;
        if (__all_sync(0xffffffffu, mbar_test_wait(emptyA2 + s, ph ^ 1))) {
          if (elect_one()) {
            if (rank == 0) mbar_expect_tx(fullA2 + s, 2 * Cfg::kSlot);
            tma2_load_3d(sA2 + s * Cfg::kSlot, &tmA2, mapa_u32(fullA2 + s, 0), (cluster_id + itA * n_clusters) * kFRows, (int)rank * 128, 0);
          }
          __syncwarp();
          ++itA; progress = true;
        }
      }
      if (progress) spins = 0;
      else if (++spins > (1u << 26)) { if (lane == 0) printf("pigan: fused_bwd producer timed out (block %d)\n", (int)blockIdx.x); __trap(); }
    }
  } else if (warp == 1) {
    // ===================== MMA1 issuer (leader CTA; converged warp, one elected lane issues) =====================
    // The two GEMMs have their own issuing warps: MMA1 of a tile waits for its M1 box and for the epilogue to have pulled
    // the previous D1, MMA2 for its A2 and H boxes (H is held by the epilogue of tile it - kNH until it has copied out).
    // One in-order issuer chained "load latency + MMA" of both behind one another (measured: the epilogue warps then
    // waited 46 % of their time on tfull / m2done).
    if (rank == 0) {
      constexpr uint32_t idesc1 = umma_idesc(Fmt<T>::umma, 0, 1, 256, 32 * C);
      const uint32_t d1 = tmem_base + kFD1Col;
      const uint32_t aW = smem_u32(sW);
      mbar_wait(wfull, 0);
      int it = 0;
      for (int t = cluster_id; t < p.n_tiles; t += n_clusters, ++it) {
        // ---- MMA1: D1 = W^T ahat^l (contraction over the 256 out units, 16 k-steps) ----
        const int s = it % Cfg::kNM; const uint32_t ph = (uint32_t)(it / Cfg::kNM) & 1;
        mbar_wait(fullM1 + s, ph);
        mbar_wait_cluster(tempty, (uint32_t)(it & 1) ^ 1);     // both CTAs' epilogues hold D1 of the previous tile in registers
        tc_fence_after();
        const uint32_t bM = smem_u32(sM1 + s * Cfg::kSlot);
        if (elect_one()) {
#pragma unroll
          for (int ks = 0; ks < 16; ++ks) {
            // A: k-block ks / 4 (16 KB each), +32 B per 16 elements inside the 128-byte swizzle span
            // B (MN-major SW32): 16-row chunks (channels) 8 KB apart (LBO), 8-unit groups 256 B apart (SBO), 16 units = +512 B
            tc2_mma(d1, umma_desc_sw128(aW + (ks >> 2) * (kFWBytes / 4) + (ks & 3) * 32, 16, 1024), umma_desc_sw32(bM + ks * 512, 8192, 256), idesc1,
                    ks ? 1u : 0u);
          }
          tc2_commit(emptyM1 + s);
          tc2_commit(tfull);
        }
        __syncwarp();
      }
    }
  } else if (warp == 3) {
    // ===================== MMA2 issuer (leader CTA) =====================
    if (rank == 0) {
      constexpr uint32_t idesc2 = umma_idesc(Fmt<T>::umma, 0, 0, 256, 256);
      const uint32_t d2 = tmem_base;
      int it = 0;
      for (int t = cluster_id; t < p.n_tiles; t += n_clusters, ++it) {
        // ---- MMA2: D2 += ahat^l h^{l-1 T} (contraction over the tile's 32 rows of every channel, 2 C k-steps) ----
        const int sa = it % Cfg::kNA; const uint32_t pa = (uint32_t)(it / Cfg::kNA) & 1;
        const int sh = it % Cfg::kNH; const uint32_t phh = (uint32_t)(it / Cfg::kNH) & 1;
        mbar_wait(fullA2 + sa, pa);
        mbar_wait(fullH + sh, phh);
        tc_fence_after();
        const uint32_t aA = smem_u32(sA2 + sa * Cfg::kSlot), bH = smem_u32(sH + sh * Cfg::kSlot);
        if (elect_one()) {
#pragma unroll
          for (int c = 0; c < C; ++c)
#pragma unroll
            for (int k = 0; k < 2; ++k)
              tc2_mma(d2, umma_desc_sw64(aA + c * 8192 + k * 32, 16, 512), umma_desc_sw64(bH + c * 8192 + k * 32, 16, 512), idesc2,
                      (it | c | k) ? 1u : 0u);
          tc2_commit(emptyA2 + sa);
          tc2_commit(m2done + sh);
        }
        __syncwarp();
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue: warp (q, hs) owns TMEM lanes / in units [32 q, 32 q + 32) x rows [16 hs, 16 hs + 16) =====
    const int e = warp - 4, q = e & 3, hs = e >> 2;
    const int ul = q * 32 + lane;                            // unit within this CTA's 128
    const int unit = (int)rank * 128 + ul;
    const uint32_t lane_base = tmem_base + ((uint32_t)(q * 32) << 16);
    const uint32_t tD1 = lane_base + kFD1Col + hs * (16 * C);
    const float inv_amax = adj_inv_scale(p.amax);
    float bias_tot = 0.f, sx = 0.f, sy = 0.f;
    int it = 0;
    for (int t = cluster_id; t < p.n_tiles; t += n_clusters, ++it) {
      const int sh = it % Cfg::kNH;
      const int row0 = t * kFRows + hs * 16;
      mbar_wait(tfull, (uint32_t)(it & 1));
      tc_fence_after();
      float hh[C][16];
#pragma unroll
      for (int c = 0; c < C; ++c) { tmem_ld8(tD1 + c * 16, hh[c]); tmem_ld8(tD1 + c * 16 + 8, hh[c] + 8); }
      tmem_ld_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(mapa_u32(tempty, 0));
      // MMA2 of this tile reads the H box this warp is about to overwrite in place
      mbar_wait(m2done + sh, (uint32_t)(it / Cfg::kNH) & 1);
      fused_epi_tile<T, C, MODE>(p, hh, sH + sh * Cfg::kSlot, q, hs, lane, (int)rank * 128, row0, inv_amax, bias_tot, sx, sy);
      __syncwarp();
      if (lane == 0) mbar_arrive(hfree + sh);
    }
    atomicAdd(p.g_bias + unit, bias_tot * inv_amax);
    if (MODE == 3) {
      atomicAdd(p.gW1 + (size_t)unit * p.in_dim, sx * inv_amax);
      atomicAdd(p.gW1 + (size_t)unit * p.in_dim + 1, sy * inv_amax);
    }
    // ---- D2 -> W_hat_l: every MMA of this pair has retired (the last tfull / m2done), this CTA holds out units [128 rank, +128) ----
    {
      const int last = it - 1;
      mbar_wait(m2done + last % Cfg::kNH, (uint32_t)(last / Cfg::kNH) & 1);
      tc_fence_after();
      fused_drain(lane_base + hs * 128, p.gW + (size_t)unit * 256 + hs * 128, 128, inv_amax);
    }
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();                                        // neither CTA leaves while the pair still uses its smem / TMEM
  if (warp == 2) { tc_fence_after(); tmem2_dealloc(tmem_base, 512); }
}

// =============================================================================================================
// host side
// =============================================================================================================
bool tc2_fused_bwd_supported(const Launcher& L, int H, int C) { return tc2_supported(L, H) && H == 256 && (C == 1 || C == 3 || C == 5); }

template <int C, int MODE>
static void launch_fused(Launcher& L, const CUtensorMap& w, const CUtensorMap& a2, const CUtensorMap& h, const CUtensorMap& m1, const FusedParams& p) {
  using Cfg = FusedCfg<C>;
  static unsigned long long attr_done = 0;
  auto kern = fused_bwd256_kernel<__half, C, MODE>;
  ensure_smem_attr(L, kern, Cfg::kSmem, attr_done);
  const int clusters = std::min(p.n_tiles, L.num_sms / 2);
  kern<<<2 * clusters, kFThreads, Cfg::kSmem, L.stream>>>(w, a2, h, m1, p);
  L.check("jet_layer_bwd_wgrad");
}

void tc2_fused_bwd(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* w16T_l, const void* ahat_in, const void* h_prev,
                   void* ahat_out, float* gW, float* g_bias_prev, const float* amax, const FirstLayerFuse* fl) {
  if (R <= 0) return;
  CUtensorMap w, a2, h, m1;
  bool ok = weight_map(L, &w, precision, w16T_l, H) && plane_map(L, &a2, precision, ahat_in, H, R_ld, C, 32, 128, C, CU_TENSOR_MAP_SWIZZLE_64B) &&
            plane_map(L, &h, precision, h_prev, H, R_ld, C, 32, 128, C, CU_TENSOR_MAP_SWIZZLE_64B) &&
            plane_map(L, &m1, precision, ahat_in, H, R_ld, C, 16, 256, C, CU_TENSOR_MAP_SWIZZLE_32B);
  if (!ok) return;
  FusedParams p{};
  p.H = H; p.n_tiles = R / kFRows; p.gW = gW; p.g_bias = g_bias_prev; p.out = ahat_out; p.R_ld = R_ld; p.amax = amax;
  if (fl) {
    p.xy = fl->xy; p.row0 = fl->row0; p.npts = fl->npts; p.in_dim = fl->in_dim; p.gW1 = fl->gW1; p.An = fl->An; p.per_sample = fl->per_sample;
    if (C == 1) launch_fused<1, 3>(L, w, a2, h, m1, p); else if (C == 3) launch_fused<3, 3>(L, w, a2, h, m1, p); else launch_fused<5, 3>(L, w, a2, h, m1, p);
    return;
  }
  if (C == 1) launch_fused<1, 1>(L, w, a2, h, m1, p); else if (C == 3) launch_fused<3, 1>(L, w, a2, h, m1, p); else launch_fused<5, 1>(L, w, a2, h, m1, p);
}

}  // namespace pigan
