// sm_100a tensor-core kernels of the jet MLP on CTA PAIRS (tcgen05 cta_group::2), used when the width is a multiple
// of 256.  Same math and plane layout as tc_kernels.cu; what changes is
// how much every SM must pull in per flop: the SM's inbound path (~64 B/clk) bounds the one-CTA kernels, and a pair
// shares the activation operand, so each CTA loads its own 128 x K weight rows but only HALF of the activation tile.
//
// jet layer:  D[256 units][(channel, row) columns] = W_tile[256 x K] . act[K x (C * 64 rows)]
//   A = weights, K-major, SW128: CTA r of the pair loads units [128 r, 128 r + 128) of the tile.
//   B = activation planes [channel][unit][row], MN-major, SW64: CTA r loads rows [32 r, 32 r + 32) of the 64-row tile
//       for all C channels (one 3D TMA box 32 rows x 64 units x C).  One MMA covers a group of nc channels,
//       N = 64 nc; its accumulator columns are [CTA half h][channel][32 rows].
//   C = 5 needs 320 of the 512 TMEM columns, so tiles alternate between columns [0, 320) and [192, 512) with the
//       (xx, yy) group always at [192, 320): the epilogue pulls that group into registers first and releases it, so
//       the next tile's MMAs start while the rest of the epilogue runs.  C <= 3 double-buffers.
//   Epilogue: 8 warps per CTA; warp (q, h) owns units [32 q, 32 q + 32) (TMEM lanes) x rows [32 h, 32 h + 32).
// wgrad:  D[256 out units][256 in units] += sum_{c, row} ahat_c[out][row] h_c[in][row], both operands K-major SW128.
#include "tc_ptx.cuh"

namespace pigan {

constexpr int k2AStage = 128 * 64 * 2;      // 16 KB: 128 units x 64 contraction elements
constexpr int k2BPlane = 64 * 32 * 2;       // 4 KB: 64 contraction units x 32 rows of one channel
constexpr int k2StgPlane = 32 * 64;         // epilogue staging plane: 32 units x 32 rows x 2 B
constexpr int k2EpiWarps = 8;
constexpr int k2Threads = (4 + k2EpiWarps) * 32;


template <int C, int MODE> struct Jet2Cfg {
  static constexpr int kStageBytes = k2AStage + C * k2BPlane;
  static constexpr int kCols = C * 64;                                 // accumulator columns of one tile
  static constexpr int kNumBuf = C == 5 ? 1 : 2;                       // C = 5: alternating placement, early release
  static constexpr int kTmemCols = C == 5 ? 512 : 2 * kCols <= 128 ? 128 : 2 * kCols <= 256 ? 256 : 512;
  static constexpr int kSlots = C;                                     // staging planes per epilogue warp
  // plain forward at C = 5: the epilogue stages and copies out 16 rows at a time (planes of 32 units x 16 rows), which frees
  // 40 KB for a fifth operand stage -- the deferred (xx, yy) MMAs hold two stages of the ring at the start of every tile
  static constexpr bool kHalfStg = MODE == 0 && C == 5;
  static constexpr int kStgBytes = k2EpiWarps * kSlots * (kHalfStg ? k2StgPlane / 2 : k2StgPlane);
  static constexpr int kBudget = 232448 - 1024 - 512 - kStgBytes;
  static constexpr int kNumStages = kBudget / kStageBytes > 6 ? 6 : kBudget / kStageBytes;
  static constexpr int kSmemBytes = kNumStages * kStageBytes + kStgBytes + 1024 /*align*/ + 512 /*barriers*/;
};

struct Jet2Params {
  int H;                 // width (K and number of output units), multiple of 256
  int n_row_tiles;       // R / 64
  const float* bias;     // MODE 0, 2: b_l
  float* g_bias;         // MODE 1: b_hat_{l-1}
  void* out;             // MODE 0, 2: h_out planes; MODE 1: ahat_out planes  [C][H][R_ld] 16-bit
  int R_ld;              // leading dimension (rows) of the output planes
  const float* amax;     // MODE 1, 3: block-scale source of the adjoint planes
  // MODE 3 (dgrad of layer 2 + adjoint of the FIRST tanh layer + first-layer reduction, O4 'First layer'): ahat^1 is
  // consumed in registers and never written.  Requires npts % 64 == 0 (a row tile lies inside one latent sample).
  const float* xy;       // [npts][2]
  long long row0;        // first global row of the chunk
  int npts, in_dim, per_sample;
  float* gW1;            // W_hat_1 [H][in_dim]: columns 0, 1 += sum_r (ahat x_r + ahat_x), (ahat y_r + ahat_y)
  float* An;             // [N][H] += sum_{r in sample n} ahat
  // MODE 4, 5 (last hidden layer + output layer a4): o_c[r] += sum_units w_out[unit] h_c[unit][r], reduced over the lanes of a
  // warp by shuffles and over warps / CTAs / unit tiles by fp32 atomics (o is zeroed by the launcher; b_out enters once).
  const float* w_out;    // [H]
  const float* b_out;    // [1]
  float* o;              // [C][o_stride] fp32 (MODE 5: one plane)
  long long o_stride;
  int valid;             // rows of the chunk that exist: rows >= valid are not accumulated
  int reverse;           // sweep the row tiles from the last to the first: consecutive layers alternate direction, so a layer starts on
                         // the rows its predecessor wrote last, which are still in the 126 MB L2 (matters where a layer is HBM-bound: H = 256)
  int linear;            // MODE 0 only: plain GEMM, out_c = W in_c (no bias, no tanh): the raw adjoint planes of a skip layer (NEXT-1)
};

// MODE 0: forward; MODE 1: dgrad + adjoint of the previous tanh; MODE 2: value-only forward on split (hi, lo) planes;
// MODE 3: MODE 1 with the first-layer backward reduction fused (no adjoint planes written);
// MODE 4 / 5: MODE 0 / 2 for the LAST hidden layer with the output dot (a4) fused into the epilogue; p.out == nullptr then
//             skips the h^L planes (forward-only callers).
template <typename T, int C, int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(k2Threads, 1)
jet2_layer_kernel(const __grid_constant__ CUtensorMap tmA,      // weights [H][H] 16-bit, box 64 x 128, SW128
                  const __grid_constant__ CUtensorMap tmB,      // input planes, box 32 rows x 64 units x C, SW64
                  const __grid_constant__ CUtensorMap tmT,      // MODE 1, 3: h_prev planes in; MODE 4: h_out planes (box 32 rows x 32 units x C, SW64)
                  Jet2Params p) {
  using Cfg = Jet2Cfg<C, MODE>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* stages = smem;
  uint8_t* staging = smem + Cfg::kNumStages * Cfg::kStageBytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(staging + Cfg::kStgBytes);
  uint64_t* full = bars;                                   // [kNumStages]  leader's is used
  uint64_t* empty = bars + Cfg::kNumStages;                // [kNumStages]  per CTA
  uint64_t* tfull = empty + Cfg::kNumStages;               // [kNumBuf]     per CTA
  uint64_t* tempty = tfull + Cfg::kNumBuf;                 // [kNumBuf]     leader's is used, 16 arrivals
  uint64_t* sbar = tempty + Cfg::kNumBuf;                  // [8]           staging loads (MODE 1), one per epilogue warp
  uint64_t* tempty0 = sbar + k2EpiWarps;                   // [2]  C = 5: group-0 columns of tile it (parity it & 1) fully read, 16 arrivals
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty0 + 2);

  const int warp = uniform_warp_idx(), lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int cluster_id = blockIdx.x >> 1, n_clusters = gridDim.x >> 1;
  const int n_ut = p.H / 256;
  const int n_tiles = n_ut * p.n_row_tiles;
  const int n_kb = p.H / 64;
  constexpr bool kFwd = MODE == 0 || MODE == 4, kSplit = MODE == 2 || MODE == 5, kOutDot = MODE == 4 || MODE == 5;

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmA); prefetch_tmap(&tmB);
    if (MODE == 1 || MODE == 3 || MODE == 4) prefetch_tmap(&tmT);
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < Cfg::kNumStages; ++i) { mbar_init(full + i, 1); mbar_init(empty + i, 1); }
    for (int i = 0; i < Cfg::kNumBuf; ++i) { mbar_init(tfull + i, 1); mbar_init(tempty + i, 2 * k2EpiWarps); }
    for (int i = 0; i < k2EpiWarps; ++i) mbar_init(sbar + i, 1);
    for (int i = 0; i < 2; ++i) mbar_init(tempty0 + i, 2 * k2EpiWarps);
    fence_barrier_init();
  }
  if (warp == 2) tmem2_alloc(tmem_slot, Cfg::kTmemCols);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();                                      // the peer's barriers are initialised before anything signals them
  tc_fence_after();
  const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot, 0);       // uniform: TMEM addresses live in uniform registers

  // accumulator columns: tile `it` of this cluster; channel group 0 = channels [0, min(C, 3)), group 1 = (xx, yy)
  auto g0_col = [&](int it) -> uint32_t { return C == 5 ? ((it & 1) ? 320u : 0u) : (uint32_t)((it % Cfg::kNumBuf) * Cfg::kCols); };
  constexpr uint32_t g1_col = 192;
  constexpr int nc0 = C == 5 ? 3 : C;                      // channels in group 0

  if (warp == 0) {
    // ===================== TMA producer (both CTAs; the warp stays converged, one elected lane issues) =====================
    {
      int stage = 0; uint32_t phase = 0;
      for (int t = cluster_id; t < n_tiles; t += n_clusters) {
        const int ut = t % n_ut, rt = p.reverse ? p.n_row_tiles - 1 - t / n_ut : t / n_ut;
        for (int kb = 0; kb < n_kb; ++kb) {
          mbar_wait(empty + stage, phase ^ 1);
          uint8_t* sA = stages + stage * Cfg::kStageBytes;
          const uint32_t lbar = mapa_u32(full + stage, 0);
          if (elect_one()) {
            if (rank == 0) mbar_expect_tx(full + stage, 2 * Cfg::kStageBytes);
            tma2_load_2d(sA, &tmA, lbar, kb * 64, ut * 256 + (int)rank * 128);
            tma2_load_3d(sA + k2AStage, &tmB, lbar, rt * 64 + (int)rank * 32, kb * 64, 0);
          }
          __syncwarp();
          if (++stage == Cfg::kNumStages) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA; converged warp, one elected lane issues) =====================
    if (rank == 0) {
      // tcgen05.mma issue returns when the MMA starts executing (the queue is about one deep), so a barrier wait
      // issued after the last MMA of a stage idles the tensor pipe for its whole latency.  The wait for the NEXT
      // stage is therefore polled behind the longest MMA of the last k-step, and only repeated (blocking) on a miss.
      int stage = 0; uint32_t phase = 0; int it = 0;
      bool ready = false;                                    // full[stage] of the upcoming k-block already seen complete
      constexpr uint32_t idesc0 = umma_idesc(Fmt<T>::umma, 0, 1, 256, nc0 * 64);
      constexpr uint32_t idesc1 = umma_idesc(Fmt<T>::umma, 0, 1, 256, 128);
      for (int t = cluster_id; t < n_tiles; t += n_clusters, ++it) {
        const int buf = it % Cfg::kNumBuf;
        const uint32_t bphase = (it / Cfg::kNumBuf) & 1;
        const bool last_tile = t + n_clusters >= n_tiles;
        // C <= 3: the accumulator is double-buffered.  C = 5 (320 of 512 columns): group 0 (value, x, y) alternates between
        // two placements and group 1 (xx, yy) has one, which the epilogue of the previous tile releases as soon as it has
        // pulled it into registers.  That release arrives ~700 clk after the previous tile's last MMA, so the first kDefer
        // k-blocks of a tile issue only their group-0 MMAs (whose columns the epilogue of tile it-2 freed long ago,
        // tempty0), and their group-1 MMAs follow once the release is in; their smem stages are freed after that.
        constexpr int kDefer = C == 5 ? 2 : 0;
        if (C == 5) mbar_wait_cluster(tempty0 + (it & 1), (uint32_t)(((it >> 1) & 1) ^ 1));
        else mbar_wait_cluster(tempty + buf, bphase ^ 1);    // both CTAs' epilogues have released what this tile overwrites
        tc_fence_after();
        const uint32_t d0 = tmem_base + g0_col(it), d1 = tmem_base + g1_col;
        if (C == 5) {
          int dstage[kDefer > 0 ? kDefer : 1];
#pragma unroll
          for (int kb = 0; kb < kDefer; ++kb) {
            if (!ready) mbar_wait(full + stage, phase);
            ready = false;
            tc_fence_after();
            const uint32_t sA = smem_u32(stages + stage * Cfg::kStageBytes), sB = sA + k2AStage;
            if (elect_one()) {
#pragma unroll
              for (int k = 0; k < 4; ++k)
                tc2_mma(d0, umma_desc_sw128(sA + k * 32, 16, 1024), umma_desc_sw64(sB + k * 1024, k2BPlane, 512), idesc0, (kb | k) ? 1u : 0u);
            }
            __syncwarp();
            dstage[kb] = stage;
            if (++stage == Cfg::kNumStages) { stage = 0; phase ^= 1; }
          }
          mbar_wait_cluster(tempty + buf, bphase ^ 1);       // group 1 of the previous tile is in the epilogue's registers
          tc_fence_after();
#pragma unroll
          for (int kb = 0; kb < kDefer; ++kb) {
            const uint32_t sA = smem_u32(stages + dstage[kb] * Cfg::kStageBytes), sB = sA + k2AStage;
            if (elect_one()) {
#pragma unroll
              for (int k = 0; k < 4; ++k)
                tc2_mma(d1, umma_desc_sw128(sA + k * 32, 16, 1024), umma_desc_sw64(sB + 3 * k2BPlane + k * 1024, k2BPlane, 512), idesc1, (kb | k) ? 1u : 0u);
              tc2_commit(empty + dstage[kb]);
            }
            __syncwarp();
          }
        }
        for (int kb = kDefer; kb < n_kb; ++kb) {
          if (!ready) mbar_wait(full + stage, phase);
          tc_fence_after();
          const uint32_t sA = smem_u32(stages + stage * Cfg::kStageBytes), sB = sA + k2AStage;
          int nstage = stage + 1; uint32_t nphase = phase;
          if (nstage == Cfg::kNumStages) { nstage = 0; nphase ^= 1; }
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const uint64_t ad = umma_desc_sw128(sA + k * 32, 16, 1024);                       // K-major: +32 B per 16 elements
            const uint32_t acc = (kb | k) ? 1u : 0u;
            // MN-major SW64: channel planes are 4 KB apart (LBO), 8-unit groups 512 B apart (SBO), 16 units = +1 KB
            // C = 5: the two MMAs of a k-step read the same A slice: the first fills the A collector, the second reuses it
            if (C == 5 && k < 3 && elect_one()) tc2_mma_a_fill(d1, ad, umma_desc_sw64(sB + 3 * k2BPlane + k * 1024, k2BPlane, 512), idesc1, acc);
            if (C != 5 && k == 3) ready = !(last_tile && kb == n_kb - 1) && __all_sync(0xffffffffu, mbar_try_wait(full + nstage, nphase));
            if (elect_one()) {
              if (C != 5) tc2_mma(d0, ad, umma_desc_sw64(sB + k * 1024, k2BPlane, 512), idesc0, acc);
              else if (k < 3) tc2_mma_a_lastuse(d0, ad, umma_desc_sw64(sB + k * 1024, k2BPlane, 512), idesc0, acc);
              else tc2_mma_a_fill(d0, ad, umma_desc_sw64(sB + k * 1024, k2BPlane, 512), idesc0, acc);
            }
            if (C == 5 && k == 3) {
              ready = !(last_tile && kb == n_kb - 1) && __all_sync(0xffffffffu, mbar_try_wait(full + nstage, nphase));
              if (elect_one()) tc2_mma_a_lastuse(d1, ad, umma_desc_sw64(sB + 3 * k2BPlane + k * 1024, k2BPlane, 512), idesc1, acc);
            }
          }
          if (elect_one()) tc2_commit(empty + stage);        // frees the smem slot in both CTAs when these MMAs retire
          __syncwarp();
          stage = nstage; phase = nphase;
        }
        if (elect_one()) tc2_commit(tfull + buf);            // accumulator complete (both CTAs)
        __syncwarp();
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue: warp (q, hs) owns TMEM lanes / units [32q, 32q+32) x rows [32hs, 32hs+32) ==========
    const int e = warp - 4, q = e & 3, hs = e >> 2;
    uint8_t* stg = staging + e * (Cfg::kSlots * (Cfg::kHalfStg ? k2StgPlane / 2 : k2StgPlane));
    const uint32_t swz = (uint32_t)((lane >> 1) & 3);       // 64B swizzle of a 64-byte row: chunk ^= (row >> 1) & 3
    uint8_t* my_row = stg + lane * 64;
    const uint32_t lane_base = tmem_base + ((uint32_t)(q * 32) << 16);
    uint32_t sphase = 0;
    int it = 0;
    const float inv_amax = (MODE == 1 || MODE == 3) ? adj_inv_scale(p.amax) : 1.f;   // constant over the launch: one global load, not one per tile
    for (int t = cluster_id; t < n_tiles; t += n_clusters, ++it) {
      const int ut = t % n_ut, rt = p.reverse ? p.n_row_tiles - 1 - t / n_ut : t / n_ut;
      const int buf = it % Cfg::kNumBuf;
      const uint32_t bphase = (it / Cfg::kNumBuf) & 1;
      const int unit0 = ut * 256 + (int)rank * 128 + q * 32, unit = unit0 + lane;
      const int row0 = rt * 64 + hs * 32;
      // TMEM address of (channel c, row 0 of this warp's half)
      const uint32_t tb0 = lane_base + g0_col(it) + hs * (nc0 * 32), tb1 = lane_base + g1_col + hs * 64;
      auto tcol = [&](int c) -> uint32_t { return (C == 5 && c >= 3) ? tb1 + (c - 3) * 32 : tb0 + c * 32; };
      float bias = 0.f, bias_acc = 0.f;
      if ((kFwd || kSplit) && p.bias) bias = p.bias[unit];
      float wo = 0.f;
      if (kOutDot) wo = p.w_out[unit];
      // MODE 4, 5: lane -> row (4 * bit4 + 2 * bit3 + bit2) of each group of 8 rows; one lane of four adds
      const int orow = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
      auto out_dot = [&](int c, int rc, const float* hv) {  // hv[8]: this unit's h_c at rows rc * 8 .. + 8 (fp32, unrounded)
        float pv[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) pv[i] = wo * hv[i];
        float tot = warp_reduce8(pv, lane);
        const int r = row0 + rc * 8 + orow;
        if (c == 0 && ut == 0 && rank == 0 && q == 0) tot += p.b_out[0];
        if ((lane & 3) == 0 && r < p.valid) atomicAdd(p.o + (size_t)c * p.o_stride + r, tot);
      };
      // Staged planes -> global with the epilogue warp's own 16-byte stores (4 lanes cover the 64 contiguous bytes of one
      // unit's 32 rows).  Measured: a TMA store drains shared memory at ~26 B/clk per SM whatever the box shape, and the
      // TMA unit serves loads and stores one after the other, so storing a C = 5 tile through it cost the operand
      // pipeline ~2.6 k of the tile's ~14 k clk.
      auto copy_out = [&](int nplanes) {
        __syncwarp();
        T* gout = reinterpret_cast<T*>(p.out);
        const int ch = lane & 3, ul = lane >> 2;
        if (MODE == 1) {
          // The next tile's TMA load (async proxy) overwrites these staging planes: every lane pulls its share into
          // registers, then orders its generic-proxy accesses before later async-proxy ones (fence.proxy.async), and only
          // then issues the global stores -- so the fence waits for shared-memory reads, not for store acknowledgements.
          uint4 v[C][4];
#pragma unroll
          for (int c = 0; c < C; ++c)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              const int u = j * 8 + ul;
              v[c][j] = lds128(stg + c * k2StgPlane + u * 64 + ((ch ^ ((u >> 1) & 3)) << 4));
            }
          fence_proxy_async();
#pragma unroll
          for (int c = 0; c < C; ++c)
#pragma unroll
            for (int j = 0; j < 4; ++j)
              *reinterpret_cast<uint4*>(gout + ((size_t)c * p.H + unit0 + j * 8 + ul) * p.R_ld + row0 + ch * 8) = v[c][j];
        } else {
#pragma unroll
          for (int c = 0; c < 5; ++c) {
            if (c < nplanes) {
#pragma unroll
              for (int j = 0; j < 4; ++j) {
                const int u = j * 8 + ul;
                const uint4 v = lds128(stg + c * k2StgPlane + u * 64 + ((ch ^ ((u >> 1) & 3)) << 4));
                *reinterpret_cast<uint4*>(gout + ((size_t)c * p.H + unit0 + u) * p.R_ld + row0 + ch * 8) = v;
              }
            }
          }
        }
        __syncwarp();                                        // the staging rows are rewritten by other lanes in the next tile
      };
      auto release0 = [&]() {                                // C = 5: this warp has read all of group 0 of this tile
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(mapa_u32(tempty0 + (it & 1), 0));
      };
      auto release = [&]() {                                 // this warp no longer reads what the next MMAs overwrite
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(mapa_u32(tempty + buf, 0));
      };

      if ((MODE == 1 || MODE == 3) && elect_one()) {         // the previous layer's output jet h^{l-1} -> staging
        // Generic-proxy accesses of the staging planes by the previous tile were fenced (fence.proxy.async) by every lane
        // inside copy_out (MODE 1) before its trailing __syncwarp; MODE 3 only reads them (see the fence after its loop).
        // one 3D box (32 rows x 32 units x C channels) lands as C consecutive 2 KB planes: one TMA issue instead of C
        // (measured: each extra issue stalled the warp ~400 samples behind the producer's loads in the TMA queue)
        mbar_expect_tx(sbar + e, C * k2StgPlane);
        tma_load_3d(stg, &tmT, sbar + e, row0, unit0, 0);
      }
      mbar_wait(tfull + buf, bphase);
      tc_fence_after();

      // C = 5: the (xx, yy) group leaves TMEM first
      float kxx[C == 5 ? 32 : 1], kyy[C == 5 ? 32 : 1];
      if (C == 5) {
#pragma unroll
        for (int rc = 0; rc < 4; ++rc) { tmem_ld8(tcol(3) + rc * 8, kxx + rc * 8); tmem_ld8(tcol(4) + rc * 8, kyy + rc * 8); }
        tmem_ld_wait();
        release();
      }

      if (Cfg::kHalfStg) {
        // ---- h_c = tanh-jet(a_c), 16 rows at a time through staging planes of 32 units x 32 bytes (16-byte chunk ^= (unit >> 2) & 1) ----
        const uint32_t swz32 = (uint32_t)((lane >> 2) & 1);
        T* gout = reinterpret_cast<T*>(p.out);
#pragma unroll
        for (int hf = 0; hf < 2; ++hf) {
#pragma unroll
          for (int r2 = 0; r2 < 2; ++r2) {
            const int rc = hf * 2 + r2;
            float v[C][8], o[C][8];
#pragma unroll
            for (int c = 0; c < nc0; ++c) tmem_ld8(tcol(c) + rc * 8, v[c]);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              float a[5], h[5];
#pragma unroll
              for (int c = 0; c < nc0; ++c) a[c] = v[c][i];
              a[3] = kxx[rc * 8 + i]; a[4] = kyy[rc * 8 + i];
              a[0] += bias;
              if (p.linear) {
#pragma unroll
                for (int c = 0; c < C; ++c) h[c] = a[c];
              } else {
                jet_act_fwd<C>(fast_tanh(a[0]), a, h);
              }
#pragma unroll
              for (int c = 0; c < C; ++c) o[c][i] = h[c];
            }
#pragma unroll
            for (int c = 0; c < C; ++c) sts128(stg + c * 1024 + lane * 32 + (((uint32_t)r2 ^ swz32) << 4), pack8<T>(o[c]));
          }
          if (hf == 1) release0();
          __syncwarp();
          const int chw = lane & 1, ulw = lane >> 1;        // two lanes cover the 32 contiguous bytes (one sector) of one unit's 16 rows
#pragma unroll
          for (int c = 0; c < C; ++c)
#pragma unroll
            for (int j = 0; j < 2; ++j) {
              const int u = j * 16 + ulw;
              const uint4 v = lds128(stg + c * 1024 + u * 32 + (((uint32_t)chw ^ (uint32_t)((u >> 2) & 1)) << 4));
              *reinterpret_cast<uint4*>(gout + ((size_t)c * p.H + unit0 + u) * p.R_ld + row0 + hf * 16 + chw * 8) = v;
            }
          __syncwarp();                                      // the staging rows are rewritten by other lanes in the next half
        }
      } else if (kFwd) {
        // MODE 4: the previous tile's TMA store has read the staging planes
        if (MODE == 4 && p.out) { if (elect_one()) tma_wait_read_all(); __syncwarp(); }
        // ---- h_c = tanh-jet(a_c) ----
#pragma unroll
        for (int rc = 0; rc < 4; ++rc) {
          float v[C][8], o[C][8];
#pragma unroll
          for (int c = 0; c < nc0; ++c) tmem_ld8(tcol(c) + rc * 8, v[c]);
          tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            float a[5], h[5];
#pragma unroll
            for (int c = 0; c < nc0; ++c) a[c] = v[c][i];
            if (C == 5) { a[3] = kxx[rc * 8 + i]; a[4] = kyy[rc * 8 + i]; }
            a[0] += bias;
            if (MODE == 0 && p.linear) {
#pragma unroll
              for (int c = 0; c < C; ++c) h[c] = a[c];
            } else {
              jet_act_fwd<C>(fast_tanh(a[0]), a, h);
            }
#pragma unroll
            for (int c = 0; c < C; ++c) o[c][i] = h[c];
          }
          const uint32_t off = ((uint32_t)rc ^ swz) << 4;
          if (!kOutDot || p.out) {
#pragma unroll
            for (int c = 0; c < C; ++c) sts128(my_row + c * k2StgPlane + off, pack8<T>(o[c]));
          }
          if (kOutDot) {
#pragma unroll
            for (int c = 0; c < C; ++c) out_dot(c, rc, o[c]);
          }
        }
        if (C != 5) release(); else release0();
        if (MODE == 4 && p.out) {
          // The output dot's shuffles and atomics make this epilogue the longest of the forward: the tile leaves through ONE
          // asynchronous TMA store per warp instead of the warp's own 20 LDS + 20 STG (measured on B200, last layer of a
          // 131072-row chunk: -22 % at H = 256, -21 % at H = 512, -2 % at H = 1024; the plain forward layers gain nothing
          // from it and lose 3 % at H = 1024, where the TMA unit is the busier side, so they keep their own stores)
          fence_proxy_async();
          __syncwarp();
          if (elect_one()) { tma_store_3d(&tmT, stg, row0, unit0, 0); tma_commit_group(); }
          __syncwarp();
        } else if (!kOutDot) {
          copy_out(C);
        }
      } else if (kSplit) {
        // ---- value-only layer with split activations: a = W (h_hi + h_lo) + b; t = tanh a; t_hi = rn16(t), t_lo = rn16(t - t_hi) ----
#pragma unroll 1
        for (int rc = 0; rc < 4; ++rc) {
          float v0[8], v1[8], hi[8], lo[8], tv[8];
          tmem_ld8(tcol(0) + rc * 8, v0);
          tmem_ld8(tcol(1) + rc * 8, v1);
          tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const float tt = tanhf(v0[i] + v1[i] + bias);
            tv[i] = tt;
            hi[i] = to_f<T>(from_f<T>(tt));
            lo[i] = tt - hi[i];
          }
          const uint32_t off = ((uint32_t)rc ^ swz) << 4;
          if (!kOutDot || p.out) {
            sts128(my_row + off, pack8<T>(hi));
            sts128(my_row + k2StgPlane + off, pack8<T>(lo));
          }
          if (kOutDot) out_dot(0, rc, tv);
        }
        release();
        if (!kOutDot || p.out) copy_out(2);
      } else {
        // ---- adjoint of the previous layer's tanh: ahat^{l-1} = J^T hhat^{l-1} ----
        mbar_wait(sbar + e, sphase); sphase ^= 1;
        float sx = 0.f, sy = 0.f;                            // MODE 3
        const long long grow = p.row0 + row0;                // MODE 3: global row of this warp's first row
        const float2* xyp = MODE == 3 ? reinterpret_cast<const float2*>(p.xy) + (p.per_sample ? grow : grow % p.npts) : nullptr;
#pragma unroll
        for (int rc = 0; rc < 4; ++rc) {
          float hh[C][8], hp[C][8], o[C][8];
#pragma unroll
          for (int c = 0; c < nc0; ++c) tmem_ld8(tcol(c) + rc * 8, hh[c]);
          const uint32_t off = ((uint32_t)rc ^ swz) << 4;
#pragma unroll
          for (int c = 0; c < C; ++c) unpack8<T>(lds128(my_row + c * k2StgPlane + off), hp[c]);
          tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            float hx[5], hj[5], aa[5];
#pragma unroll
            for (int c = 0; c < nc0; ++c) hx[c] = hh[c][i];
            if (C == 5) { hx[3] = kxx[rc * 8 + i]; hx[4] = kyy[rc * 8 + i]; }
#pragma unroll
            for (int c = 0; c < C; ++c) hj[c] = hp[c][i];
            jet_act_bwd<C>(hj, hx, aa);
            bias_acc += aa[0];
            if (MODE == 3) {
              const float2 q = __ldg(xyp + rc * 8 + i);      // same address in every lane: one broadcast load
              sx = fmaf(aa[0], q.x, sx); sy = fmaf(aa[0], q.y, sy);
              if (C >= 3) { sx += aa[1]; sy += aa[2]; }
            }
#pragma unroll
            for (int c = 0; c < C; ++c) o[c][i] = aa[c];
          }
          if (MODE == 1) {
#pragma unroll
            for (int c = 0; c < C; ++c) sts128(my_row + c * k2StgPlane + off, pack8<T>(o[c]));
          }
        }
        if (C != 5) release(); else release0();
        if (MODE == 1) {
          copy_out(C);
        } else {
          fence_proxy_async();                               // generic reads of the staging planes before the next tile's TMA writes
          __syncwarp();                                      // every lane is done reading the staging planes before the next loads land
          const float inv = inv_amax;
          atomicAdd(p.An + (size_t)(grow / p.npts) * p.H + unit, bias_acc * inv);
          atomicAdd(p.gW1 + (size_t)unit * p.in_dim, sx * inv);
          atomicAdd(p.gW1 + (size_t)unit * p.in_dim + 1, sy * inv);
        }
        atomicAdd(p.g_bias + unit, bias_acc * inv_amax);
      }
    }
  }
  if (MODE == 4 && warp >= 4) { if (elect_one()) tma_wait_all(); __syncwarp(); }   // the last stores have left shared memory and are complete
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();                                        // neither CTA leaves while the pair still uses its smem / TMEM
  if (warp == 2) { tc_fence_after(); tmem2_dealloc(tmem_base, Cfg::kTmemCols); }
}

// =============================================================================================================
// wgrad on CTA pairs: gW[j][k] += sum_{c, r} ahat_c[j][r] h_c[k][r], 256 x 256 output tiles, rows split into slices
// =============================================================================================================
constexpr int kW2Stages = 6;
constexpr int kW2StageBytes = 2 * k2AStage;     // A: 128 out units x 64 rows, B: 128 in units x 64 rows (this CTA's halves)
struct Wgrad2Params {
  int H, C;
  int n_slices;        // row slices
  int slice_rows;      // rows per slice (multiple of 64)
  int R;               // rows of the chunk (multiple of 64)
  float* gW;           // [H][H] fp32
  const float* amax;   // block-scale source of the adjoint planes
};

template <typename T>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(192, 1)
wgrad2_kernel(const __grid_constant__ CUtensorMap tmA,    // ahat planes, box 64 rows x 128 units x 1, SW128
              const __grid_constant__ CUtensorMap tmB,    // h_prev planes, box 64 rows x 128 units x 1, SW128
              Wgrad2Params p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* stages = smem;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kW2Stages * kW2StageBytes);
  uint64_t* full = bars; uint64_t* empty = bars + kW2Stages; uint64_t* tfull = empty + kW2Stages; uint64_t* tempty = tfull + 2;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 2);
  const int warp = uniform_warp_idx(), lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int cluster_id = blockIdx.x >> 1, n_clusters = gridDim.x >> 1;
  const int n_t = p.H / 256;
  const int n_items = n_t * n_t * p.n_slices;

  if (warp == 0 && lane == 0) { prefetch_tmap(&tmA); prefetch_tmap(&tmB); }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < kW2Stages; ++i) { mbar_init(full + i, 1); mbar_init(empty + i, 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(tfull + i, 1); mbar_init(tempty + i, 8); }
    fence_barrier_init();
  }
  __syncwarp();
  if (warp == 1) tmem2_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot, 0);       // uniform: TMEM addresses live in uniform registers

  auto decode = [&](int w, int& mt, int& nt, int& r0, int& r1) {
    const int tile = w % (n_t * n_t), sl = w / (n_t * n_t);
    mt = tile % n_t; nt = tile / n_t;
    r0 = sl * p.slice_rows; r1 = min(p.R, r0 + p.slice_rows);
  };

  if (warp == 0) {
    {
      int stage = 0; uint32_t phase = 0;
      for (int w = cluster_id; w < n_items; w += n_clusters) {
        int mt, nt, r0, r1; decode(w, mt, nt, r0, r1);
        for (int c = 0; c < p.C; ++c)
          for (int r = r0; r < r1; r += 64) {
            mbar_wait(empty + stage, phase ^ 1);
            uint8_t* sA = stages + stage * kW2StageBytes;
            const uint32_t lbar = mapa_u32(full + stage, 0);
            if (elect_one()) {
              if (rank == 0) mbar_expect_tx(full + stage, 2 * kW2StageBytes);
              tma2_load_3d(sA, &tmA, lbar, r, mt * 256 + (int)rank * 128, c);
              tma2_load_3d(sA + k2AStage, &tmB, lbar, r, nt * 256 + (int)rank * 128, c);
            }
            __syncwarp();
            if (++stage == kW2Stages) { stage = 0; phase ^= 1; }
          }
      }
    }
  } else if (warp == 1) {
    if (rank == 0) {
      int stage = 0; uint32_t phase = 0; int it = 0;
      constexpr uint32_t idesc = umma_idesc(Fmt<T>::umma, 0, 0, 256, 256);
      for (int w = cluster_id; w < n_items; w += n_clusters, ++it) {
        int mt, nt, r0, r1; decode(w, mt, nt, r0, r1);
        const int buf = it & 1; const uint32_t bphase = (it >> 1) & 1;
        mbar_wait_cluster(tempty + buf, bphase ^ 1);
        tc_fence_after();
        const uint32_t d0 = tmem_base + buf * 256;
        uint32_t acc = 0;
        for (int c = 0; c < p.C; ++c)
          for (int r = r0; r < r1; r += 64) {
            mbar_wait_cluster(full + stage, phase);
            tc_fence_after();
            const uint32_t sA = smem_u32(stages + stage * kW2StageBytes), sB = sA + k2AStage;
            if (elect_one()) {
#pragma unroll
              for (int k = 0; k < 4; ++k)
                tc2_mma(d0, umma_desc_sw128(sA + k * 32, 16, 1024), umma_desc_sw128(sB + k * 32, 16, 1024), idesc, (acc | k) ? 1u : 0u);
              tc2_commit(empty + stage);
            }
            __syncwarp();
            acc = 1;
            if (++stage == kW2Stages) { stage = 0; phase ^= 1; }
          }
        if (elect_one()) tc2_commit(tfull + buf);
        __syncwarp();
      }
    }
  } else {
    // epilogue warps 2..5 -> TMEM lane quarter (warp % 4); this CTA holds out units [128 rank, 128 rank + 128) of the tile
    const int q = warp & 3;
    int it = 0;
    for (int w = cluster_id; w < n_items; w += n_clusters, ++it) {
      int mt, nt, r0, r1; decode(w, mt, nt, r0, r1);
      const int buf = it & 1; const uint32_t bphase = (it >> 1) & 1;
      mbar_wait(tfull + buf, bphase);
      tc_fence_after();
      const uint32_t tbase = tmem_base + ((uint32_t)(q * 32) << 16) + buf * 256;
      float* dst = p.gW + (size_t)(mt * 256 + (int)rank * 128 + q * 32 + lane) * p.H + nt * 256;
      const float inv_sc = adj_inv_scale(p.amax);
      for (int n = 0; n < 256; n += 8) {
        float v[8];
        tmem_ld8(tbase + n, v);
        tmem_ld_wait();
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] *= inv_sc;
        asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst + n), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]) : "memory");
        asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst + n + 4), "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7]) : "memory");
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(mapa_u32(tempty + buf, 0));
    }
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == 1) { tc_fence_after(); tmem2_dealloc(tmem_base, 512); }
}

// =============================================================================================================
// host side
// =============================================================================================================
bool tc2_supported(const Launcher& L, int H) { return !L.one_cta && H % 256 == 0; }

template <typename T, int C, int MODE>
static void launch_jet2(Launcher& L, const CUtensorMap& a, const CUtensorMap& b, const CUtensorMap& t,
                        const Jet2Params& p) {
  using Cfg = Jet2Cfg<C, MODE>;
  static unsigned long long attr_done = 0;
  auto kern = jet2_layer_kernel<T, C, MODE>;
  ensure_smem_attr(L, kern, Cfg::kSmemBytes, attr_done);
  const int tiles = (p.H / 256) * p.n_row_tiles;
  const int clusters = std::min(tiles, L.num_sms / 2);
  kern<<<2 * clusters, k2Threads, Cfg::kSmemBytes, L.stream>>>(a, b, t, p);
  L.check(((MODE == 0 && !p.linear) || MODE == 4) ? "jet_layer_fwd" : (MODE == 2 || MODE == 5) ? "jet_layer_fwd_split" : "jet_layer_bwd");   // linear = a dgrad GEMM
}

template <int MODE>
static void dispatch_jet2(Launcher& L, int C, const CUtensorMap& a, const CUtensorMap& b, const CUtensorMap& t,
                          const Jet2Params& p) {
  if (C == 1) launch_jet2<__half, 1, MODE>(L, a, b, t, p);
  else if (C == 3) launch_jet2<__half, 3, MODE>(L, a, b, t, p);
  else launch_jet2<__half, 5, MODE>(L, a, b, t, p);
}

static void set_out_dot(Jet2Params& p, const OutDot* od) {
  p.w_out = od->w_out; p.b_out = od->b_out; p.o = od->o; p.o_stride = od->o_stride; p.valid = od->valid;
}

void tc2_layer_fwd(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* w16_l, const float* bias, const void* h_in, void* h_out,
                   const OutDot* od, bool linear, bool reverse) {
  CUtensorMap a, b;
  bool ok = weight_map(L, &a, precision, w16_l, H) && plane_map(L, &b, precision, h_in, H, R_ld, C, 32, 64, C, CU_TENSOR_MAP_SWIZZLE_64B);
  if (!ok) return;
  Jet2Params p{};
  p.H = H; p.n_row_tiles = R / 64; p.bias = bias; p.out = h_out; p.R_ld = R_ld; p.linear = linear ? 1 : 0; p.reverse = reverse ? 1 : 0;
  if (od) {
    CUtensorMap o = b;
    if (h_out && !plane_map(L, &o, precision, h_out, H, R_ld, C, 32, 32, C, CU_TENSOR_MAP_SWIZZLE_64B)) return;
    set_out_dot(p, od); dispatch_jet2<4>(L, C, a, b, o, p); return;
  }
  dispatch_jet2<0>(L, C, a, b, b, p);
}

void tc2_layer_fwd_split(Launcher& L, int precision, int H, int R, int R_ld, const void* w16_l, const float* bias, const void* h_in, void* h_out,
                         const OutDot* od) {
  CUtensorMap a, b;
  if (!(weight_map(L, &a, precision, w16_l, H) && plane_map(L, &b, precision, h_in, H, R_ld, 2, 32, 64, 2, CU_TENSOR_MAP_SWIZZLE_64B))) return;
  Jet2Params p{};
  p.H = H; p.n_row_tiles = R / 64; p.bias = bias; p.out = h_out; p.R_ld = R_ld;
  if (od) { set_out_dot(p, od); launch_jet2<__half, 2, 5>(L, a, b, b, p); return; }
  launch_jet2<__half, 2, 2>(L, a, b, b, p);
}

void tc2_layer_bwd(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* w16T_l, const void* ahat_in, const void* h_prev,
                   void* ahat_out, float* g_bias_prev, const float* amax, const FirstLayerFuse* fl) {
  CUtensorMap a, b, t;
  bool ok = weight_map(L, &a, precision, w16T_l, H) && plane_map(L, &b, precision, ahat_in, H, R_ld, C, 32, 64, C, CU_TENSOR_MAP_SWIZZLE_64B) &&
            plane_map(L, &t, precision, h_prev, H, R_ld, C, 32, 32, C, CU_TENSOR_MAP_SWIZZLE_64B);
  if (!ok) return;
  Jet2Params p{};
  p.H = H; p.n_row_tiles = R / 64; p.g_bias = g_bias_prev; p.amax = amax; p.out = ahat_out; p.R_ld = R_ld;
  if (fl) {
    p.xy = fl->xy; p.row0 = fl->row0; p.npts = fl->npts; p.in_dim = fl->in_dim; p.gW1 = fl->gW1; p.An = fl->An; p.per_sample = fl->per_sample;
    dispatch_jet2<3>(L, C, a, b, t, p);
    return;
  }
  dispatch_jet2<1>(L, C, a, b, t, p);
}

void tc2_wgrad(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* ahat, const void* h_prev, float* gW, const float* amax) {
  Wgrad2Params p{};
  p.H = H; p.C = C; p.R = R; p.gW = gW; p.amax = amax;
  const int n_tiles = (H / 256) * (H / 256);
  const int n_cl = L.num_sms / 2;
  // row slices: one work item per CTA (pair) when that fills >= 90 % of the machine, else two; every extra slice costs one
  // more fp32 red.add pass over the H x H gradient (measured on c2 / c3: 1 slice per CTA is 10 % faster than 2)
  const int units = n_cl;
  int slices = std::max(1, units / n_tiles);
  if (n_tiles * slices * 10 < units * 9) slices = std::max(1, (2 * units) / n_tiles);
  int slice_rows = ((R + slices - 1) / slices + 63) / 64 * 64;
  if (slice_rows < 64) slice_rows = 64;
  p.slice_rows = slice_rows; p.n_slices = (R + slice_rows - 1) / slice_rows;
  CUtensorMap a, b;
  if (!(plane_map(L, &a, precision, ahat, H, R_ld, C, 64, 128, 1, CU_TENSOR_MAP_SWIZZLE_128B) &&
        plane_map(L, &b, precision, h_prev, H, R_ld, C, 64, 128, 1, CU_TENSOR_MAP_SWIZZLE_128B)))
    return;
  const int smem = kW2Stages * kW2StageBytes + 1024 + 256;
  static unsigned long long attr_done = 0;
  const int clusters = std::min(n_tiles * p.n_slices, n_cl);
  ensure_smem_attr(L, wgrad2_kernel<__half>, smem, attr_done);
  wgrad2_kernel<__half><<<2 * clusters, 192, smem, L.stream>>>(a, b, p);
  L.check("wgrad");
}

}  // namespace pigan
