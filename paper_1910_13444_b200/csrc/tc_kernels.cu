// sm_100a tensor-core kernels of the jet MLP: tcgen05.mma with TMEM accumulators, operands
// staged by TMA, the tanh-jet chain rule (forward) or its adjoint (backward) fused into the epilogue.
//
// Orientation ("units as lanes"): D[unit (128 TMEM lanes)][(channel, row) columns] = W_tile[128 x K] . act[K x (C*64)].
//   A = 16-bit weights, K-major, 128B swizzle (TMA 2D box 64 x 128).
//   B = activation planes [channel][unit][row] -- rows contiguous, i.e. MN-major -- 128B swizzle (TMA 3D box
//       64 rows x 64 units x C channels): the C jet channels are stacked as extra GEMM columns of ONE tile pass.
//   An epilogue thread owns one unit (TMEM lane) and sees all C channels of a (row, unit) pair, so the chain rule
//   is thread-local; its outputs are contiguous along rows and leave through swizzled smem + TMA stores.
// wgrad: D[out unit][in unit] += sum_{c,row} ahat_c[out][row] h_c[in][row]; both operands K-major (rows contiguous).
#include "tc_ptx.cuh"

namespace pigan {

// =============================================================================================================
// jet layer kernel: forward (MODE 0) and dgrad + adjoint (MODE 1)
// =============================================================================================================
constexpr int kBM = 128;          // units per tile (TMEM lanes)
constexpr int kRT = 64;           // rows per tile
constexpr int kBK = 64;           // contraction elements per pipeline stage (128 B of K-major A)
constexpr int kAStage = kBM * kBK * 2;                 // 16 KB
constexpr int kBPlane = kBK * kRT * 2;                 // 8 KB per channel per stage
constexpr int kStgPlane = 32 * 64;                     // epilogue staging: 32 units x 32 rows x 2 B per warp per plane

template <int C> struct JetCfg {
  static constexpr int kNumStages = C == 5 ? 3 : 4;
  static constexpr int kStageBytes = kAStage + C * kBPlane;
  static constexpr int kCols = C * kRT;                               // accumulator columns of one tile
  static constexpr int kNumBuf = (2 * kCols <= 512) ? 2 : 1;          // TMEM double buffering when it fits
  static constexpr int kTmemCols = kNumBuf * kCols <= 64 ? 64 : kNumBuf * kCols <= 128 ? 128 : kNumBuf * kCols <= 256 ? 256 : 512;
  static constexpr int kStgBytes = 4 * C * kStgPlane;                 // 4 epilogue warps x C planes
  static constexpr int kSmemBytes = kNumStages * kStageBytes + kStgBytes + 1024 /*align*/ + 256 /*barriers*/;
};

struct JetParams {
  int H;                 // width (K and number of output units)
  int n_row_tiles;       // R / 64
  const float* bias;     // MODE 0: b_l
  float* g_bias;         // MODE 1: b_hat_{l-1}
  const float* amax;     // MODE 1, 3: block-scale source of the adjoint planes (common.cuh adj_inv_scale)
  // MODE 3 (MODE 1 + first-layer reduction, O4 'First layer'; see tc2_kernels.cu): ahat^1 is consumed in registers
  const float* xy; long long row0; int npts, in_dim, per_sample; float* gW1; float* An;
  int linear;            // MODE 0 only: plain GEMM, out_c = W in_c (no bias, no tanh) -- see tc2_kernels.cu
};

template <typename T, int C, int MODE>
__global__ void __launch_bounds__(256, 1) jet_layer_kernel(const __grid_constant__ CUtensorMap tmA,      // weights [H][H] 16-bit, box 64 x 128, SW128
                                                           const __grid_constant__ CUtensorMap tmB,      // input planes, box 64 rows x 64 units x C, SW128
                                                           const __grid_constant__ CUtensorMap tmO,      // MODE 0: h_out; MODE 1: ahat_out (box 32 x 32 x 1, SW64)
                                                           const __grid_constant__ CUtensorMap tmT,      // MODE 1: h_prev planes in
                                                           JetParams p) {
  using Cfg = JetCfg<C>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* stages = smem;
  uint8_t* staging = smem + Cfg::kNumStages * Cfg::kStageBytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(staging + Cfg::kStgBytes);
  uint64_t* full = bars;                                   // [kNumStages]
  uint64_t* empty = bars + Cfg::kNumStages;                // [kNumStages]
  uint64_t* tfull = empty + Cfg::kNumStages;               // [kNumBuf]
  uint64_t* tempty = tfull + Cfg::kNumBuf;                 // [kNumBuf]
  uint64_t* sbar = tempty + Cfg::kNumBuf;                  // [4] staging-load barriers (MODE 1), one per epilogue warp
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(sbar + 4);

  const int warp = uniform_warp_idx(), lane = threadIdx.x & 31;
  const int n_ut = p.H / kBM;
  const int n_tiles = n_ut * p.n_row_tiles;
  const int n_kb = p.H / kBK;

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmA); prefetch_tmap(&tmB); prefetch_tmap(&tmO);
    if (MODE == 1 || MODE == 3) prefetch_tmap(&tmT);
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < Cfg::kNumStages; ++i) { mbar_init(full + i, 1); mbar_init(empty + i, 1); }
    for (int i = 0; i < Cfg::kNumBuf; ++i) { mbar_init(tfull + i, 1); mbar_init(tempty + i, 4); }
    for (int i = 0; i < 4; ++i) mbar_init(sbar + i, 1);
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc(tmem_slot, Cfg::kTmemCols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot, 0);       // uniform: TMEM addresses live in uniform registers

  if (warp == 0) {
    // ===================== TMA producer (converged warp, one elected lane issues; see tc_ptx.cuh) =====================
    {
      int stage = 0; uint32_t phase = 0;
      for (int t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        const int ut = t % n_ut, rt = t / n_ut;
        for (int kb = 0; kb < n_kb; ++kb) {
          mbar_wait(empty + stage, phase ^ 1);
          uint8_t* sA = stages + stage * Cfg::kStageBytes;
          if (elect_one()) {
            mbar_expect_tx(full + stage, Cfg::kStageBytes);
            tma_load_2d(sA, &tmA, full + stage, kb * kBK, ut * kBM);
            tma_load_3d(sA + kAStage, &tmB, full + stage, rt * kRT, kb * kBK, 0);
          }
          __syncwarp();
          if (++stage == Cfg::kNumStages) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (converged warp, one elected lane issues) =====================
    {
      int stage = 0; uint32_t phase = 0; int it = 0;
      for (int t = blockIdx.x; t < n_tiles; t += gridDim.x, ++it) {
        const int buf = it % Cfg::kNumBuf;
        const uint32_t bphase = (it / Cfg::kNumBuf) & 1;
        mbar_wait(tempty + buf, bphase ^ 1);                 // epilogue has drained this accumulator
        tc_fence_after();
        const uint32_t d0 = tmem_base + buf * Cfg::kCols;
        for (int kb = 0; kb < n_kb; ++kb) {
          mbar_wait(full + stage, phase);
          tc_fence_after();
          const uint32_t sA = smem_u32(stages + stage * Cfg::kStageBytes), sB = sA + kAStage;
#pragma unroll
          for (int k = 0; k < kBK / 16; ++k) {
            const uint64_t ad = umma_desc_sw128(sA + k * 32, 16, 1024);                      // K-major: +32 B per 16 elements
            const uint32_t acc = (kb | k) ? 1u : 0u;
            // N is issued in groups of <= 3 channel blocks (N <= 256); channel blocks are 8 KB apart (LBO)
#pragma unroll
            for (int c0 = 0; c0 < C; c0 += 3) {
              const int nc = (C - c0) < 3 ? (C - c0) : 3;
              const uint64_t bd = umma_desc_sw128(sB + c0 * kBPlane + k * 2048, kBPlane, 1024);   // MN-major: +16 k-rows of 128 B
              if (elect_one()) tc_mma(d0 + c0 * kRT, ad, bd, umma_idesc(Fmt<T>::umma, 0, 1, kBM, nc * kRT), acc);
            }
          }
          if (elect_one()) tc_commit(empty + stage);         // frees the smem slot when these MMAs retire
          __syncwarp();
          if (++stage == Cfg::kNumStages) { stage = 0; phase ^= 1; }
        }
        if (elect_one()) tc_commit(tfull + buf);             // accumulator complete
        __syncwarp();
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue: 4 warps, warp q owns TMEM lanes / units [32q, 32q+32) =====================
    const int q = warp - 4;
    uint8_t* stg = staging + q * (C * kStgPlane);
    const uint32_t swz = (uint32_t)((lane >> 1) & 3);       // 64B swizzle of a 64-byte row: chunk ^= (row >> 1) & 3
    uint8_t* my_row = stg + lane * 64;
    uint32_t sphase = 0;
    int it = 0;
    for (int t = blockIdx.x; t < n_tiles; t += gridDim.x, ++it) {
      const int ut = t % n_ut, rt = t / n_ut;
      const int buf = it % Cfg::kNumBuf;
      const uint32_t bphase = (it / Cfg::kNumBuf) & 1;
      const int unit0 = ut * kBM + q * 32, unit = unit0 + lane;
      const uint32_t tbase = tmem_base + ((uint32_t)(q * 32) << 16) + buf * Cfg::kCols;
      float bias = 0.f, bias_acc = 0.f;
      if ((MODE == 0 || MODE == 2) && p.bias) bias = p.bias[unit];

      auto issue_stage_loads = [&](int hf) {                 // MODE 1: the previous layer's output jet h^{l-1} -> staging
        if (elect_one()) {
          tma_wait_read_all();                               // earlier stores have finished reading the staging buffer
          mbar_expect_tx(sbar + q, C * kStgPlane);
          for (int c = 0; c < C; ++c) tma_load_3d(stg + c * kStgPlane, &tmT, sbar + q, rt * kRT + hf * 32, unit0, c);
        }
      };
      if (MODE == 1 || MODE == 3) issue_stage_loads(0);
      float sx = 0.f, sy = 0.f;                              // MODE 3
      mbar_wait(tfull + buf, bphase);
      tc_fence_after();

#pragma unroll 1
      for (int hf = 0; hf < 2; ++hf) {
        if (MODE == 0) {
          // ---- h_c = tanh-jet(a_c) ----
          if (elect_one()) tma_wait_read_all();
          __syncwarp();
#pragma unroll 1
          for (int rc = 0; rc < 4; ++rc) {
            float v[C][8], o[C][8];
#pragma unroll
            for (int c = 0; c < C; ++c) tmem_ld8(tbase + c * kRT + hf * 32 + rc * 8, v[c]);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              float a[5], h[5];
#pragma unroll
              for (int c = 0; c < C; ++c) a[c] = v[c][i];
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
            const uint32_t off = ((uint32_t)rc ^ swz) << 4;
#pragma unroll
            for (int c = 0; c < C; ++c) *reinterpret_cast<uint4*>(my_row + c * kStgPlane + off) = pack8<T>(o[c]);
          }
          fence_proxy_async();
          __syncwarp();
          if (elect_one()) {
            for (int c = 0; c < C; ++c) tma_store_3d(&tmO, stg + c * kStgPlane, rt * kRT + hf * 32, unit0, c);
            tma_commit_group();
          }
        } else if (MODE == 2) {
          // ---- value-only layer with split activations: a = W (h_hi + h_lo) + b; t = tanh a; t_hi = rn16(t), t_lo = rn16(t - t_hi) ----
          if (elect_one()) tma_wait_read_all();
          __syncwarp();
#pragma unroll 1
          for (int rc = 0; rc < 4; ++rc) {
            float v0[8], v1[8], hi[8], lo[8];
            tmem_ld8(tbase + hf * 32 + rc * 8, v0);
            tmem_ld8(tbase + kRT + hf * 32 + rc * 8, v1);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const float t = tanhf(v0[i] + v1[i] + bias);
              hi[i] = to_f<T>(from_f<T>(t));
              lo[i] = t - hi[i];
            }
            const uint32_t off = ((uint32_t)rc ^ swz) << 4;
            *reinterpret_cast<uint4*>(my_row + off) = pack8<T>(hi);
            *reinterpret_cast<uint4*>(my_row + kStgPlane + off) = pack8<T>(lo);
          }
          fence_proxy_async();
          __syncwarp();
          if (elect_one()) {
            tma_store_3d(&tmO, stg, rt * kRT + hf * 32, unit0, 0);
            tma_store_3d(&tmO, stg + kStgPlane, rt * kRT + hf * 32, unit0, 1);
            tma_commit_group();
          }
        } else {
          // ---- adjoint of the previous layer's tanh: ahat^{l-1} = J^T hhat^{l-1} ----
          if (hf == 1) issue_stage_loads(1);
          __syncwarp();
          mbar_wait(sbar + q, sphase); sphase ^= 1;
          const float2* xyp = MODE == 3 ? reinterpret_cast<const float2*>(p.xy) + (p.per_sample ? (p.row0 + rt * kRT + hf * 32) : (p.row0 + rt * kRT + hf * 32) % p.npts) : nullptr;
#pragma unroll 1
          for (int rc = 0; rc < 4; ++rc) {
            float hh[C][8], hp[C][8], o[C][8];
#pragma unroll
            for (int c = 0; c < C; ++c) tmem_ld8(tbase + c * kRT + hf * 32 + rc * 8, hh[c]);
            const uint32_t off = ((uint32_t)rc ^ swz) << 4;
#pragma unroll
            for (int c = 0; c < C; ++c) unpack8<T>(*reinterpret_cast<const uint4*>(my_row + c * kStgPlane + off), hp[c]);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              float hx[5], hj[5], aa[5];
#pragma unroll
              for (int c = 0; c < C; ++c) { hx[c] = hh[c][i]; hj[c] = hp[c][i]; }
              jet_act_bwd<C>(hj, hx, aa);
              bias_acc += aa[0];
              if (MODE == 3) {
                const float2 q2 = __ldg(xyp + rc * 8 + i);   // same address in every lane: one broadcast load
                sx = fmaf(aa[0], q2.x, sx); sy = fmaf(aa[0], q2.y, sy);
                if (C >= 3) { sx += aa[1]; sy += aa[2]; }
              }
#pragma unroll
              for (int c = 0; c < C; ++c) o[c][i] = aa[c];
            }
            if (MODE == 1) {
#pragma unroll
              for (int c = 0; c < C; ++c) *reinterpret_cast<uint4*>(my_row + c * kStgPlane + off) = pack8<T>(o[c]);
            }
          }
          if (MODE == 1) {
            fence_proxy_async();
            __syncwarp();
            if (elect_one()) {
              for (int c = 0; c < C; ++c) tma_store_3d(&tmO, stg + c * kStgPlane, rt * kRT + hf * 32, unit0, c);
              tma_commit_group();
            }
          } else {
            __syncwarp();                                    // every lane is done reading the staging planes before they are refilled
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(tempty + buf);
      if (MODE == 1 || MODE == 3) atomicAdd(p.g_bias + unit, bias_acc * adj_inv_scale(p.amax));
      if (MODE == 3) {
        const float inv = adj_inv_scale(p.amax);
        atomicAdd(p.An + (size_t)((p.row0 + rt * kRT) / p.npts) * p.H + unit, bias_acc * inv);
        atomicAdd(p.gW1 + (size_t)unit * p.in_dim, sx * inv);
        atomicAdd(p.gW1 + (size_t)unit * p.in_dim + 1, sy * inv);
      }
    }
    __syncwarp();
    if (elect_one()) tma_wait_all();                         // global writes of the last stores are complete before exit
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) { tc_fence_after(); tmem_dealloc(tmem_base, Cfg::kTmemCols); }
}

// =============================================================================================================
// wgrad kernel: gW[j][k] += sum_{c, r} ahat_c[j][r] h_c[k][r]
// =============================================================================================================
constexpr int kWStages = 4;
struct WgradParams {
  int H, C;
  int NW;              // output tile width: 256 when it divides H, else 128
  int n_slices;        // row slices
  int slice_rows;      // rows per slice (multiple of 64)
  int R;               // rows of the chunk (multiple of 64)
  float* gW;           // [H][H] fp32
  const float* amax;   // block-scale source of the adjoint planes
};

template <typename T>
__global__ void __launch_bounds__(192, 1) wgrad_kernel(const __grid_constant__ CUtensorMap tmA,    // ahat planes, box 64 rows x 128 units x 1, SW128
                                                       const __grid_constant__ CUtensorMap tmB,    // h_prev planes, box 64 rows x NW units x 1, SW128
                                                       WgradParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int stage_bytes = kAStage + p.NW * 128;
  uint8_t* stages = smem;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kWStages * (kAStage + 256 * 128));
  uint64_t* full = bars; uint64_t* empty = bars + kWStages; uint64_t* tfull = empty + kWStages; uint64_t* tempty = tfull + 2;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 2);
  const int warp = uniform_warp_idx(), lane = threadIdx.x & 31;
  const int n_mt = p.H / kBM, n_nt = p.H / p.NW;
  const int n_items = n_mt * n_nt * p.n_slices;

  if (warp == 0 && lane == 0) { prefetch_tmap(&tmA); prefetch_tmap(&tmB); }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < kWStages; ++i) { mbar_init(full + i, 1); mbar_init(empty + i, 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(tfull + i, 1); mbar_init(tempty + i, 4); }
    fence_barrier_init();
  }
  __syncwarp();
  if (warp == 1) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot, 0);       // uniform: TMEM addresses live in uniform registers

  auto decode = [&](int w, int& mt, int& nt, int& r0, int& r1) {
    const int tile = w % (n_mt * n_nt), sl = w / (n_mt * n_nt);
    mt = tile % n_mt; nt = tile / n_mt;
    r0 = sl * p.slice_rows; r1 = min(p.R, r0 + p.slice_rows);
  };

  if (warp == 0) {
    {
      int stage = 0; uint32_t phase = 0;
      for (int w = blockIdx.x; w < n_items; w += gridDim.x) {
        int mt, nt, r0, r1; decode(w, mt, nt, r0, r1);
        for (int c = 0; c < p.C; ++c)
          for (int r = r0; r < r1; r += 64) {
            mbar_wait(empty + stage, phase ^ 1);
            uint8_t* sA = stages + stage * stage_bytes;
            if (elect_one()) {
              mbar_expect_tx(full + stage, stage_bytes);
              tma_load_3d(sA, &tmA, full + stage, r, mt * kBM, c);
              tma_load_3d(sA + kAStage, &tmB, full + stage, r, nt * p.NW, c);
            }
            __syncwarp();
            if (++stage == kWStages) { stage = 0; phase ^= 1; }
          }
      }
    }
  } else if (warp == 1) {
    {
      int stage = 0; uint32_t phase = 0; int it = 0;
      const uint32_t idesc = umma_idesc(Fmt<T>::umma, 0, 0, kBM, p.NW);
      for (int w = blockIdx.x; w < n_items; w += gridDim.x, ++it) {
        int mt, nt, r0, r1; decode(w, mt, nt, r0, r1);
        const int buf = it & 1; const uint32_t bphase = (it >> 1) & 1;
        mbar_wait(tempty + buf, bphase ^ 1);
        tc_fence_after();
        const uint32_t d0 = tmem_base + buf * 256;
        uint32_t acc = 0;
        for (int c = 0; c < p.C; ++c)
          for (int r = r0; r < r1; r += 64) {
            mbar_wait(full + stage, phase);
            tc_fence_after();
            const uint32_t sA = smem_u32(stages + stage * stage_bytes), sB = sA + kAStage;
            if (elect_one()) {
#pragma unroll
              for (int k = 0; k < 4; ++k)
                tc_mma(d0, umma_desc_sw128(sA + k * 32, 16, 1024), umma_desc_sw128(sB + k * 32, 16, 1024), idesc, (acc | k) ? 1u : 0u);
              tc_commit(empty + stage);
            }
            __syncwarp();
            acc = 1;
            if (++stage == kWStages) { stage = 0; phase ^= 1; }
          }
        if (elect_one()) tc_commit(tfull + buf);
        __syncwarp();
      }
    }
  } else {
    // epilogue warps 2..5 -> TMEM lane quarter (warp % 4)
    const int q = warp & 3;
    int it = 0;
    for (int w = blockIdx.x; w < n_items; w += gridDim.x, ++it) {
      int mt, nt, r0, r1; decode(w, mt, nt, r0, r1);
      const int buf = it & 1; const uint32_t bphase = (it >> 1) & 1;
      mbar_wait(tfull + buf, bphase);
      tc_fence_after();
      const uint32_t tbase = tmem_base + ((uint32_t)(q * 32) << 16) + buf * 256;
      float* dst = p.gW + (size_t)(mt * kBM + q * 32 + lane) * p.H + nt * p.NW;
      const float inv_sc = adj_inv_scale(p.amax);
      for (int n = 0; n < p.NW; n += 8) {
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
      if (lane == 0) mbar_arrive(tempty + buf);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) { tc_fence_after(); tmem_dealloc(tmem_base, 512); }
}

// =============================================================================================================
// 16-bit weight copies: W_l and W_l^T for l = 2..L
// =============================================================================================================
template <typename T>
__global__ void __launch_bounds__(256) convert_weights_kernel(NetShape s, const float* __restrict__ theta, T* __restrict__ w16) {
  __shared__ float tile[32][33];
  const int l = blockIdx.z + 2, H = s.H;
  const float* W = theta + s.W_off(l);
  T* out = w16 + (size_t)(l - 2) * 2 * H * H;
  T* outT = out + (size_t)H * H;
  const int bx = blockIdx.x * 32, by = blockIdx.y * 32, tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  for (int i = ty; i < 32; i += 8) {
    const float v = W[(size_t)(by + i) * H + bx + tx];
    tile[i][tx] = v;
    out[(size_t)(by + i) * H + bx + tx] = from_f<T>(v);
  }
  __syncthreads();
  for (int i = ty; i < 32; i += 8) outT[(size_t)(bx + i) * H + by + tx] = from_f<T>(tile[tx][i]);
}

void tc_convert_weights(Launcher& L, int precision, const NetShape& s, const float* theta, void* w16) {
  if (s.L < 2) return;
  dim3 grid(s.H / 32, s.H / 32, s.L - 1);
  (void)precision;   // PIGAN_FP16 is the only 16-bit mode (pigan_create refuses PIGAN_BF16)
  convert_weights_kernel<__half><<<grid, 256, 0, L.stream>>>(s, theta, (__half*)w16);
  L.check("convert_weights");
}

// =============================================================================================================
// host side: tensor maps and launches
// =============================================================================================================
bool tc_supported(int H, std::string* why) {
  if (H % 128 != 0) { if (why) *why = "16-bit precision needs a width that is a multiple of 128"; return false; }
  return true;
}

template <typename T, int C, int MODE>
static void launch_jet(Launcher& L, const CUtensorMap& a, const CUtensorMap& b, const CUtensorMap& o, const CUtensorMap& t,
                       const JetParams& p) {
  using Cfg = JetCfg<C>;
  static unsigned long long attr_done = 0;
  auto kern = jet_layer_kernel<T, C, MODE>;
  ensure_smem_attr(L, kern, Cfg::kSmemBytes, attr_done);
  const int tiles = (p.H / kBM) * p.n_row_tiles;
  const int grid = std::min(tiles, L.num_sms);
  kern<<<grid, 256, Cfg::kSmemBytes, L.stream>>>(a, b, o, t, p);
  L.check((MODE == 0 && !p.linear) ? "jet_layer_fwd" : MODE == 2 ? "jet_layer_fwd_split" : "jet_layer_bwd");   // linear = a dgrad GEMM
}

template <int MODE>
static void dispatch_jet(Launcher& L, int precision, int C, const CUtensorMap& a, const CUtensorMap& b, const CUtensorMap& o,
                         const CUtensorMap& t, const JetParams& p) {
#define PIGAN_JET(TT)                                                  \
  if (C == 1) launch_jet<TT, 1, MODE>(L, a, b, o, t, p);            \
  else if (C == 3) launch_jet<TT, 3, MODE>(L, a, b, o, t, p);       \
  else launch_jet<TT, 5, MODE>(L, a, b, o, t, p)
  (void)precision;                                          // both 16-bit modes compute with fp16 operands
  PIGAN_JET(__half);
#undef PIGAN_JET
}

bool tc_out_dot_fusable(const Launcher& L, int H) { return tc2_supported(L, H); }   // the one-CTA kernels keep the separate out_fwd pass

void tc_layer_fwd(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* w16_l, const float* bias, const void* h_in, void* h_out,
                  const OutDot* od, bool linear, bool reverse) {
  if (R <= 0) return;
  if (tc2_supported(L, H)) { tc2_layer_fwd(L, precision, C, H, R, R_ld, w16_l, bias, h_in, h_out, od, linear, reverse); return; }
  CUtensorMap a, b, o;
  bool ok = weight_map(L, &a, precision, w16_l, H) && plane_map(L, &b, precision, h_in, H, R_ld, C, kRT, kBK, C, CU_TENSOR_MAP_SWIZZLE_128B) &&
            plane_map(L, &o, precision, h_out, H, R_ld, C, 32, 32, 1, CU_TENSOR_MAP_SWIZZLE_64B);
  if (!ok) return;
  JetParams p{};
  p.H = H; p.n_row_tiles = R / kRT; p.bias = bias; p.linear = linear ? 1 : 0;
  dispatch_jet<0>(L, precision, C, a, b, o, o, p);
}

// value-only layer on split activations (2 planes: hi, lo) -> 2 planes; used where the snapshot X_fake is built
void tc_layer_fwd_split(Launcher& L, int precision, int H, int R, int R_ld, const void* w16_l, const float* bias, const void* h_in, void* h_out,
                        const OutDot* od) {
  if (R <= 0) return;
  if (tc2_supported(L, H)) { tc2_layer_fwd_split(L, precision, H, R, R_ld, w16_l, bias, h_in, h_out, od); return; }
  CUtensorMap a, b, o;
  if (!(weight_map(L, &a, precision, w16_l, H) && plane_map(L, &b, precision, h_in, H, R_ld, 2, kRT, kBK, 2, CU_TENSOR_MAP_SWIZZLE_128B) &&
        plane_map(L, &o, precision, h_out, H, R_ld, 2, 32, 32, 1, CU_TENSOR_MAP_SWIZZLE_64B)))
    return;
  JetParams p{};
  p.H = H; p.n_row_tiles = R / kRT; p.bias = bias;
  launch_jet<__half, 2, 2>(L, a, b, o, o, p);
}

bool tc_first_layer_fusable(int H, const ChunkGeom& g) { return H % 128 == 0 && g.npts % 64 == 0 && g.R == g.valid && g.R > 0; }

void tc_layer_bwd(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* w16T_l, const void* ahat_in, const void* h_prev,
                  void* ahat_out, float* g_bias_prev, const float* amax, const FirstLayerFuse* fl) {
  if (R <= 0) return;
  if (tc2_supported(L, H)) { tc2_layer_bwd(L, precision, C, H, R, R_ld, w16T_l, ahat_in, h_prev, ahat_out, g_bias_prev, amax, fl); return; }
  CUtensorMap a, b, o, t;
  bool ok = weight_map(L, &a, precision, w16T_l, H) && plane_map(L, &b, precision, ahat_in, H, R_ld, C, kRT, kBK, C, CU_TENSOR_MAP_SWIZZLE_128B) &&
            plane_map(L, &o, precision, ahat_out, H, R_ld, C, 32, 32, 1, CU_TENSOR_MAP_SWIZZLE_64B) &&
            plane_map(L, &t, precision, h_prev, H, R_ld, C, 32, 32, 1, CU_TENSOR_MAP_SWIZZLE_64B);
  if (!ok) return;
  JetParams p{};
  p.H = H; p.n_row_tiles = R / kRT; p.g_bias = g_bias_prev; p.amax = amax;
  if (fl) {
    p.xy = fl->xy; p.row0 = fl->row0; p.npts = fl->npts; p.in_dim = fl->in_dim; p.gW1 = fl->gW1; p.An = fl->An; p.per_sample = fl->per_sample;
    dispatch_jet<3>(L, precision, C, a, b, o, t, p);
    return;
  }
  dispatch_jet<1>(L, precision, C, a, b, o, t, p);
}

void tc_wgrad(Launcher& L, int precision, int C, int H, int R, int R_ld, const void* ahat, const void* h_prev, float* gW, const float* amax) {
  if (R <= 0) return;
  if (tc2_supported(L, H)) { tc2_wgrad(L, precision, C, H, R, R_ld, ahat, h_prev, gW, amax); return; }
  WgradParams p{};
  p.H = H; p.C = C; p.NW = (H % 256 == 0) ? 256 : 128; p.R = R; p.gW = gW; p.amax = amax;   // NW must divide H (H = 384, 640, ...)
  const int n_tiles = (H / kBM) * (H / p.NW);
  // row slices: one work item per CTA (pair) when that fills >= 90 % of the machine, else two; every extra slice costs one
  // more fp32 red.add pass over the H x H gradient (measured on c2 / c3: 1 slice per CTA is 10 % faster than 2)
  const int units = L.num_sms;
  int slices = std::max(1, units / n_tiles);
  if (n_tiles * slices * 10 < units * 9) slices = std::max(1, (2 * units) / n_tiles);
  int slice_rows = ((R + slices - 1) / slices + 63) / 64 * 64;
  if (slice_rows < 64) slice_rows = 64;
  p.slice_rows = slice_rows; p.n_slices = (R + slice_rows - 1) / slice_rows;
  CUtensorMap a, b;
  if (!(plane_map(L, &a, precision, ahat, H, R_ld, C, 64, kBM, 1, CU_TENSOR_MAP_SWIZZLE_128B) &&
        plane_map(L, &b, precision, h_prev, H, R_ld, C, 64, p.NW, 1, CU_TENSOR_MAP_SWIZZLE_128B)))
    return;
  const int smem = kWStages * (kAStage + 256 * 128) + 1024 + 256;
  static unsigned long long attr_done = 0;
  const int grid = std::min(n_tiles * p.n_slices, L.num_sms);
  ensure_smem_attr(L, wgrad_kernel<__half>, smem, attr_done);
  wgrad_kernel<__half><<<grid, 192, smem, L.stream>>>(a, b, p);
  L.check("wgrad");
}

}  // namespace pigan
