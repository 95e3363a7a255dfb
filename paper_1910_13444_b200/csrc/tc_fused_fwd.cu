// Forward of a width-128 generator for a chunk of collocation rows in ONE kernel (
// P:153 is why the paper's rows are narrow and many): the first layer and every hidden tanh layer of a 64-row tile run
// back to back on one CTA, the activations never leave the SM between layers.
//
//   weights   W_2 .. W_L (16-bit, 32 KB each) are loaded ONCE per CTA and stay in shared memory (K-major, SW128).
//   act       the tile's current jet h^l as the B operand of the next layer's MMA: [k-block 2][channel C][64 units][64 rows],
//             MN-major, 128-byte swizzle -- exactly what a TMA box of 64 rows x 64 units x C lands as, so the same bytes are the
//             source of the TMA STORE that writes h^l to the activation stash (the reverse sweep needs every h^l: HBM sees one
//             write per plane and no read; layer by layer it was a write and a read).
//   per tile  epilogue warps compute the first layer from (x, y), Zp and W_1 (fp32, a1 / a2) into act; then for l = 2 .. L:
//             the MMA warp contracts W_l with act into TMEM (C channels stacked as GEMM columns, N = 64 C), the epilogue warps
//             (warp (q, hs): units [32 q, +32) = TMEM lanes, rows [32 hs, +32)) apply bias, tanh.approx and the chain rule O2
//             and write h^l over act, the store warp sends it to HBM.  A tile's layers are a serial chain (one accumulator,
//             one act buffer).  Measured on B200 (c2: 65536 rows, two launches instead of ten, 0.235 -> 0.149 ms): what a
//             layer of a tile waits for is the TMA store reading act (80 KB at the ~26 B/clk an SM's outbound path takes),
//             not the math -- elimination builds without tanh, chain rule, TMEM loads or packing run within 3 % of the full kernel.
// Versions of act are counted: h^l of the it-th tile of this CTA is version it * L + l - 1.
#include "tc_ptx.cuh"

namespace pigan {

constexpr int kFFMaxL = 5;                   // hidden layers: (L - 1) x 32 KB of weights + 80 KB of act fit 227 KB up to L = 5
constexpr int kFFEpi = 8;                    // epilogue warps: warp (q, hs) owns units [32 q, +32) (TMEM lanes) x kFFRows rows of the tile
constexpr int kFFRows = 256 / kFFEpi, kFFGroups = kFFRows / 8;   // 32 rows per warp in 4 groups of 8 (16 warps x 16 rows: measured, no faster)
constexpr int kFFThreads = (4 + kFFEpi) * 32; // warp 0: weights + stores, 1: MMA, 2: TMEM, 3: idle, 4..: epilogue

struct FusedFwdMaps {
  CUtensorMap w[kFFMaxL - 1];                // w[l - 2]: W_l [128][128] 16-bit, box 64 x 128, SW128
  CUtensorMap out[kFFMaxL];                  // out[l - 1]: planes of h^l, box 64 rows x 64 units x C, SW128
};

struct FusedFwdParams {
  int L;                                     // hidden layers
  int n_tiles;                               // R / 64
  int in_dim;                                // 2 + m
  const float* theta;                        // flat fp32 parameters of the net (W_1, b_1 .. b_L are read from here)
  long long b_off[kFFMaxL + 1];              // b_off[l]: offset of b_l, l = 1 .. L
  const float* Zp;                           // [N][128] z-part of the first layer (a1)
  const float* xy;                           // [npts][2], or [rows][2] when per_sample
  long long row0;                            // first global row of the chunk (multiple of 64)
  int npts, per_sample;
  // output layer (a4) in the epilogue of the last hidden layer: o_c[r] += sum_units w_out[unit] h^L_c[unit][r] (+ b_out on the value
  // channel); o is zeroed by the launcher; o == nullptr: no output dot
  const float* w_out; const float* b_out; float* o; long long o_stride;
};

template <typename T, int C>
__global__ void __launch_bounds__(kFFThreads, 1) fused_fwd128_kernel(const __grid_constant__ FusedFwdMaps maps, FusedFwdParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sW = smem;                                        // (L - 1) x [k-block 2][128 units][64 K]
  uint8_t* act = sW + (p.L - 1) * 32768;                     // [k-block 2][C][64 units][64 rows]
  uint64_t* bars = reinterpret_cast<uint64_t*>(act + 2 * C * 8192);
  uint64_t* wbar = bars;                                     // the resident weights have landed
  uint64_t* act_full = bars + 1;                             // 8 arrivals: the epilogue warps have written (and fenced) a version of act
  uint64_t* act_free = bars + 2;                             // 1 arrival: the store of that version has read act
  uint64_t* tfull = bars + 3;                                // commit: the accumulator of a layer is complete
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 4);

  const int warp = uniform_warp_idx(), lane = threadIdx.x & 31;
  const int n_my = (p.n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;

  if (warp == 0 && lane == 0) {
    for (int l = 2; l <= p.L; ++l) prefetch_tmap(&maps.w[l - 2]);
    for (int l = 1; l <= p.L; ++l) prefetch_tmap(&maps.out[l - 1]);
  }
  if (warp == 1 && lane == 0) {
    mbar_init(wbar, 1); mbar_init(act_full, kFFEpi); mbar_init(act_free, 1); mbar_init(tfull, 1);
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot, 0);

  if (warp == 0) {
    // ===================== weights once, then one TMA store per version of act =====================
    if (elect_one()) {
      mbar_expect_tx(wbar, (uint32_t)(p.L - 1) * 32768u);
      for (int l = 2; l <= p.L; ++l)
        for (int kb = 0; kb < 2; ++kb) tma_load_2d(sW + (l - 2) * 32768 + kb * 16384, &maps.w[l - 2], wbar, kb * 64, 0);
    }
    __syncwarp();
    uint32_t ver = 0;
    for (int it = 0; it < n_my; ++it) {
      const int t = (int)blockIdx.x + it * (int)gridDim.x;
      for (int l = 1; l <= p.L; ++l, ++ver) {
        mbar_wait(act_full, ver & 1);
        if (elect_one()) {
          tma_store_3d(&maps.out[l - 1], act, t * 64, 0, 0);
          tma_store_3d(&maps.out[l - 1], act + C * 8192, t * 64, 64, 0);
          tma_commit_group();
          tma_wait_read_all();                               // act may be overwritten (the MMA that reads it too is tracked by tfull)
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(act_free);
      }
    }
    if (elect_one()) tma_wait_all();                         // the last stores are complete before the CTA leaves
    __syncwarp();
  } else if (warp == 1) {
    // ===================== MMA issuer: layer l contracts W_l with version (h^{l-1}) of act =====================
    mbar_wait(wbar, 0);
    uint32_t ver = 0;
    for (int it = 0; it < n_my; ++it) {
      for (int l = 2; l <= p.L + 1; ++l, ++ver) {
        mbar_wait(act_full, ver & 1);                        // every version is awaited in order (a parity cannot tell v from v - 2)
        if (l > p.L) continue;                               // h^L has no consumer here
        tc_fence_after();
        const uint32_t aW = smem_u32(sW + (l - 2) * 32768), bA = smem_u32(act);
#pragma unroll
        for (int kb = 0; kb < 2; ++kb)
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const uint64_t ad = umma_desc_sw128(aW + kb * 16384 + k * 32, 16, 1024);            // K-major: +32 B per 16 elements
#pragma unroll
            for (int c0 = 0; c0 < C; c0 += 3) {
              const int nc = (C - c0) < 3 ? (C - c0) : 3;
              // MN-major: channel planes 8 KB apart (LBO), 8-unit groups 1 KB apart (SBO), 16 units = +2 KB
              const uint64_t bd = umma_desc_sw128(bA + kb * (C * 8192) + c0 * 8192 + k * 2048, 8192, 1024);
              if (elect_one()) tc_mma(tmem_base + c0 * 64, ad, bd, umma_idesc(Fmt<T>::umma, 0, 1, 128, nc * 64), (kb | k) ? 1u : 0u);
            }
          }
        if (elect_one()) tc_commit(tfull);
        __syncwarp();
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue: warp (q, hs) owns units [32 q, +32) (TMEM lanes) x rows [32 hs, +32) of the tile =====================
    const int e = warp - 4, q = e & 3, hs = e >> 2;
    const int u = q * 32 + lane;
    // this unit's row of an act plane: 128 bytes = 64 rows; 16-byte chunk j (8 rows) sits at (j ^ (u & 7))
    uint8_t* my_row = act + (u >> 6) * (C * 8192) + (u & 63) * 128;
    const uint32_t sw = (uint32_t)(u & 7);
    const uint32_t tbase = tmem_base + ((uint32_t)(q * 32) << 16) + hs * kFFRows;
    const float wx = p.theta[(size_t)u * p.in_dim], wy = p.theta[(size_t)u * p.in_dim + 1], b1 = p.theta[p.b_off[1] + u];
    const float wo = p.o ? p.w_out[u] : 0.f, bo = p.o ? p.b_out[0] : 0.f;
    uint32_t ver = 0, tf = 0;
    for (int it = 0; it < n_my; ++it) {
      const int t = (int)blockIdx.x + it * (int)gridDim.x;
      // ---- first layer (a1, a2): a = Zp[n] + b_1 + W_1[:,0] x + W_1[:,1] y; a_x = W_1[:,0], a_y = W_1[:,1], a_xx = a_yy = 0 ----
      {
        const long long grow = p.row0 + (long long)t * 64 + hs * kFFRows;       // a tile lies inside one latent sample (npts % 64 == 0)
        const int n = (int)(grow / p.npts);
        const float2* xyp = reinterpret_cast<const float2*>(p.xy) + (p.per_sample ? grow : grow - (long long)n * p.npts);
        const float zb = p.Zp[(size_t)n * 128 + u] + b1;
        if (ver > 0) mbar_wait(act_free, (ver - 1) & 1);     // the store of the previous tile's h^L has read act
#pragma unroll
        for (int rc = 0; rc < kFFGroups; ++rc) {
          float o[C][8];
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const float2 pt = __ldg(xyp + rc * 8 + i);       // same address in every lane: one broadcast load
            const float a0 = zb + wx * pt.x + wy * pt.y;
            float a[5] = {a0, wx, wy, 0.f, 0.f}, h[5];
            jet_act_fwd<C>(fast_tanh(a0), a, h);
#pragma unroll
            for (int c = 0; c < C; ++c) o[c][i] = h[c];
          }
          const uint32_t off = (((uint32_t)(hs * kFFGroups + rc)) ^ sw) << 4;
#pragma unroll
          for (int c = 0; c < C; ++c) sts128(my_row + c * 8192 + off, pack8<T>(o[c]));
        }
        fence_proxy_async();                                 // generic writes of act before the tensor core's and the TMA store's reads
        __syncwarp();
        if (lane == 0) mbar_arrive(act_full);
        ++ver;
      }
      // ---- hidden layers l = 2 .. L: h^l = tanh-jet(W_l h^{l-1} + b_l) ----
      for (int l = 2; l <= p.L; ++l) {
        const float bias = p.theta[p.b_off[l] + u];
        mbar_wait(tfull, tf & 1); ++tf;                      // the accumulator is complete: the MMAs have read act
        tc_fence_after();
        mbar_wait(act_free, (ver - 1) & 1);                  // ... and so has the store of h^{l-1}
        // the accumulator rows are pulled one group of 8 rows ahead of the math (every asm statement keeps program order, so
        // a load issued next to its wait exposes the TMEM latency once per group)
        float vv[2][C][8];
#pragma unroll
        for (int c = 0; c < C; ++c) tmem_ld8(tbase + c * 64, vv[0][c]);
#pragma unroll
        for (int rc = 0; rc < kFFGroups; ++rc) {
          float o[C][8];
          tmem_ld_wait();
          if (rc + 1 < kFFGroups) {
#pragma unroll
            for (int c = 0; c < C; ++c) tmem_ld8(tbase + c * 64 + (rc + 1) * 8, vv[(rc + 1) & 1][c]);
          }
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            float a[5], h[5];
#pragma unroll
            for (int c = 0; c < C; ++c) a[c] = vv[rc & 1][c][i];
            a[0] += bias;
            jet_act_fwd<C>(fast_tanh(a[0]), a, h);
#pragma unroll
            for (int c = 0; c < C; ++c) o[c][i] = h[c];
          }
          const uint32_t off = (((uint32_t)(hs * kFFGroups + rc)) ^ sw) << 4;
#pragma unroll
          for (int c = 0; c < C; ++c) sts128(my_row + c * 8192 + off, pack8<T>(o[c]));
          if (l == p.L && p.o) {
            // a4: the unrounded fp32 h^L_c times w_out[unit], summed over the warp's 32 units by a transposing shuffle reduction
            // (lane -> row 4 bit4 + 2 bit3 + bit2 of the group of 8), over the four unit quarters by fp32 atomics
            const int r = t * 64 + hs * kFFRows + rc * 8 + ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
#pragma unroll
            for (int c = 0; c < C; ++c) {
              float pv[8];
#pragma unroll
              for (int i = 0; i < 8; ++i) pv[i] = wo * o[c][i];
              float tot = warp_reduce8(pv, lane);
              if (c == 0 && q == 0) tot += bo;
              if ((lane & 3) == 0) atomicAdd(p.o + (size_t)c * p.o_stride + r, tot);
            }
          }
        }
        fence_proxy_async();
        tc_fence_before();                                   // this warp's TMEM reads are done before the next layer's MMAs overwrite them
        __syncwarp();
        if (lane == 0) mbar_arrive(act_full);
        ++ver;
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) { tc_fence_after(); tmem_dealloc(tmem_base, 512); }
}

// =============================================================================================================
// host side
// =============================================================================================================
bool tc_fused_fwd_supported(const Launcher& L, const NetShape& s, int C, const ChunkGeom& g) {
  (void)L;
  return s.H == 128 && (C == 3 || C == 5) && s.L >= 2 && s.L <= kFFMaxL && g.npts % 64 == 0 && g.R == g.valid && g.R > 0 && g.row0 % 64 == 0;
}

template <int C>
static void launch_fused_fwd(Launcher& L, const FusedFwdMaps& maps, const FusedFwdParams& p) {
  static unsigned long long attr_done = 0;
  auto kern = fused_fwd128_kernel<__half, C>;
  const int smem = (p.L - 1) * 32768 + 2 * C * 8192 + 1024 /*align*/ + 256 /*barriers*/;
  ensure_smem_attr(L, kern, (kFFMaxL - 1) * 32768 + 2 * C * 8192 + 1024 + 256, attr_done);
  kern<<<std::min(p.n_tiles, L.num_sms), kFFThreads, smem, L.stream>>>(maps, p);
  L.check("gen_fwd_fused");
}

void tc_fused_fwd(Launcher& L, int precision, int C, const NetShape& s, const float* theta, const void* const* w16 /*[L - 1]: W_2 .. W_L*/,
                  const float* Zp, const float* xy, const ChunkGeom& g, void* const* h /*[L]: planes of h^1 .. h^L*/, const OutDot* od) {
  FusedFwdMaps maps{};
  FusedFwdParams p{};
  for (int l = 2; l <= s.L; ++l)
    if (!weight_map(L, &maps.w[l - 2], precision, w16[l - 2], s.H)) return;
  for (int l = 1; l <= s.L; ++l) {
    if (!plane_map(L, &maps.out[l - 1], precision, h[l - 1], s.H, g.R_ld, C, 64, 64, C, CU_TENSOR_MAP_SWIZZLE_128B)) return;
    p.b_off[l] = (long long)s.b_off(l);
  }
  p.L = s.L; p.n_tiles = g.R / 64; p.in_dim = s.in_dim; p.theta = theta; p.Zp = Zp; p.xy = xy; p.row0 = g.row0; p.npts = g.npts;
  p.per_sample = g.per_sample;
  if (od) { p.w_out = od->w_out; p.b_out = od->b_out; p.o = od->o; p.o_stride = od->o_stride; }
  if (C == 3) launch_fused_fwd<3>(L, maps, p); else launch_fused_fwd<5>(L, maps, p);
}

}  // namespace pigan
