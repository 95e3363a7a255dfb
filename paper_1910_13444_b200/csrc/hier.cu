// NEXT-3 (R10): hierarchical multi-discriminator loss.  One generator, K critics;
// critic k scores the columns idx_k of the 2S-entry snapshot (the log k and u entries of its subdomain's sensors) with its
// own WGAN-GP loss, and the generator's loss is the weighted sum of the negative critics, w_k = 1 / (levels x subdomains in
// the level).  The critics run one after the other on ONE critic workspace (grouped small MLPs on one GPU): gather the
// sub-snapshots, run the critic kernels of the base step, scatter-add w_k grad_X D_k into the snapshot gradient.
#include "ctx.cuh"

namespace pigan {

namespace {

__global__ void gather_cols_kernel(const float* __restrict__ fake, const float* __restrict__ real, const int* __restrict__ idx, int N, int d_full,
                                   int d_sub, float* __restrict__ Xf, float* __restrict__ Xr) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N * d_sub) return;
  const int n = i / d_sub, col = idx[i - n * d_sub];
  Xf[i] = fake[(size_t)n * d_full + col];
  Xr[i] = real[(size_t)n * d_full + col];
}
// dX[n][idx[j]] += w * dXk[n][j]   (the columns of one critic are distinct; critics run one after the other)
__global__ void scatter_add_cols_kernel(const float* __restrict__ dXk, const int* __restrict__ idx, int N, int d_full, int d_sub, float w,
                                        float* __restrict__ dX) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N * d_sub) return;
  const int n = i / d_sub;
  dX[(size_t)n * d_full + idx[i - n * d_sub]] += w * dXk[i];
}
// folds one critic's accumulators (sum D fake, sum D real, sum (nu - 1)^2) into the totals and clears them
__global__ void fold_acc_kernel(double* __restrict__ acc, double* __restrict__ tot, int N, float lambda, float w) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const double df = acc[0] / N, dr = acc[1] / N, gp = lambda * acc[2] / N;
  tot[0] += df - dr + gp; tot[1] += w * df; tot[2] += w * dr; tot[3] += gp;
  acc[0] = 0.0; acc[1] = 0.0; acc[2] = 0.0;
}
__global__ void write_losses_hier_kernel(const double* __restrict__ tot, const double* __restrict__ acc, long long NP, float w_pde, float* __restrict__ losses) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const double lp = acc[3] / NP;
  losses[0] = (float)tot[0]; losses[1] = (float)tot[1]; losses[2] = (float)tot[2]; losses[3] = (float)tot[3];
  losses[4] = (float)(-tot[1] + w_pde * lp); losses[5] = (float)lp;
}

}  // namespace

void hier_critic_stage(pigan_ctx* c, const float* thD, const float* real, const float* eps, float* gD) {
  Launcher& L = c->L;
  const NetShape& ds = c->disc;
  const int N = c->cfg.n_samples, S = c->cfg.n_sensors, d_full = 2 * S, d_sub = ds.in_dim, HD = ds.H, K = c->hier.K;
  const size_t cnt = ds.count();
  cudaStream_t st = L.stream;
  cudaMemsetAsync(c->dX, 0, (size_t)N * d_full * 4, st);
  cudaMemsetAsync(c->htot, 0, 4 * sizeof(double), st);
  const int nb = (N * d_sub + 255) / 256;
  for (int k = 0; k < K; ++k) {
    const int* idx = c->hier.subsets + (size_t)k * d_sub;
    const float* th = thD + k * cnt;
    float* g = gD + k * cnt;
    const float w = c->hier.weights[k];
    gather_cols_kernel<<<nb, 256, 0, st>>>(c->xfake, real, idx, N, d_full, d_sub, c->hXf, c->hXr);
    L.check("gather_cols");
    if (critic_fused_supported(ds)) {
      critic_fused(L, ds, th, c->hXf, c->hXr, eps, N, 1, c->cfg.gp_lambda, c->cw, g, c->hdX, nullptr);
    } else {
      build_snapshots(L, c->hXf, c->hXr, eps, N, d_sub, c->cw.X);
      critic_forward(L, ds, th, c->cw.X, 3 * N, c->cw.g, c->cw.D);
      reduce_scores(L, c->cw.D, N, c->cw.acc);
      fill_seed(L, c->seed, N);
      const int gstride = 3 * N * HD;
      critic_backward(L, ds, th, c->cw.X, c->cw.g, 2 * N, gstride, c->seed, g, c->hdX, c->cw.t0, c->cw.t1);
      critic_gp(L, ds, th, c->cw.X + (size_t)2 * N * d_sub, c->cw.g + (size_t)2 * N * HD, N, gstride, c->cfg.gp_lambda, c->cw, g, nullptr);
    }
    scatter_add_cols_kernel<<<nb, 256, 0, st>>>(c->hdX, idx, N, d_full, d_sub, w, c->dX);
    L.check("scatter_add_cols");
    fold_acc_kernel<<<1, 32, 0, st>>>(c->cw.acc, c->htot, N, c->cfg.gp_lambda, w);
    L.check("fold_acc");
  }
}

void hier_write_losses(pigan_ctx* c, long long NP, float* losses) {
  write_losses_hier_kernel<<<1, 32, 0, c->L.stream>>>(c->htot, c->cw.acc, NP, c->cfg.pde_weight, losses);
  c->L.check("write_losses");
}

}  // namespace pigan
