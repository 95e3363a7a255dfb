// pigan_darcy_residual_static: the Darcy residual (a5, Eq. 1) for hosts that may not allocate device memory.
//
// WHO THIS IS FOR.  Every other entry point of the library needs a pigan_ctx, and pigan_create cudaMallocs the context's
// workspaces.  Some programs that want to evaluate the residual cannot do that:
//   - a plug-in living inside a solver, a simulator or a serving process whose owner grabbed (nearly) all of the GPU's memory
//     for its own pool at start-up: cudaMalloc then fails, or the host's rules forbid calling it at all;
//   - a control or time-stepping loop with a latency budget: cudaMalloc / cudaFree may synchronise the whole device and take
//     an unpredictable time, so such loops keep every allocation out of their steady state.
// Those callers own the input and output buffers already; what they lack is the few kilobytes of SCRATCH the reduction of
// mean r^2 needs.  Here that scratch is a fixed array compiled into the library image (below), so the call allocates
// nothing: no cudaMalloc, no cudaFree, no library routine that allocates.
//
// THE PRICE.  The array has a fixed size, so the problem size is bounded (PIGAN_STATIC_MAX_ROWS rows); every GPU onto which the
// library's device code is loaded carries the array (about 128 KiB) until the process exits; and ALL calls on a device share it.
// The array still holds whatever the previous call left there; the call clears the one word that must start at zero (the
// ticket counter) itself.  Two calls that overlap on the same GPU (different streams, or different host threads on different
// streams) would race on the array: callers must order them, e.g. by using one stream.
//
// This file does not touch, and is not used by, the context-based path (api.cu / simt_kernels.cu).
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "pigan.h"

namespace {

constexpr int kThreads = 256;
constexpr int kRowsPerThread = 4;
constexpr int kRowsPerBlock = kThreads * kRowsPerThread;                       // 1024
constexpr long long kMaxRows = PIGAN_STATIC_MAX_ROWS;                          // 2^24
constexpr int kMaxBlocks = (int)(kMaxRows / kRowsPerBlock);                    // 16384 partial sums
constexpr int kHeaderDoubles = 32;                                             // 256 bytes: word 0 is the ticket counter
constexpr int kMaxDevices = 64;

// The scratch.  doubles [0, 32): header (the first 4 bytes are the ticket counter, the rest is padding so that the partial sums
// start on their own 256-byte line); doubles [32, 32 + 16384): one partial sum of r^2 per thread block.
// NOTE for whoever edits the host code below: in HOST code the name `g_residual_scratch` is only a handle the runtime uses to
// look the array up -- it is not a device address.  Handing `g_residual_scratch` itself to a kernel or to cudaMemsetAsync would
// make the GPU fault or, on systems where the GPU can reach host memory, quietly work on the wrong memory.  The device address
// comes from cudaGetSymbolAddress (scratch_of_current_device below).  Device code may use the name directly.
static __device__ __align__(256) double g_residual_scratch[kHeaderDoubles + kMaxBlocks];

thread_local char t_err[256] = "";

pigan_status fail(pigan_status s, const char* msg) {
  snprintf(t_err, sizeof t_err, "%s", msg);
  return s;
}

pigan_status fail_cuda(const char* what, cudaError_t e) {
  snprintf(t_err, sizeof t_err, "%s: %s", what, cudaGetErrorString(e));
  cudaGetLastError();
  return PIGAN_ERR_CUDA;
}

// Same arithmetic, in the same order, as residual_kernel (simt_kernels.cu): r = exp(Y)(Y_x u_x + Y_y u_y + u_xx + u_yy) - f.
// Each block writes the sum of its rows' r^2 to its own slot of the scratch; the block that draws the last ticket adds the
// slots up in a fixed order (so the mean does not depend on the order in which blocks finish) and writes mean r^2.
__global__ void __launch_bounds__(kThreads) residual_static_kernel(const float* __restrict__ Y, const float* __restrict__ U,
                                                                   const float* __restrict__ f, int total, long long plane, int npts,
                                                                   float* __restrict__ r_out, float* __restrict__ mean_sq,
                                                                   double* __restrict__ scratch) {
  __shared__ double red[kThreads / 32];
  __shared__ bool is_last;
  double sq = 0.0;
  const int base = blockIdx.x * kRowsPerBlock + threadIdx.x;
#pragma unroll
  for (int i = 0; i < kRowsPerThread; ++i) {
    const int r = base + i * kThreads;
    if (r < total) {
      const int p = r % npts;
      const float y0 = Y[r], yx = Y[plane + r], yy = Y[2 * plane + r];
      const float ux = U[plane + r], uy = U[2 * plane + r], uxx = U[3 * plane + r], uyy = U[4 * plane + r];
      const float k = expf(y0);
      const float D = fmaf(yx, ux, fmaf(yy, uy, uxx + uyy));
      const float res = fmaf(k, D, -f[p]);
      if (r_out) r_out[r] = res;
      sq += (double)res * (double)res;
    }
  }
  if (!mean_sq) return;                                                        // uniform over the grid
  unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch);
  double* partial = scratch + kHeaderDoubles;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = sq;
  __syncthreads();
  if (threadIdx.x == 0) {
    double v = 0.0;
#pragma unroll
    for (int w = 0; w < kThreads / 32; ++w) v += red[w];
    partial[blockIdx.x] = v;
    __threadfence();                                                           // the slot is visible before the ticket is drawn
    is_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  double s = 0.0;
  for (int b = threadIdx.x; b < (int)gridDim.x; b += kThreads) s += __ldcg(partial + b);   // L2 reads: other blocks wrote these
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double v = 0.0;
#pragma unroll
    for (int w = 0; w < kThreads / 32; ++w) v += red[w];
    *mean_sq = (float)(v / (double)total);
  }
}

// Device address of the scratch array on the CURRENT device, looked up once per device (with that device current) and kept.
std::mutex g_mu;
double* g_scratch_addr[kMaxDevices] = {};

pigan_status scratch_of_current_device(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail_cuda("cudaGetDevice", e);
  if (dev < 0 || dev >= kMaxDevices) return fail(PIGAN_ERR_UNSUPPORTED, "device ordinal beyond the 64 devices this entry point keeps an address for");
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_residual_scratch);
    if (e != cudaSuccess || !p) return fail_cuda("cudaGetSymbolAddress(static scratch)", e != cudaSuccess ? e : cudaErrorInvalidSymbol);
    g_scratch_addr[dev] = static_cast<double*>(p);
  }
  *out = g_scratch_addr[dev];
  return PIGAN_OK;
}

}  // namespace

extern "C" {

const char* pigan_static_last_error(void) { return t_err; }

pigan_status pigan_darcy_residual_static(const float* logk_jet, const float* u_jet, const float* f, int n_samples, int n_pts, float* r,
                                         float* mean_sq, void* cuda_stream) {
  if (n_samples < 0 || n_pts < 0) return fail(PIGAN_ERR_INVALID_ARG, "negative size");
  const long long total = (long long)n_samples * n_pts;
  if (total > kMaxRows) {
    snprintf(t_err, sizeof t_err,
             "n_samples * n_pts = %lld rows exceeds PIGAN_STATIC_MAX_ROWS = %lld, the size the built-in scratch array is made for; "
             "split the rows over several calls or use pigan_darcy_residual on a context",
             total, kMaxRows);
    return PIGAN_ERR_UNSUPPORTED;
  }
  if (total > 0 && (!logk_jet || !u_jet || !f)) return fail(PIGAN_ERR_INVALID_ARG, "null pointer");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (total == 0) {                                                            // as pigan_darcy_residual: the mean over no rows is 0
    if (mean_sq) {
      const cudaError_t e = cudaMemsetAsync(mean_sq, 0, sizeof(float), st);
      if (e != cudaSuccess) return fail_cuda("cudaMemsetAsync(mean_sq)", e);
    }
    t_err[0] = 0;
    return PIGAN_OK;
  }
  if (!r && !mean_sq) { t_err[0] = 0; return PIGAN_OK; }
  double* scratch = nullptr;
  const pigan_status s = scratch_of_current_device(&scratch);
  if (s != PIGAN_OK) return s;
  if (mean_sq) {                                                               // the ticket counter must start at zero; the partial sums need not
    const cudaError_t e = cudaMemsetAsync(scratch, 0, sizeof(unsigned int), st);
    if (e != cudaSuccess) return fail_cuda("cudaMemsetAsync(ticket)", e);
  }
  const int blocks = (int)((total + kRowsPerBlock - 1) / kRowsPerBlock);
  residual_static_kernel<<<blocks, kThreads, 0, st>>>(logk_jet, u_jet, f, (int)total, total, n_pts, r, mean_sq, scratch);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail_cuda("residual_static_kernel launch", e);
  t_err[0] = 0;
  return PIGAN_OK;
}

}  // extern "C"
