/* pigan.h -- C-ABI boundary of the B200-native PI-GAN hot path (arXiv 1910.13444, Yang et al. 2019).
 *
 * One WGAN-GP training step's dense compute, single GPU, hand-written sm_100a CUDA underneath.
 * Citations: P:<n> = PAPER.md line n; S8x = SURVEY.md section 8(x); DESIGN.md section 3 lists the readings (G1..G21)
 * taken where the paper is silent.
 *
 *   generator  (x, y, z) -> log k, u : tanh fully-connected layers, narrow per-point input ........ P:139
 *   induced network f = div(k grad u) obtained by differentiating the generator in (x, y) ........... P:93 Eq. 1
 *   snapshot   [log k(s_1..s_S), u(s_1..s_S)] per latent sample, scored by the discriminator ........ P:139
 *   WGAN-GP    critic loss with the two-sided gradient penalty of ref. [24] ......................... P:83
 *   precision  16-bit activations and gradients, FP32 accumulation / master weights, loss scaling ... P:155
 *
 * CONVENTIONS
 *   - Every call returns a pigan_status and never throws; pigan_last_error(ctx) gives a message.
 *   - ALL array arguments are DEVICE pointers owned by the caller, fp32 (int for flags), contiguous, 16-byte
 *     aligned.  The library never frees or retains them past the call.  The context owns only its workspaces
 *     and its 16-bit weight copies.
 *   - Calls are asynchronous on the CUDA stream given at creation (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream).  One context per stream; a context is not thread-safe.
 *   - Scalars that the host passes by value are marked so; scalars the device produces (losses, found_inf, gp,
 *     mean_sq) are device pointers and are valid once the stream has reached the end of the call.
 *   - fp16 overflow is not an error: it is reported through *found_inf.
 *   - Randomness (z, eps, sensor locations, weights) is input data; nothing is drawn inside the library.
 *   - There is no CPU fallback: without a CUDA device pigan_create fails with PIGAN_ERR_CUDA.
 *
 * FLAT PARAMETER PACKING (fp32), per network: for l = 1..n_hidden+1: W_l row-major [out][in], then b_l [out];
 *   the last layer has out = 1.  Generator W_1 columns are ordered [x, y, z_1..z_m].  Gradients use the same packing.
 *
 * JET CHANNEL ORDER: 0 value, 1 d/dx, 2 d/dy, 3 d2/dx2, 4 d2/dy2 (no mixed derivative: k is isotropic, Eq. 1).
 */
#ifndef PIGAN_H_
#define PIGAN_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pigan_ctx pigan_ctx;

typedef enum {
  PIGAN_OK = 0,
  PIGAN_ERR_INVALID_ARG = 1,   /* NULL pointer, non-positive size, unknown enum value */
  PIGAN_ERR_SHAPE = 2,         /* a size disagrees with the pigan_config the context was created with */
  PIGAN_ERR_ALLOC = 3,         /* workspace allocation failed */
  PIGAN_ERR_CUDA = 4,          /* a CUDA runtime / driver call failed (no device, launch error, ...) */
  PIGAN_ERR_UNSUPPORTED = 5    /* e.g. 16-bit precision with a width that is not a multiple of 128; PIGAN_BF16 */
} pigan_status;

/* Arithmetic of the hidden jet layers (S8a a3, a10).  FP32: plain FP32 FMA.  FP16: tcgen05 tensor cores, fp16
 * operands (the paper's arithmetic), fp32 accumulation in TMEM, fp32 epilogue; first layer, output dot, residual,
 * critic, norms, reductions and weight-gradient accumulation stay fp32 (reading G18).
 * PIGAN_BF16 is NOT IMPLEMENTED: pigan_create returns PIGAN_ERR_UNSUPPORTED for it (reading R1: bf16 activation
 * planes measure 1-2e-2 against the 2e-2 tolerance, so the library's one 16-bit arithmetic is the paper's FP16; the
 * enum value is kept so that the numbering of pigan_precision is stable).  Consequence of FP16: activation and jet planes
 * have fp16 RANGE (65504); the derivative channels grow with products of layer gains, and a forward overflow surfaces
 * as inf/nan gradients with *found_inf = 1 (never as silently wrong finite values). */
typedef enum { PIGAN_FP32 = 0, PIGAN_BF16 = 1, PIGAN_FP16 = 2 } pigan_precision;

/* pigan_config.flags (debug / measurement switches; 0 is the product path) */
#define PIGAN_FLAG_NO_GRAPH   1u   /* never capture / replay pigan_train_step_grads as a CUDA graph: every call runs eagerly */
#define PIGAN_FLAG_ONE_CTA    2u   /* use the one-CTA tcgen05 kernels even where the CTA-pair (cta_group::2) kernels apply */

typedef struct { int in_dim, n_hidden, width; } pigan_mlp_shape;   /* scalar linear output implied (G10) */

/* Which generator the context trains.
 *   TWO_MLPS    BASELINE.json's variant: two separate plain MLPs G_logk (3 jet channels) and G_u (5)  (reading G4).
 *   TRUNK       the paper's: ONE set of weights, separate log k and u outputs in the final layer.  The last
 *               layer is W [2][H] (row 0: log k, row 1: u) then b [2]; the 5-channel jet of the last hidden layer serves
 *               both heads, so a step costs 5 channel passes instead of 8 (R7).
 *   TRUNK_SKIP  TRUNK with residual connections that skip intermediate layers: h^l = tanh(a^l) + h^{l-2} for odd
 *               l >= 3 (two-layer residual blocks of ref. [30]; R8). */
typedef enum { PIGAN_GEN_TWO_MLPS = 0, PIGAN_GEN_TRUNK = 1, PIGAN_GEN_TRUNK_SKIP = 2 } pigan_gen_variant;

typedef struct {
  pigan_mlp_shape gen;       /* in_dim = 2 + latent_dim; the same shape is used for G_logk and G_u (G4) */
  pigan_mlp_shape disc;      /* in_dim = 2 * n_sensors (G6) */
  int latent_dim;            /* m */
  int n_samples;             /* N, latent samples per step (= real batch size, G11) */
  int n_colloc;              /* P, collocation points shared by all samples (G13) */
  int n_sensors;             /* S */
  pigan_precision precision;
  float gp_lambda;           /* WGAN-GP weight, 10 (G2) */
  float pde_weight;          /* w_pde in L_G = -mean D(fake) + w_pde mean r^2 (G8), default 1 */
  size_t workspace_bytes;    /* 0 = library default; bounds the row-chunk size of the step (S7 H1) */
  int chunk_rows;            /* 0 = library default (131072); rows per chunk of the generator passes, rounded to 256 */
  unsigned flags;            /* PIGAN_FLAG_* */
  int gen_variant;           /* pigan_gen_variant; 0 = BASELINE.json's two MLPs */
  int n_free;                /* NEXT-2: 0 = BASELINE.json's step.  F > 0: every latent sample has its own F free-sensor
                                points (n_colloc must equal F, xy_colloc is [N][F][2], f is ignored and may be NULL); the critic's
                                snapshot is [log k(S), u(S), f(F), x(F), y(F)], so disc.in_dim = 2 S + 3 F; L_G = -mean D(fake) +
                                pde_weight * mean f^2 (the paper's choice is pde_weight = 0); losses[5] = mean f^2.  Two-MLP generator only. */
  int n_critics;             /* NEXT-3: 0 = one critic on the whole snapshot.  K > 0: K critics of shape `disc`, each on
                                disc.in_dim columns of the 2S-entry snapshot; such a context steps through
                                pigan_train_step_grads_hier.  Two-MLP generator, n_free = 0 only. */
} pigan_config;

/* Creates a context: validates cfg, allocates the workspace on the CURRENT CUDA device and binds the context to it
 * (every later call on the context switches to that device for its duration and restores the caller's).  *out is NULL
 * on failure (the status says why).  cuda_stream is a cudaStream_t of that device. */
pigan_status pigan_create(const pigan_config* cfg, void* cuda_stream, pigan_ctx** out);
void         pigan_destroy(pigan_ctx* ctx);                       /* NULL is allowed */
size_t       pigan_param_count(const pigan_mlp_shape* shape);     /* H*in + H + (L-1)(H*H + H) + H + 1; 0 if shape is NULL/invalid */
size_t       pigan_trunk_param_count(const pigan_mlp_shape* shape); /* shared trunk: the plain count + H + 1 (second head) */
const char*  pigan_last_error(const pigan_ctx* ctx);              /* never NULL; "" when no error */
/* Number of kernels this context has launched since creation (bench.py reports it as gpu_launches). */
unsigned long long pigan_launch_count(const pigan_ctx* ctx);

/* Measurement helpers (bench.py's roofline): while enabled, one CUDA event is recorded on the context's stream after
 * every kernel launch.  pigan_profile_report synchronises the stream and writes a JSON object
 * {"<kernel class>": [launches, total_ms], ...} (durations = differences of consecutive events) into buf (NUL-terminated,
 * truncated to cap), then clears the trace.  Returns PIGAN_ERR_INVALID_ARG if profiling was never enabled. */
pigan_status pigan_profile_enable(pigan_ctx* ctx, int enable);
pigan_status pigan_profile_report(pigan_ctx* ctx, char* buf, size_t cap);

/* a1-a4 (S8a): generator value and spatial jet at n_pts points for n_samples latent vectors.
 *   gen_params [param_count(cfg.gen)]; xy [n_pts][2]; z [n_samples][m]; n_samples, n_pts >= 0 (0 = no-op).
 *   jet_order 0: C=1 (value); 1: C=3 (value, d/dx, d/dy); 2: C=5 (+ d2/dx2, d2/dy2).
 *   out [C][n_samples][n_pts] fp32, overwritten.   Defines: S8c O1, O2. */
pigan_status pigan_gen_jet_forward(pigan_ctx* ctx, const float* gen_params, const float* xy, int n_pts,
                                   const float* z, int n_samples, int jet_order, float* out);

/* NEXT-1: the shared-trunk generator (context created with gen_variant TRUNK or TRUNK_SKIP).  Same arguments as
 *   pigan_gen_jet_forward; trunk_params [pigan_trunk_param_count(cfg.gen)]; out [2][C][n_samples][n_pts]: head 0 = log k,
 *   head 1 = u, each with its C jet channels.   Defines: P:139; R7, R8. */
pigan_status pigan_trunk_jet_forward(pigan_ctx* ctx, const float* trunk_params, const float* xy, int n_pts,
                                     const float* z, int n_samples, int jet_order, float* out);

/* a5: Darcy residual r[n][p] = exp(Y)(Y_x u_x + Y_y u_y + u_xx + u_yy) - f[p]  (Eq. 1, with k = exp Y).
 *   logk_jet [>=3][N][P] (only channels 0..2 are read; plane stride N*P), u_jet [5][N][P], f [P].
 *   r [N][P] overwritten (may be NULL); mean_sq device scalar = mean r^2, overwritten (may be NULL). */
pigan_status pigan_darcy_residual(pigan_ctx* ctx, const float* logk_jet, const float* u_jet, const float* f,
                                  int n_samples, int n_pts, float* r, float* mean_sq);

/* a7: critic score D(X) = v_out . g^{L_D} + c_out, g^l = tanh(V_l g^{l-1} + c_l)  (S8c O1).
 *   snap [B][2S]; score [B] overwritten; 0 <= B. */
pigan_status pigan_disc_forward(pigan_ctx* ctx, const float* disc_params, const float* snap, int B, float* score);

/* a8 (+ the GP part of a9): gp = lambda * mean_n (||grad_X D(xhat_n)||_2 - 1)^2, xhat_n = eps_n real_n + (1-eps_n) fake_n
 *   (ref. [24] via P:83; S8c O5, O6; ||G|| = 0 gives a zero gradient seed, G12).
 *   real, fake [B][2S]; eps [B]; gp device scalar; grad_norm [B]; d_disc_params [param_count(cfg.disc)] = d gp/d theta_D,
 *   overwritten.  gp, grad_norm, d_disc_params may each be NULL.  1 <= B. */
pigan_status pigan_gradient_penalty(pigan_ctx* ctx, const float* disc_params, const float* real, const float* fake,
                                    const float* eps, int B, float* gp, float* grad_norm, float* d_disc_params);

/* a1-a10: both gradient sets of one step at the SAME current weights (G16):
 *   L_D = mean D(fake) - mean D(real) + GP            -> g_disc  (X_fake held constant)
 *   L_G = -mean D(fake) + w_pde * mean_{n,p} r^2      -> g_logk, g_u  (theta_D held constant)
 *   xy_colloc [P][2], f [P], xy_sensors [S][2], z [N][m], real_snap [N][2S], eps [N]; sizes from the config.
 *   loss_scale (host value, > 0) multiplies the adjoints of the 16-bit backward pass; gradients are returned
 *   UNSCALED in fp32 (overwritten).  losses[6] = {L_D, mean D(fake), mean D(real), GP, L_G, L_pde}.
 *   *found_inf (device int, overwritten) = 1 if any gradient is inf/nan, else 0.  losses, found_inf may be NULL.
 *   Execution: asynchronous on the context's stream.  The first call with a given argument set (all pointers and loss_scale)
 *   runs eagerly, the second call with that set is captured into a CUDA graph and later ones replay it; the four most recently
 *   used argument sets are remembered, so alternating between a few sets of buffers replays as well.  The arrays are read when the
 *   step RUNS, so updating them in place between calls (an optimiser step, new z / eps copied into the same buffers)
 *   behaves exactly as an eager call.  cfg.flags & PIGAN_FLAG_NO_GRAPH disables the replay; cfg.chunk_rows sets the
 *   row-chunk size (default 131072 rows; workspace_bytes of the config bounds it as well).  No environment variable
 *   changes the behaviour of the library. */
/*   Shared-trunk contexts (gen_variant != 0): logk_params = the trunk's parameters, g_logk = their gradient
 *   [pigan_trunk_param_count]; u_params and g_u are ignored and may be NULL. */
pigan_status pigan_train_step_grads(pigan_ctx* ctx, const float* logk_params, const float* u_params,
                                    const float* disc_params, const float* xy_colloc, const float* f,
                                    const float* xy_sensors, const float* z, const float* real_snap,
                                    const float* eps, float loss_scale, float* g_logk, float* g_u, float* g_disc,
                                    float* losses, int* found_inf);

/* NEXT-3: the step with the hierarchical multi-discriminator loss (R10), for contexts created with
 *   n_critics = K > 0.  As pigan_train_step_grads, except:
 *   disc_params, g_disc  [K][param_count(cfg.disc)]: critic k's parameters / the gradient of ITS loss
 *                        L_Dk = mean D_k(fake_k) - mean D_k(real_k) + GP_k (shared eps);
 *   subsets  DEVICE int [K][cfg.disc.in_dim]: the snapshot columns (0 .. 2S-1, distinct within a critic) that critic k sees; they are
 *            not checked here (a device array): a column out of range or repeated within a critic is undefined behaviour;
 *   weights  HOST float [K], read during the call only (it may be freed or changed as soon as the call returns): w_k = 1 / (levels * subdomains in k's level); L_G = sum_k w_k (-mean D_k(fake_k)) + w_pde mean r^2;
 *   real_snap [N][2S];  losses[6] = {sum_k L_Dk, sum_k w_k mean D_k(fake), sum_k w_k mean D_k(real), sum_k GP_k, L_G, L_pde}.
 *   Runs eagerly (no CUDA-graph replay). */
pigan_status pigan_train_step_grads_hier(pigan_ctx* ctx, const float* logk_params, const float* u_params, const float* disc_params,
                                         const int* subsets, const float* weights, const float* xy_colloc, const float* f,
                                         const float* xy_sensors, const float* z, const float* real_snap, const float* eps,
                                         float loss_scale, float* g_logk, float* g_u, float* g_disc, float* losses, int* found_inf);

/* a11: Adam with bias correction on fp32 master weights (S8c O8, G3: eps outside the square root).
 *   params, m, v [n] updated in place; grads [n]; step is 1-based; if skip_flag != NULL and *skip_flag != 0
 *   (device int, e.g. found_inf) the update is a no-op and params, m, v stay bit-identical. */
pigan_status pigan_adam_update(pigan_ctx* ctx, float* params, const float* grads, float* m, float* v, size_t n,
                               int step, float lr, float beta1, float beta2, float adam_eps, const int* skip_flag);

/* a5 WITHOUT A CONTEXT AND WITHOUT ANY ALLOCATION: the Darcy residual of pigan_darcy_residual (Eq. 1) for callers that
 * cannot allocate device memory.  Who they are: code hosted inside another program (a solver, a simulator, a serving process)
 * that took nearly all GPU memory for its own pool when it started, so that cudaMalloc fails or is forbidden by the host's
 * rules; and control / time-stepping loops that must not call cudaMalloc or cudaFree in steady state because those calls can
 * stall the whole device for an unpredictable time.  pigan_create allocates workspaces, so such callers cannot have a context.
 * This call makes no cudaMalloc, cudaFree or allocating library call, on its first use or later.  The scratch its reduction needs
 * (one partial sum of r^2 per 1024 rows, plus a ticket counter) is a fixed array built into the library image.
 *   logk_jet [>=3][N][P] (channels 0..2 read; plane stride N*P), u_jet [5][N][P], f [P]: DEVICE pointers, fp32, owned by the caller.
 *   r [N][P] overwritten (may be NULL); mean_sq device scalar = mean r^2, overwritten (may be NULL); N*P = 0 writes mean_sq = 0.
 *   cuda_stream: a cudaStream_t (NULL = legacy default stream) of the CURRENT device; the call is asynchronous on it.
 * Limits and sharing:
 *   - N*P <= PIGAN_STATIC_MAX_ROWS (2^24 rows); more is refused with PIGAN_ERR_UNSUPPORTED and a message naming the limit
 *     (split the rows over several calls, or use a context).
 *   - The array (about 128 KiB) sits on every GPU that loads the library's device code, until the process exits.
 *   - All calls on one GPU share the array and it keeps the previous call's contents; each call zeroes the counter it depends on.
 *     Calls that can overlap on the same GPU (two streams, two threads) race on it: the caller must order them (one stream does).
 *   - The first call on each device looks up the array's device address (cudaGetSymbolAddress, with that device current) and
 *     keeps it; make that first call before starting any stream capture.
 * Returns a pigan_status; pigan_static_last_error() gives the message of the calling thread's last failed call ("" after success). */
#define PIGAN_STATIC_MAX_ROWS (1LL << 24)
pigan_status pigan_darcy_residual_static(const float* logk_jet, const float* u_jet, const float* f, int n_samples, int n_pts,
                                         float* r, float* mean_sq, void* cuda_stream);
const char*  pigan_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PIGAN_H_ */
