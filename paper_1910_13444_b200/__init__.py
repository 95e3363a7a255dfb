"""B200-native PI-GAN hot path (arXiv 1910.13444): thin Python binding over the C-ABI library libpigan.so.

The binding only marshals arguments: every step of the path runs in the library's CUDA kernels (include/pigan.h).
PyTorch is used for device memory and streams.  There is no CPU fallback: importing works anywhere (so that the
exported symbols can be checked), but creating a context without a CUDA device raises.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, Structure, c_char_p, c_float, c_int, c_size_t, c_ulonglong, c_void_p

from .build import LIB, build, is_stale

__all__ = ["PiGan", "PiganError", "load_library", "param_count", "EXPORTED_SYMBOLS", "PRECISIONS", "FLAG_NO_GRAPH", "FLAG_ONE_CTA",
           "darcy_residual_static", "STATIC_MAX_ROWS"]

FLAG_NO_GRAPH, FLAG_ONE_CTA = 1, 2                     # pigan_config.flags (include/pigan.h)

PRECISIONS = {"fp32": 0, "bf16": 1, "fp16": 2}
STATUS = {0: "PIGAN_OK", 1: "PIGAN_ERR_INVALID_ARG", 2: "PIGAN_ERR_SHAPE", 3: "PIGAN_ERR_ALLOC", 4: "PIGAN_ERR_CUDA",
          5: "PIGAN_ERR_UNSUPPORTED"}
EXPORTED_SYMBOLS = ["pigan_create", "pigan_destroy", "pigan_param_count", "pigan_trunk_param_count", "pigan_last_error", "pigan_launch_count",
                    "pigan_profile_enable", "pigan_profile_report", "pigan_trunk_jet_forward",
                    "pigan_gen_jet_forward", "pigan_darcy_residual", "pigan_disc_forward", "pigan_gradient_penalty",
                    "pigan_train_step_grads", "pigan_train_step_grads_hier", "pigan_adam_update",
                    "pigan_darcy_residual_static", "pigan_static_last_error"]
STATIC_MAX_ROWS = 1 << 24                              # PIGAN_STATIC_MAX_ROWS (include/pigan.h)


class PiganError(RuntimeError):
    def __init__(self, status: int, message: str = ""):
        super().__init__(f"{STATUS.get(status, status)}: {message}")
        self.status = status


class _MlpShape(Structure):
    _fields_ = [("in_dim", c_int), ("n_hidden", c_int), ("width", c_int)]


class _Config(Structure):
    _fields_ = [("gen", _MlpShape), ("disc", _MlpShape), ("latent_dim", c_int), ("n_samples", c_int), ("n_colloc", c_int),
                ("n_sensors", c_int), ("precision", c_int), ("gp_lambda", c_float), ("pde_weight", c_float),
                ("workspace_bytes", c_size_t), ("chunk_rows", c_int), ("flags", ctypes.c_uint), ("gen_variant", c_int), ("n_free", c_int), ("n_critics", c_int)]


_lib = None


def load_library():
    """Loads libpigan.so, building it first if it is missing or older than any source under csrc/ or include/pigan.h
    (nvcc is needed for that; a GPU box receives the built library with the snapshot).  Raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    path = LIB
    if not os.path.exists(path) or is_stale():
        path = build()
    lib = ctypes.CDLL(path)
    fp, ip = POINTER(c_float), POINTER(c_int)
    lib.pigan_create.argtypes = [POINTER(_Config), c_void_p, POINTER(c_void_p)]
    lib.pigan_create.restype = c_int
    lib.pigan_destroy.argtypes = [c_void_p]
    lib.pigan_destroy.restype = None
    lib.pigan_param_count.argtypes = [POINTER(_MlpShape)]
    lib.pigan_param_count.restype = c_size_t
    lib.pigan_trunk_param_count.argtypes = [POINTER(_MlpShape)]
    lib.pigan_trunk_param_count.restype = c_size_t
    lib.pigan_trunk_jet_forward.argtypes = [c_void_p, c_void_p, c_void_p, c_int, c_void_p, c_int, c_int, c_void_p]
    lib.pigan_trunk_jet_forward.restype = c_int
    lib.pigan_last_error.argtypes = [c_void_p]
    lib.pigan_last_error.restype = c_char_p
    lib.pigan_launch_count.argtypes = [c_void_p]
    lib.pigan_launch_count.restype = c_ulonglong
    lib.pigan_gen_jet_forward.argtypes = [c_void_p, c_void_p, c_void_p, c_int, c_void_p, c_int, c_int, c_void_p]
    lib.pigan_darcy_residual.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_int, c_int, c_void_p, c_void_p]
    lib.pigan_disc_forward.argtypes = [c_void_p, c_void_p, c_void_p, c_int, c_void_p]
    lib.pigan_gradient_penalty.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int, c_void_p, c_void_p, c_void_p]
    lib.pigan_train_step_grads.argtypes = [c_void_p] + [c_void_p] * 9 + [c_float] + [c_void_p] * 5
    lib.pigan_train_step_grads_hier.argtypes = [c_void_p] * 4 + [c_void_p, POINTER(c_float)] + [c_void_p] * 6 + [c_float] + [c_void_p] * 5
    lib.pigan_adam_update.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_size_t, c_int, c_float, c_float, c_float,
                                      c_float, c_void_p]
    lib.pigan_profile_enable.argtypes = [c_void_p, c_int]
    lib.pigan_profile_report.argtypes = [c_void_p, c_char_p, c_size_t]
    lib.pigan_darcy_residual_static.argtypes = [c_void_p, c_void_p, c_void_p, c_int, c_int, c_void_p, c_void_p, c_void_p]
    lib.pigan_static_last_error.argtypes = []
    lib.pigan_static_last_error.restype = c_char_p
    for name in EXPORTED_SYMBOLS:
        if name not in ("pigan_create", "pigan_destroy", "pigan_param_count", "pigan_trunk_param_count", "pigan_last_error", "pigan_launch_count",
                        "pigan_static_last_error"):
            getattr(lib, name).restype = c_int
    del fp, ip
    _lib = lib
    return lib


def param_count(in_dim: int, n_hidden: int, width: int) -> int:
    return int(load_library().pigan_param_count(ctypes.byref(_MlpShape(in_dim, n_hidden, width))))


def trunk_param_count(in_dim: int, n_hidden: int, width: int) -> int:
    return int(load_library().pigan_trunk_param_count(ctypes.byref(_MlpShape(in_dim, n_hidden, width))))


GEN_VARIANTS = {"two_mlps": 0, "trunk": 1, "trunk_skip": 2}     # pigan_gen_variant (include/pigan.h)


def _ptr(t, name, dtype=None):
    """Device pointer of a contiguous CUDA tensor (None -> NULL)."""
    import torch
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda or not t.is_contiguous():
        raise TypeError(f"{name} must be a contiguous CUDA tensor")
    if t.dtype != (dtype or torch.float32):
        raise TypeError(f"{name} must have dtype {dtype or torch.float32}, got {t.dtype}")
    return c_void_p(t.data_ptr())


def darcy_residual_static(logk_jet, u_jet, f, r=None, mean_sq=None, stream=None):
    """The Darcy residual through pigan_darcy_residual_static: no context, and no device allocation inside the library.

    For programs that cannot allocate GPU memory when they call us -- code embedded in a host application that gave all device
    memory to its own pool at start-up (cudaMalloc fails or is off limits there), or a latency-bound loop that keeps
    cudaMalloc / cudaFree out of its steady state because they can stall the device.  A PiGan context allocates workspaces when
    it is created, so it is not an option for them.  Such a caller passes its OWN output tensors: `r` [N][P] and / or `mean_sq` [1]
    (fp32, CUDA, contiguous) are written in place and returned; at least one must be given, and nothing is allocated here or
    in the library.  logk_jet [>=3][N][P], u_jet [5][N][P], f [P].
    Limits: N*P <= STATIC_MAX_ROWS (2^24), else PiganError(PIGAN_ERR_UNSUPPORTED).  The library's built-in scratch array is shared by
    every call on a GPU: calls that may overlap (different streams / threads) must be ordered by the caller.  The first call on
    a device also looks up the array's address; make it before any stream capture starts.  Runs on `stream` (default: the
    current stream) of the tensors' device."""
    import torch
    if logk_jet.shape[1:] != u_jet.shape[1:] or logk_jet.shape[0] < 3 or u_jet.shape[0] != 5:
        raise ValueError("logk_jet must be [>=3][N][P] and u_jet [5][N][P]")
    if r is None and mean_sq is None:
        raise ValueError("pass r and / or mean_sq: the caller owns the outputs, nothing is allocated here")
    lib = load_library()
    N, P = u_jet.shape[1], u_jet.shape[2]
    if r is not None and r.numel() != N * P or mean_sq is not None and mean_sq.numel() < 1:
        raise ValueError("r must hold N*P values and mean_sq one")
    with torch.cuda.device(u_jet.device):
        st = stream if stream is not None else torch.cuda.current_stream(u_jet.device)
        rc = lib.pigan_darcy_residual_static(_ptr(logk_jet, "logk_jet"), _ptr(u_jet, "u_jet"), _ptr(f, "f"), N, P, _ptr(r, "r"),
                                             _ptr(mean_sq, "mean_sq"), c_void_p(st.cuda_stream))
    if rc != 0:
        raise PiganError(rc, lib.pigan_static_last_error().decode())
    return r, mean_sq


class PiGan:
    """One context = one CUDA stream + the workspaces of one PI-GAN configuration (mirrors pigan_ctx)."""

    def __init__(self, *, latent_dim, gen_hidden, gen_width, disc_hidden, disc_width, n_samples, n_colloc, n_sensors,
                 precision="fp32", gp_lambda=10.0, pde_weight=1.0, workspace_bytes=0, chunk_rows=0, flags=0, gen_variant="two_mlps", n_free=0, n_critics=0, critic_inputs=None, stream=None, device=None):
        import torch
        self._lib = load_library()
        self._ctx = c_void_p()
        if not torch.cuda.is_available():
            raise PiganError(4, "no CUDA device: the PI-GAN hot path has no CPU fallback")
        self.device = torch.device(device if device is not None else f"cuda:{torch.cuda.current_device()}")
        self.m, self.N, self.P, self.S = latent_dim, n_samples, n_colloc, n_sensors
        self.gen_shape = (2 + latent_dim, gen_hidden, gen_width)
        self.disc_shape = ((critic_inputs if n_critics else 2 * n_sensors + 3 * n_free), disc_hidden, disc_width)
        self.n_free, self.n_critics = n_free, n_critics
        self.precision = precision
        cfg = _Config(_MlpShape(*self.gen_shape), _MlpShape(*self.disc_shape), latent_dim, n_samples, n_colloc, n_sensors,
                      PRECISIONS[precision], gp_lambda, pde_weight, workspace_bytes, chunk_rows, flags, GEN_VARIANTS[gen_variant], n_free, n_critics)
        self.gen_variant = gen_variant
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        with torch.cuda.device(self.device):
            st = self._lib.pigan_create(ctypes.byref(cfg), c_void_p(self._stream.cuda_stream), ctypes.byref(self._ctx))
        if st != 0:
            self._ctx = c_void_p()
            raise PiganError(st, "pigan_create failed")
        self.n_gen = param_count(*self.gen_shape) if gen_variant == "two_mlps" else trunk_param_count(*self.gen_shape)
        self.n_disc = param_count(*self.disc_shape)

    @classmethod
    def from_config(cls, cfg, **kw):
        """cfg: a workloads.Config."""
        return cls(latent_dim=cfg.m, gen_hidden=cfg.L, gen_width=cfg.H, disc_hidden=cfg.LD, disc_width=cfg.HD, n_samples=cfg.N,
                   n_colloc=cfg.P, n_sensors=cfg.S, precision=cfg.precision, **kw)

    def close(self):
        if getattr(self, "_ctx", None) and self._ctx.value:
            self._lib.pigan_destroy(self._ctx)
            self._ctx = c_void_p()

    __del__ = close

    def _check(self, st):
        if st != 0:
            raise PiganError(st, self._lib.pigan_last_error(self._ctx).decode())

    def _new(self, *shape, dtype=None):
        import torch
        return torch.empty(*shape, dtype=dtype or torch.float32, device=self.device)

    @property
    def launch_count(self) -> int:
        return int(self._lib.pigan_launch_count(self._ctx))

    def profile_enable(self, enable=True):
        self._check(self._lib.pigan_profile_enable(self._ctx, 1 if enable else 0))

    def profile_report(self) -> dict:
        """{kernel class: [launches, total_ms]} since profiling was enabled (synchronises the stream)."""
        import json
        buf = ctypes.create_string_buffer(1 << 16)
        self._check(self._lib.pigan_profile_report(self._ctx, buf, len(buf)))
        return json.loads(buf.value.decode())

    # ---- the six calls of include/pigan.h ---------------------------------------------------------------------
    def gen_jet_forward(self, gen_params, xy, z, jet_order, out=None):
        n_pts, n_samples = xy.shape[0], z.shape[0]
        C = (1, 3, 5)[jet_order]
        if out is None:
            out = self._new(C, n_samples, n_pts)
        self._check(self._lib.pigan_gen_jet_forward(self._ctx, _ptr(gen_params, "gen_params"), _ptr(xy, "xy"), n_pts, _ptr(z, "z"),
                                                    n_samples, jet_order, _ptr(out, "out")))
        return out

    def trunk_jet_forward(self, trunk_params, xy, z, jet_order, out=None):
        """NEXT-1: out [2][C][N][P], head 0 = log k, head 1 = u (contexts created with gen_variant 'trunk' / 'trunk_skip')."""
        n_pts, n_samples = xy.shape[0], z.shape[0]
        C = (1, 3, 5)[jet_order]
        if out is None:
            out = self._new(2, C, n_samples, n_pts)
        self._check(self._lib.pigan_trunk_jet_forward(self._ctx, _ptr(trunk_params, "trunk_params"), _ptr(xy, "xy"), n_pts, _ptr(z, "z"),
                                                      n_samples, jet_order, _ptr(out, "out")))
        return out

    def darcy_residual(self, logk_jet, u_jet, f, want_r=True, want_mean=True):
        if logk_jet.shape[1:] != u_jet.shape[1:] or logk_jet.shape[0] < 3 or u_jet.shape[0] != 5:
            raise ValueError("logk_jet must be [>=3][N][P] and u_jet [5][N][P]")
        N, P = u_jet.shape[1], u_jet.shape[2]
        r = self._new(N, P) if want_r else None
        msq = self._new(1) if want_mean else None
        self._check(self._lib.pigan_darcy_residual(self._ctx, _ptr(logk_jet, "logk_jet"), _ptr(u_jet, "u_jet"), _ptr(f, "f"), N, P,
                                                   _ptr(r, "r"), _ptr(msq, "mean_sq")))
        return r, msq

    def disc_forward(self, disc_params, snap):
        B = snap.shape[0]
        score = self._new(B)
        self._check(self._lib.pigan_disc_forward(self._ctx, _ptr(disc_params, "disc_params"), _ptr(snap, "snap"), B, _ptr(score, "score")))
        return score

    def gradient_penalty(self, disc_params, real, fake, eps, want_grad=True):
        B = real.shape[0]
        gp, nu = self._new(1), self._new(B)
        d = self._new(self.n_disc) if want_grad else None
        self._check(self._lib.pigan_gradient_penalty(self._ctx, _ptr(disc_params, "disc_params"), _ptr(real, "real"), _ptr(fake, "fake"),
                                                     _ptr(eps, "eps"), B, _ptr(gp, "gp"), _ptr(nu, "grad_norm"), _ptr(d, "d_disc_params")))
        return gp, nu, d

    def train_step_grads(self, logk_params, u_params, disc_params, xy_colloc, f, xy_sensors, z, real_snap, eps, loss_scale=1.0,
                         out=None):
        import torch
        if out is None:
            out = (self._new(self.n_gen), self._new(self.n_gen) if self.gen_variant == "two_mlps" else None, self._new(self.n_disc), self._new(6),
                   self._new(1, dtype=torch.int32))
        g_logk, g_u, g_disc, losses, found_inf = out
        n_xy = self.N * self.P if self.n_free else self.P                    # free-sensor mode: xy_colloc is [N][F][2]
        if (xy_colloc.numel() // 2, xy_sensors.shape[0], tuple(z.shape), tuple(real_snap.shape)) != (n_xy, self.S, (self.N, self.m), (self.N, self.disc_shape[0])):
            raise ValueError("input sizes disagree with the configuration of this context")
        self._check(self._lib.pigan_train_step_grads(
            self._ctx, _ptr(logk_params, "logk_params"), _ptr(u_params, "u_params"), _ptr(disc_params, "disc_params"),
            _ptr(xy_colloc, "xy_colloc"), _ptr(f, "f"), _ptr(xy_sensors, "xy_sensors"), _ptr(z, "z"), _ptr(real_snap, "real_snap"),
            _ptr(eps, "eps"), float(loss_scale), _ptr(g_logk, "g_logk"), _ptr(g_u, "g_u"), _ptr(g_disc, "g_disc"), _ptr(losses, "losses"),
            _ptr(found_inf, "found_inf", torch.int32)))
        return out

    def train_step_grads_hier(self, logk_params, u_params, disc_params, subsets, weights, xy_colloc, f, xy_sensors, z, real_snap, eps, loss_scale=1.0):
        """NEXT-3: K critics (context created with n_critics = K, critic_inputs = columns per critic).  disc_params [K][n_disc];
        subsets: int32 CUDA tensor [K][critic_inputs]; weights: K host floats.  Returns (g_logk, g_u, g_disc [K][n_disc], losses, found_inf)."""
        import torch
        K = self.n_critics
        # the kernels index the snapshot with `subsets` and add into it without atomics: columns out of range or repeated within a
        # critic are undefined behaviour in the C call.  Checked here once per tensor (and again if it is modified in place).
        key = (subsets.data_ptr(), subsets._version, tuple(subsets.shape))
        if getattr(self, "_subsets_checked", None) != key:
            s = subsets.detach().cpu()
            if tuple(s.shape) != (K, self.disc_shape[0]) or int(s.min()) < 0 or int(s.max()) >= 2 * self.S:
                raise ValueError(f"subsets must be [{K}][{self.disc_shape[0]}] with entries in [0, {2 * self.S})")
            if any(len(set(row.tolist())) != row.numel() for row in s):
                raise ValueError("the columns of one critic must be distinct")
            self._subsets_checked = key
        out = (self._new(self.n_gen), self._new(self.n_gen), self._new(K, self.n_disc), self._new(6), self._new(1, dtype=torch.int32))
        w = (c_float * K)(*[float(x) for x in weights])
        self._check(self._lib.pigan_train_step_grads_hier(
            self._ctx, _ptr(logk_params, "logk_params"), _ptr(u_params, "u_params"), _ptr(disc_params, "disc_params"),
            _ptr(subsets, "subsets", torch.int32), w, _ptr(xy_colloc, "xy_colloc"), _ptr(f, "f"), _ptr(xy_sensors, "xy_sensors"), _ptr(z, "z"),
            _ptr(real_snap, "real_snap"), _ptr(eps, "eps"), float(loss_scale), _ptr(out[0], "g_logk"), _ptr(out[1], "g_u"), _ptr(out[2], "g_disc"),
            _ptr(out[3], "losses"), _ptr(out[4], "found_inf", torch.int32)))
        return out            # no synchronise: the library reads the host array `weights` during the call and passes w_k to its kernels by value

    def adam_update(self, params, grads, m, v, step, lr, beta1, beta2, adam_eps, skip_flag=None):
        import torch
        self._check(self._lib.pigan_adam_update(self._ctx, _ptr(params, "params"), _ptr(grads, "grads"), _ptr(m, "m"), _ptr(v, "v"),
                                                params.numel(), int(step), lr, beta1, beta2, adam_eps,
                                                _ptr(skip_flag, "skip_flag", torch.int32) if skip_flag is not None else None))
