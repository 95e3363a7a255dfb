"""Seeded synthetic inputs for the five BASELINE.json configs (SURVEY.md section 8(d) recipe).

This module is shared by the oracle-side tests, the GPU parity tests and bench.py.  It holds NONE of the
method's arithmetic: only shapes, seeds, random draws, the collocation grid, the source term f and the
rounding of inputs to the operand precision (reading G21: weights and z are pre-rounded to bf16 / fp16 and
stored as fp32 so that oracle and GPU consume identical values).  The "real" snapshots are produced by the
caller (tests: the oracle evaluates the teacher; bench: the GPU library does, outside the timed region).

Seeds: numpy default_rng(1000 * config_index + stream); draws in float64, then cast to float32.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np

PRECISIONS = {"fp32": 0, "bf16": 1, "fp16": 2}       # values of pigan_precision in include/pigan.h


@dataclass(frozen=True)
class Config:
    name: str
    index: int            # 1-based config index (c1..c5)
    precision: str        # "fp32" | "bf16" | "fp16"
    m: int                # latent (stochastic) dimension
    L: int                # generator hidden layers
    H: int                # generator width
    G: int                # collocation grid is G x G, P = G*G
    N: int                # latent samples per step
    S: int                # sensors
    LD: int               # discriminator hidden layers
    HD: int               # discriminator width
    f_kind: str = "zero"  # "zero" | "sin8"
    variant: str = "two_mlps"   # generator: "two_mlps" (BASELINE.json) | "trunk" | "trunk_skip" (the paper's, NEXT-1)

    @property
    def P(self) -> int: return self.G * self.G
    @property
    def gen_shape(self): return (2 + self.m, self.L, self.H)
    @property
    def disc_shape(self): return (2 * self.S, self.LD, self.HD)
    def reduced(self, N: int, G: int) -> "Config":
        """Full network dimensions, fewer rows (parity protocol for c4/c5)."""
        return replace(self, name=f"{self.name}-rows{N}x{G}x{G}", N=N, G=G)


CONFIGS = {
    "c1": Config("c1", 1, "fp32", 4, 3, 32, 8, 16, 10, 3, 32),
    # BASELINE.json names c2-c4 "bf16"; the library's one 16-bit arithmetic is the paper's FP16 (R1), and
    # PIGAN_BF16 is refused by pigan_create, so the configs carry the precision that actually runs.
    "c2": Config("c2", 2, "fp16", 30, 4, 128, 32, 64, 100, 4, 128),
    "c3": Config("c3", 3, "fp16", 60, 4, 256, 64, 128, 200, 4, 256, "sin8"),
    "c4": Config("c4", 4, "fp16", 1000, 6, 512, 128, 256, 1000, 6, 512),
    "c5": Config("c5", 5, "fp16", 4000, 6, 1024, 256, 64, 5000, 6, 1024),
}


# The workload of the paper's Table II: 21 x 1024 network (20 hidden layers + the output layer),
# generator worker with local batch 6 on the top-level subdomain of Dataset 6 (100 log k + 100 u sensors, 2000 f sensors).
# Stand-ins: a 45 x 45 cell-centred grid (2025 points) for the 2000 free f sensors; latent dimension 1000 (the paper does
# not give the generator's noise dimension); the critic gets the same 21 x 1024 shape.
TABLE2 = Config("t2", 6, "fp16", 1000, 20, 1024, 45, 6, 100, 20, 1024, "zero", "trunk_skip")


def param_count(in_dim: int, n_hidden: int, width: int) -> int:
    return width * in_dim + width + (n_hidden - 1) * (width * width + width) + width + 1


def round_to_precision(a: np.ndarray, precision: str) -> np.ndarray:
    """Round-to-nearest-even to the operand precision, returned as float32 (G21)."""
    a = np.asarray(a, dtype=np.float32)
    if precision == "fp32":
        return a.copy()
    if precision == "fp16":
        return a.astype(np.float16).astype(np.float32)
    if precision == "bf16":
        u = a.view(np.uint32).astype(np.uint64)
        u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
        return u.astype(np.uint32).view(np.float32).reshape(a.shape)
    raise ValueError(precision)


def _rng(cfg: Config, stream: int) -> np.random.Generator:
    return np.random.default_rng(1000 * cfg.index + stream)


def xavier_params(rng, in_dim: int, n_hidden: int, width: int, bias_std: float = 0.0) -> np.ndarray:
    """Flat packing: W_l row-major [out][in] then b_l.  Xavier-normal std = sqrt(2/(fan_in+fan_out)); zero biases
    unless bias_std > 0 (tests use non-zero biases to exercise the bias paths)."""
    parts, fan_in = [], in_dim
    for l in range(n_hidden + 1):
        fan_out = width if l < n_hidden else 1
        parts.append(rng.normal(0.0, np.sqrt(2.0 / (fan_in + fan_out)), size=fan_out * fan_in))
        parts.append(rng.normal(0.0, bias_std, size=fan_out) if bias_std > 0 else np.zeros(fan_out))
        fan_in = fan_out
    return np.concatenate(parts)


def xavier_trunk_params(rng, in_dim: int, n_hidden: int, width: int, bias_std: float = 0.0) -> np.ndarray:
    """The paper's shared-trunk generator (NEXT-1): as xavier_params, with a last layer of TWO outputs (log k, u)."""
    parts, fan_in = [], in_dim
    for l in range(n_hidden + 1):
        fan_out = width if l < n_hidden else 2
        parts.append(rng.normal(0.0, np.sqrt(2.0 / (fan_in + fan_out)), size=fan_out * fan_in))
        parts.append(rng.normal(0.0, bias_std, size=fan_out) if bias_std > 0 else np.zeros(fan_out))
        fan_in = fan_out
    return np.concatenate(parts)


def collocation_grid(G: int) -> np.ndarray:
    """Cell-centred G x G grid on the unit square, p = j*G + i -> ((i+1/2)/G, (j+1/2)/G)  (reading G13)."""
    c = (np.arange(G, dtype=np.float64) + 0.5) / G
    X, Y = np.meshgrid(c, c, indexing="xy")
    return np.stack([X.reshape(-1), Y.reshape(-1)], axis=1).astype(np.float32)


def source_term(cfg: Config, xy: np.ndarray) -> np.ndarray:
    """f on the grid: zero (the paper solves Eq. 1 with f = 0) or a seeded sum of 8 sinusoids (c3)."""
    if cfg.f_kind == "zero":
        return np.zeros(xy.shape[0], dtype=np.float32)
    rng = _rng(cfg, 9)
    f = np.zeros(xy.shape[0], dtype=np.float64)
    for _ in range(8):
        A = rng.uniform(-1.0, 1.0)
        while True:
            p, q = rng.integers(0, 4, size=2)
            if p or q:
                break
        phi = rng.uniform(0.0, 2.0 * np.pi)
        f += A * np.sin(2.0 * np.pi * (p * xy[:, 0].astype(np.float64) + q * xy[:, 1].astype(np.float64)) + phi)
    return f.astype(np.float32)


def make_inputs(cfg: Config, bias_std: float = 0.0) -> dict:
    """All host inputs of one step except real_snap (float32 numpy arrays)."""
    pr = cfg.precision
    gen, disc = cfg.gen_shape, cfg.disc_shape
    out = {
        "theta_Y": round_to_precision(xavier_params(_rng(cfg, 0), *gen, bias_std=bias_std), pr),
        "theta_u": round_to_precision(xavier_params(_rng(cfg, 1), *gen, bias_std=bias_std), pr),
        "theta_D": round_to_precision(xavier_params(_rng(cfg, 2), *disc, bias_std=bias_std), pr),
        "teacher_Y": round_to_precision(xavier_params(_rng(cfg, 3), *gen, bias_std=bias_std), pr),
        "teacher_u": round_to_precision(xavier_params(_rng(cfg, 4), *gen, bias_std=bias_std), pr),
        "xy_sensors": _rng(cfg, 5).uniform(0.0, 1.0, size=(cfg.S, 2)).astype(np.float32),
        "z": round_to_precision(_rng(cfg, 6).normal(size=(cfg.N, cfg.m)), pr),
        "z_real": round_to_precision(_rng(cfg, 7).normal(size=(cfg.N, cfg.m)), pr),
        "eps": _rng(cfg, 8).uniform(0.0, 1.0, size=cfg.N).astype(np.float32),
        "xy_colloc": collocation_grid(cfg.G),
    }
    out["f"] = source_term(cfg, out["xy_colloc"])
    # NEXT-1: student and teacher of the shared-trunk variant (streams 10, 11)
    out["theta_G"] = round_to_precision(xavier_trunk_params(_rng(cfg, 10), *gen, bias_std=bias_std), pr)
    out["teacher_G"] = round_to_precision(xavier_trunk_params(_rng(cfg, 11), *gen, bias_std=bias_std), pr)
    return out


def free_sensor_points(cfg: Config, F: int, real: bool = False) -> np.ndarray:
    """NEXT-2: per-realization free-sensor locations [N][F][2], uniform on the unit square, re-drawn for every sample
    (P:127); stream 12 for the generated batch, 13 for the real one."""
    return _rng(cfg, 13 if real else 12).uniform(0.0, 1.0, size=(cfg.N, F, 2)).astype(np.float32)


# ---- algorithmic work model; used by bench.py for the roofline ---------------------
def jet_flops_per_point(L: int, H: int) -> int:
    """Forward flops per (sample, point), both nets: sum over C in {5,3} of (L-1) 2H^2 C + 2HC + 4H."""
    return sum((L - 1) * 2 * H * H * C + 2 * H * C + 4 * H for C in (5, 3))


def jet_gemm_flops_per_point(L: int, H: int) -> int:
    """The dense-contraction part only: (L-1) hidden H x H layers, 8 channel-passes."""
    return (L - 1) * 2 * H * H * 8


def step_flops(cfg: Config) -> dict:
    """Algorithmic flops of one train step (forward + dgrad + wgrad = 3x forward).  Two MLPs: 5 + 3 channel passes and two
    value passes at the sensors; shared trunk (NEXT-1): one 5-channel pass and one value pass."""
    if cfg.variant == "two_mlps":
        jets = 3 * cfg.N * cfg.P * jet_flops_per_point(cfg.L, cfg.H)
        jet_gemm = 3 * cfg.N * cfg.P * jet_gemm_flops_per_point(cfg.L, cfg.H)
        nets = 2
    else:
        jets = 3 * cfg.N * cfg.P * ((cfg.L - 1) * 2 * cfg.H * cfg.H * 5 + 2 * cfg.H * 8 + 2 * cfg.H)
        jet_gemm = 3 * cfg.N * cfg.P * (cfg.L - 1) * 2 * cfg.H * cfg.H * 5
        nets = 1
    zpart = cfg.N * nets * 2 * cfg.m * cfg.H * 3
    sensors = cfg.N * 3 * cfg.S * nets * ((cfg.L - 1) * 2 * cfg.H * cfg.H + 6 * cfg.H)
    critic = cfg.N * 14 * 2 * (2 * cfg.S * cfg.HD + (cfg.LD - 1) * cfg.HD * cfg.HD + cfg.HD)
    return {"jets": jets, "jet_gemm": jet_gemm, "zpart": zpart, "sensors": sensors, "critic": critic,
            "total": jets + zpart + sensors + critic}
