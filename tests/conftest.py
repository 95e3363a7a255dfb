import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def tiny():
    """A tiny PI-GAN instance with non-zero biases (exercises every term of the oracle)."""
    import numpy as np
    from workloads import Config, xavier_params, collocation_grid
    cfg = Config("tiny", 9, "fp32", m=3, L=3, H=7, G=3, N=2, S=4, LD=3, HD=6, f_kind="zero")
    rng = np.random.default_rng(1234)
    d = {
        "cfg": cfg,
        "theta_Y": xavier_params(rng, *cfg.gen_shape, bias_std=0.3),
        "theta_u": xavier_params(rng, *cfg.gen_shape, bias_std=0.3),
        "theta_D": xavier_params(rng, *cfg.disc_shape, bias_std=0.3),
        "xy_colloc": collocation_grid(cfg.G).astype(np.float64),
        "xy_sensors": rng.uniform(size=(cfg.S, 2)),
        "z": rng.normal(size=(cfg.N, cfg.m)),
        "f": rng.normal(size=cfg.P),
        "real": rng.normal(size=(cfg.N, 2 * cfg.S)),
        "eps": rng.uniform(size=cfg.N),
    }
    return d
