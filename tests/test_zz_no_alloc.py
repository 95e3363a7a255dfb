"""pigan_darcy_residual_static: the residual for callers that cannot allocate device memory.

Who needs it: a program embedded in a host that handed all GPU memory to its own pool at start-up (cudaMalloc fails there or
is against the host's rules), or a loop with a latency budget that keeps cudaMalloc / cudaFree out of its steady state because
they can stall the device.  Every other call of the library needs a context, and creating a context allocates workspaces.
The static call keeps its scratch in an array compiled into the library, shared by all calls on a GPU and never cleared
between them -- which is why this test calls it TWICE in a row with different sizes: the second, smaller call must not see
what the first one left in the array.

The reference here is the library's own context-based pigan_darcy_residual (that one is checked against the oracle in
test_gpu_parity.py), at the tolerance that test uses (1e-5 relative).  This file is named to be collected last, so that a failure
here under `pytest -x` cannot hide another test; it passes alone in a fresh process as well as after the other tests.
"""
import ctypes
import os

import numpy as np
import pytest

import paper_1910_13444_b200 as pkg
import workloads as wl

TOL = 1e-5          # test_residual_entry_point_manufactured_solution's tolerance for r and for mean r^2


def _jets(seed, N, P):
    rng = np.random.default_rng(seed)
    Y = rng.normal(scale=0.5, size=(3, N, P)).astype(np.float32)
    U = rng.normal(size=(5, N, P)).astype(np.float32)
    f = rng.normal(size=P).astype(np.float32)
    return Y, U, f


@pytest.mark.gpu
def test_static_residual_matches_the_context_path_on_two_calls_in_a_row():
    import torch
    dev = torch.device("cuda:0")
    pg = pkg.PiGan.from_config(wl.CONFIGS["c1"])          # the existing path (allocates its workspaces; the static call does not use it)
    # call 1: 5 x 1000 rows = five blocks with a ragged last one; call 2: 3 x 77 rows = one block, run straight after call 1
    # so that partial sums 1..4 and the ticket of call 1 are still in the array; call 3 repeats call 1's size on new data.
    for seed, (N, P) in enumerate([(5, 1000), (3, 77), (5, 1000)]):
        Y, U, f = (torch.from_numpy(a).to(dev) for a in _jets(100 + seed, N, P))
        r_ref, msq_ref = pg.darcy_residual(Y, U, f)
        r = torch.full((N, P), float("nan"), device=dev)  # the caller's own outputs, poisoned
        msq = torch.full((1,), float("nan"), device=dev)
        pkg.darcy_residual_static(Y, U, f, r=r, mean_sq=msq)
        torch.cuda.synchronize()
        r_ref, r = r_ref.cpu().numpy(), r.cpu().numpy()
        assert np.all(np.isfinite(r))
        assert np.max(np.abs(r - r_ref)) <= TOL * np.max(np.abs(r_ref)), (N, P)
        assert abs(msq.item() - msq_ref.item()) <= TOL * abs(msq_ref.item()), (N, P, msq.item(), msq_ref.item())
    # outputs are optional one at a time, and an empty problem has mean 0
    Y, U, f = (torch.from_numpy(a).to(dev) for a in _jets(7, 2, 300))
    only = torch.empty(1, device=dev)
    pkg.darcy_residual_static(Y, U, f, mean_sq=only)
    _, both = pg.darcy_residual(Y, U, f)
    assert abs(only.item() - both.item()) <= TOL * abs(both.item())
    lib = pkg.load_library()
    assert lib.pigan_darcy_residual_static(None, None, None, 0, 5, None, ctypes.c_void_p(only.data_ptr()), None) == 0
    torch.cuda.synchronize()
    assert only.item() == 0.0
    pg.close()


def test_static_residual_refuses_more_rows_than_its_scratch_holds():
    """Sizes are checked before any CUDA call, so this runs without a GPU: the pointers are never dereferenced."""
    lib = pkg.load_library()
    fake = ctypes.c_void_p(256)
    n = 4097                                               # 4097 * 4096 rows = 2^24 + 4096
    assert n * 4096 > pkg.STATIC_MAX_ROWS
    assert lib.pigan_darcy_residual_static(fake, fake, fake, n, 4096, fake, fake, None) == 5      # PIGAN_ERR_UNSUPPORTED
    msg = lib.pigan_static_last_error().decode()
    assert str(pkg.STATIC_MAX_ROWS) in msg and "PIGAN_STATIC_MAX_ROWS" in msg
    assert lib.pigan_darcy_residual_static(fake, fake, fake, -1, 4, fake, fake, None) == 1        # PIGAN_ERR_INVALID_ARG
    assert lib.pigan_darcy_residual_static(None, fake, fake, 2, 4, fake, fake, None) == 1
    header = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "pigan.h")).read()
    assert "#define PIGAN_STATIC_MAX_ROWS (1LL << 24)" in header and pkg.STATIC_MAX_ROWS == 1 << 24
