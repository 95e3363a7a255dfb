"""CPU-side checks of the boundary: the library builds/loads and exports every symbol include/pigan.h declares;
argument validation that needs no GPU."""
import ctypes
import os
import re

import paper_1910_13444_b200 as pkg

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_header_and_library_agree():
    header = open(os.path.join(ROOT, "include", "pigan.h")).read()
    declared = sorted(set(re.findall(r"\b(pigan_[a-z_]+)\s*\(", header)))
    lib = pkg.load_library()
    assert declared, "no declarations found"
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in pigan.h but not exported by libpigan.so"
    assert sorted(pkg.EXPORTED_SYMBOLS) == declared


def test_param_count_and_null_handling():
    assert pkg.param_count(6, 3, 32) == 2369 and pkg.param_count(10000, 6, 1024) == 15490049
    lib = pkg.load_library()
    assert lib.pigan_param_count(None) == 0
    assert lib.pigan_launch_count(None) == 0
    assert lib.pigan_last_error(None) == b"null context"
    lib.pigan_destroy(None)
    ctx = ctypes.c_void_p()
    assert lib.pigan_create(None, None, ctypes.byref(ctx)) == 1 and not ctx.value           # INVALID_ARG
    assert lib.pigan_gen_jet_forward(None, None, None, 0, None, 0, 0, None) == 1
    assert lib.pigan_adam_update(None, None, None, None, None, 0, 1, 0.0, 0.0, 0.0, 0.0, None) == 1


def test_create_validates_config_before_touching_cuda():
    lib = pkg.load_library()
    ctx = ctypes.c_void_p()
    bad_shape = pkg._Config(pkg._MlpShape(7, 3, 32), pkg._MlpShape(20, 3, 32), 4, 16, 64, 10, 0, 10.0, 1.0, 0, 0, 0)   # gen.in_dim != 2 + m
    assert lib.pigan_create(ctypes.byref(bad_shape), None, ctypes.byref(ctx)) == 2                                   # SHAPE
    unsup = pkg._Config(pkg._MlpShape(6, 3, 32), pkg._MlpShape(20, 3, 32), 4, 16, 64, 10, 1, 10.0, 1.0, 0, 0, 0)         # bf16 with width 32
    assert lib.pigan_create(ctypes.byref(unsup), None, ctypes.byref(ctx)) == 5                                       # UNSUPPORTED
    fp16_w32 = pkg._Config(pkg._MlpShape(6, 3, 32), pkg._MlpShape(20, 3, 32), 4, 16, 64, 10, 2, 10.0, 1.0, 0, 0, 0)      # fp16 with width 32
    assert lib.pigan_create(ctypes.byref(fp16_w32), None, ctypes.byref(ctx)) == 5
    bf16_w128 = pkg._Config(pkg._MlpShape(6, 3, 128), pkg._MlpShape(20, 3, 32), 4, 16, 64, 10, 1, 10.0, 1.0, 0, 0, 0)    # PIGAN_BF16 at a width fp16 supports:
    assert lib.pigan_create(ctypes.byref(bf16_w128), None, ctypes.byref(ctx)) == 5                                   # refused, never aliased to fp16
    neg = pkg._Config(pkg._MlpShape(6, 0, 32), pkg._MlpShape(20, 3, 32), 4, 16, 64, 10, 0, 10.0, 1.0, 0, 0, 0)
    assert lib.pigan_create(ctypes.byref(neg), None, ctypes.byref(ctx)) == 1


def test_no_cpu_fallback():
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(pkg.PiganError):
        pkg.PiGan(latent_dim=4, gen_hidden=3, gen_width=32, disc_hidden=3, disc_width=32, n_samples=16, n_colloc=64, n_sensors=10)


def test_create_validates_the_next_row_fields():
    """gen_variant / n_free / n_critics are checked before any CUDA call."""
    lib = pkg.load_library()
    ctx = ctypes.c_void_p()
    mk = lambda disc_in, variant, n_free, n_critics, n_colloc=64: pkg._Config(pkg._MlpShape(6, 3, 32), pkg._MlpShape(disc_in, 3, 32), 4, 16, n_colloc, 10, 0,
                                                                             10.0, 1.0, 0, 0, 0, variant, n_free, n_critics)
    assert lib.pigan_create(ctypes.byref(mk(20, 3, 0, 0)), None, ctypes.byref(ctx)) == 1          # unknown gen_variant
    assert lib.pigan_create(ctypes.byref(mk(20, 0, -1, 0)), None, ctypes.byref(ctx)) == 1         # negative n_free
    assert lib.pigan_create(ctypes.byref(mk(20, 0, 8, 0, n_colloc=8)), None, ctypes.byref(ctx)) == 2     # free sensors: disc.in_dim must be 2S + 3F
    assert lib.pigan_create(ctypes.byref(mk(44, 0, 8, 0, n_colloc=64)), None, ctypes.byref(ctx)) == 2    # ... and n_colloc = F
    assert lib.pigan_create(ctypes.byref(mk(44, 1, 8, 0, n_colloc=8)), None, ctypes.byref(ctx)) == 5     # free sensors with the shared trunk: unsupported
    assert lib.pigan_create(ctypes.byref(mk(24, 0, 0, 3)), None, ctypes.byref(ctx)) == 2          # a critic cannot see more than the 2S columns
    assert lib.pigan_create(ctypes.byref(mk(8, 2, 0, 3)), None, ctypes.byref(ctx)) == 5           # hierarchical critics with the trunk: unsupported
    assert not ctx.value
    assert pkg.trunk_param_count(6, 3, 32) == pkg.param_count(6, 3, 32) + 33
