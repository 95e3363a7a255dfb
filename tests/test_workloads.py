"""Host-side checks of the seeded input recipe and the algorithmic flop model."""
import os

import numpy as np

import workloads as wl


def test_flop_model_reproduces_paper_table_II():
    # tests/golden/table2_flops.txt cites PAPER.md Table II; the model counts only the H x H layers:
    # 8 channel-passes (5 for u, 3 for log k) at the f points, 1 at the k/u sensor points
    rows = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "table2_flops.txt")):
        if line.strip() and not line.startswith("#"):
            k, b, fl = line.split(); rows[k] = (int(b), float(fl))
    per_row_layer = 2 * 1024 * 1024; hidden_to_hidden = 20; f_pts, ku_pts = 2000, 200
    fwd = lambda batch: batch * (f_pts * 8 + ku_pts) * hidden_to_hidden * per_row_layer
    assert abs(3 * fwd(rows["generator"][0]) / rows["generator"][1] - 1) < 0.02
    assert abs(fwd(rows["discriminator"][0]) / rows["discriminator"][1] - 1) < 0.02
    assert abs(3 * fwd(rows["generator_fp32"][0]) / rows["generator_fp32"][1] - 1) < 0.02
    assert abs(fwd(rows["discriminator_fp32"][0]) / rows["discriminator_fp32"][1] - 1) < 0.02
    # and the bench's own model uses the same 8 passes per hidden-to-hidden layer
    assert wl.jet_gemm_flops_per_point(21, 1024) == 8 * hidden_to_hidden * per_row_layer


def test_config_table_matches_baseline_json():
    c = wl.CONFIGS
    assert [c[k].N * c[k].P for k in ("c1", "c2", "c3", "c4", "c5")] == [1024, 65536, 524288, 4194304, 4194304]
    assert c["c5"].disc_shape == (10000, 6, 1024) and c["c4"].gen_shape == (1002, 6, 512)
    assert wl.param_count(*c["c5"].gen_shape) == 9348097 and wl.param_count(*c["c3"].disc_shape) == 300289
    f = wl.step_flops(c["c3"]); assert abs(f["total"] / 5.02e12 - 1) < 0.01 and 0.98 < f["jets"] / f["total"] < 0.995
    assert abs(wl.step_flops(c["c5"])["total"] / 1.08e15 - 1) < 0.01


def test_inputs_are_seeded_and_prerounded():
    a = wl.make_inputs(wl.CONFIGS["c2"]); b = wl.make_inputs(wl.CONFIGS["c2"])
    assert all(np.array_equal(a[k], b[k]) for k in a)
    assert np.array_equal(a["theta_u"], a["theta_u"].astype(np.float16).astype(np.float32))     # fp16-representable (c2-c4 run the fp16 arithmetic)
    assert a["theta_u"].astype(np.float16).astype(np.float32).any()
    c5 = wl.make_inputs(wl.CONFIGS["c5"].reduced(2, 4))
    assert np.array_equal(c5["z"], c5["z"].astype(np.float16).astype(np.float32))
    assert a["xy_colloc"].shape == (1024, 2) and np.allclose(a["xy_colloc"][33], [(1 + .5) / 32, (1 + .5) / 32])
    assert np.all(a["f"] == 0) and np.abs(wl.make_inputs(wl.CONFIGS["c3"])["f"]).max() > 0.1


def test_bf16_rounding_is_nearest_even():
    x = np.array([1.0, 1.00390625, 1.005859375, 1.01171875, -3.1415927], dtype=np.float32)
    r = wl.round_to_precision(x, "bf16")
    # 1 + 2^-8 is a tie -> even (1.0); 1 + 1.5*2^-8 -> 1 + 2^-7; 1 + 3*2^-8 is a tie -> even (1 + 2^-6)
    assert list(r[:4]) == [1.0, 1.0, 1.0078125, 1.015625] and abs(r[4] + 3.140625) < 1e-7
