"""Shared helpers of the GPU parity tests: run the oracle and the CUDA path on the same seeded inputs and report,
per output tensor, max|gpu - ref| / max|ref| (reading G20 in DESIGN.md)."""
from __future__ import annotations

import numpy as np

import workloads as wl
from oracle import pigan_oracle as orc


def rel_err(gpu, ref) -> float:
    gpu = np.asarray(gpu, dtype=np.float64); ref = np.asarray(ref, dtype=np.float64)
    scale = np.abs(ref).max() if ref.size else 0.0
    if not np.all(np.isfinite(gpu)):
        return float("inf")
    if scale == 0.0:
        return float(np.abs(gpu).max()) if gpu.size else 0.0
    return float(np.abs(gpu - ref).max() / scale)


def oracle_real_snapshots(cfg, inp):
    """X_real = teacher generator pair evaluated at the sensors for z_real (by the oracle), cast to fp32."""
    Ys = orc.gen_jet_forward_ref(inp["teacher_Y"], *cfg.gen_shape, inp["xy_sensors"], inp["z_real"], 0)[0]
    Us = orc.gen_jet_forward_ref(inp["teacher_u"], *cfg.gen_shape, inp["xy_sensors"], inp["z_real"], 0)[0]
    return np.concatenate([Ys, Us], axis=1).astype(np.float32)


def per_layer(flat, shape):
    out = {}
    for l, (W, b) in enumerate(orc.unpack_params(np.asarray(flat, dtype=np.float64), *shape), start=1):
        out[f"W{l}"] = W; out[f"b{l}"] = b
    return out


def to_dev(inp, device):
    import torch
    return {k: torch.from_numpy(np.ascontiguousarray(v)).to(device) for k, v in inp.items()}


def step_parity(cfg, bias_std=0.1, loss_scale=1.0, workspace_bytes=0, pde_weight=1.0):
    """Returns (errors: dict name -> rel err, losses_gpu, losses_ref, found_inf)."""
    import torch
    from paper_1910_13444_b200 import PiGan
    inp = wl.make_inputs(cfg, bias_std=bias_std)
    inp["real"] = oracle_real_snapshots(cfg, inp)
    gY, gu, gD, losses = orc.train_step_grads_ref(cfg.gen_shape, cfg.disc_shape, inp["theta_Y"], inp["theta_u"], inp["theta_D"],
                                                  inp["xy_colloc"], inp["f"], inp["xy_sensors"], inp["z"], inp["real"], inp["eps"],
                                                  10.0, pde_weight)
    d = to_dev(inp, "cuda:0")
    pg = PiGan.from_config(cfg, workspace_bytes=workspace_bytes, pde_weight=pde_weight)
    out = pg.train_step_grads(d["theta_Y"], d["theta_u"], d["theta_D"], d["xy_colloc"], d["f"], d["xy_sensors"], d["z"], d["real"],
                              d["eps"], loss_scale)
    torch.cuda.synchronize()
    errs = {}
    for name, g_gpu, g_ref, shape in (("gY", out[0], gY, cfg.gen_shape), ("gu", out[1], gu, cfg.gen_shape), ("gD", out[2], gD, cfg.disc_shape)):
        a = per_layer(g_gpu.cpu().numpy(), shape); b = per_layer(g_ref, shape)
        for k in a:
            errs[f"{name}.{k}"] = rel_err(a[k], b[k])
    lg = out[3].cpu().numpy().astype(np.float64)
    pg.close()
    return errs, lg, losses, int(out[4].item())


def jets_parity(cfg, jet_order=2, bias_std=0.1, n_samples=None, xy=None, workspace_bytes=0):
    import torch
    from paper_1910_13444_b200 import PiGan
    inp = wl.make_inputs(cfg, bias_std=bias_std)
    z = inp["z"][:n_samples] if n_samples else inp["z"]
    xy = inp["xy_colloc"] if xy is None else xy
    ref = orc.gen_jet_forward_ref(inp["theta_u"], *cfg.gen_shape, xy, z, jet_order)
    pg = PiGan.from_config(cfg, workspace_bytes=workspace_bytes)
    dev = "cuda:0"
    out = pg.gen_jet_forward(torch.from_numpy(inp["theta_u"]).to(dev), torch.from_numpy(np.ascontiguousarray(xy)).to(dev),
                             torch.from_numpy(np.ascontiguousarray(z)).to(dev), jet_order)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    pg.close()
    return {f"ch{c}": rel_err(got[c], ref[c]) for c in range(ref.shape[0])}, got, ref
