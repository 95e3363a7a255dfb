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


_ORACLE_CACHE = {}


def oracle_step(cfg, bias_std=0.1, pde_weight=1.0, weight_gain=1.0):
    """Inputs + oracle results of one step (cached per configuration: the big cases take the oracle a minute)."""
    key = (cfg, bias_std, pde_weight, weight_gain)
    if key not in _ORACLE_CACHE:
        inp = wl.make_inputs(cfg, bias_std=bias_std)
        if weight_gain != 1.0:                             # weights larger than Xavier-at-init (the hidden layers' W only)
            for name in ("theta_Y", "theta_u"):
                inp[name] = wl.round_to_precision(scale_hidden_weights(inp[name], cfg.gen_shape, weight_gain), cfg.precision)
        inp["real"] = oracle_real_snapshots(cfg, inp)
        ref = orc.train_step_grads_ref(cfg.gen_shape, cfg.disc_shape, inp["theta_Y"], inp["theta_u"], inp["theta_D"], inp["xy_colloc"], inp["f"],
                                       inp["xy_sensors"], inp["z"], inp["real"], inp["eps"], 10.0, pde_weight)
        _ORACLE_CACHE.clear()                              # keep one entry: the tapes of the big cases are gigabytes
        _ORACLE_CACHE[key] = (inp, ref)
    return _ORACLE_CACHE[key]


def scale_hidden_weights(theta, shape, gain):
    """theta with W_2..W_L multiplied by `gain` (input generator only: no arithmetic of the method)."""
    in_dim, L, H = shape
    out = np.array(theta, dtype=np.float32)
    off = H * in_dim + H
    for _ in range(L - 1):
        out[off:off + H * H] *= gain
        off += H * H + H
    return out


def step_parity(cfg, bias_std=0.1, loss_scale=1.0, workspace_bytes=0, pde_weight=1.0, chunk_rows=0, flags=0, weight_gain=1.0, calls=1):
    """Returns (errors: dict name -> rel err, losses_gpu, losses_ref, found_inf).  calls > 1 repeats the call with the same
    arguments (call 2 captures the CUDA graph, call 3+ replays it) and reports the last one."""
    import torch
    from paper_1910_13444_b200 import PiGan
    inp, (gY, gu, gD, losses) = oracle_step(cfg, bias_std, pde_weight, weight_gain)
    d = to_dev(inp, "cuda:0")
    pg = PiGan.from_config(cfg, workspace_bytes=workspace_bytes, pde_weight=pde_weight, chunk_rows=chunk_rows, flags=flags)
    out = None
    for _ in range(calls):
        out = pg.train_step_grads(d["theta_Y"], d["theta_u"], d["theta_D"], d["xy_colloc"], d["f"], d["xy_sensors"], d["z"], d["real"],
                                  d["eps"], loss_scale, out=out)
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


# ---- NEXT-1: shared-trunk generator ------------------------------------------------------------------------------
def per_layer_trunk(flat, shape):
    out = {}
    for l, (W, b) in enumerate(orc.unpack_trunk_params(np.asarray(flat, dtype=np.float64), *shape), start=1):
        out[f"W{l}"] = W; out[f"b{l}"] = b
    return out


def trunk_step_parity(cfg, skip, bias_std=0.1, loss_scale=1.0, chunk_rows=0, pde_weight=1.0):
    """Step with the paper's generator (gen_variant trunk / trunk_skip) against train_step_grads_trunk_ref."""
    import torch
    from paper_1910_13444_b200 import PiGan
    inp = wl.make_inputs(cfg, bias_std=bias_std)
    J = orc.trunk_jet_forward_ref(inp["teacher_G"], *cfg.gen_shape, inp["xy_sensors"], inp["z_real"], 0, skip)
    inp["real"] = np.concatenate([J[0][0], J[1][0]], axis=1).astype(np.float32)
    gG, gD, losses = orc.train_step_grads_trunk_ref(cfg.gen_shape, cfg.disc_shape, inp["theta_G"], inp["theta_D"], inp["xy_colloc"], inp["f"],
                                                    inp["xy_sensors"], inp["z"], inp["real"], inp["eps"], 10.0, pde_weight, skip=skip)
    d = to_dev(inp, "cuda:0")
    pg = PiGan.from_config(cfg, pde_weight=pde_weight, chunk_rows=chunk_rows, gen_variant="trunk_skip" if skip else "trunk")
    out = pg.train_step_grads(d["theta_G"], None, d["theta_D"], d["xy_colloc"], d["f"], d["xy_sensors"], d["z"], d["real"], d["eps"], loss_scale)
    torch.cuda.synchronize()
    errs = {}
    a = per_layer_trunk(out[0].cpu().numpy(), cfg.gen_shape); b = per_layer_trunk(gG, cfg.gen_shape)
    for k in a:
        errs[f"gG.{k}"] = rel_err(a[k], b[k])
    a = per_layer(out[2].cpu().numpy(), cfg.disc_shape); b = per_layer(gD, cfg.disc_shape)
    for k in a:
        errs[f"gD.{k}"] = rel_err(a[k], b[k])
    lg = out[3].cpu().numpy().astype(np.float64)
    fi = int(out[4].item())
    # jets of both heads through the forward-only entry point
    Jg = pg.trunk_jet_forward(d["theta_G"], d["xy_colloc"], d["z"], 2).cpu().numpy()
    Jr = orc.trunk_jet_forward_ref(inp["theta_G"], *cfg.gen_shape, inp["xy_colloc"], inp["z"], 2, skip)
    for k in range(2):
        for c in range(5):
            errs[f"jet.head{k}.ch{c}"] = rel_err(Jg[k][c], Jr[k][c])
    pg.close()
    return errs, lg, losses, fi


# ---- NEXT-2: f at per-sample free sensors fed to the critic --------------------------------------------------------
def free_case(cfg, F, bias_std=0.1):
    """Seeded inputs of a NEXT-2 case (no arithmetic of the method beyond calling the oracle for the real snapshots)."""
    import dataclasses
    cfgF = dataclasses.replace(cfg, G=1)                    # the grid is unused: n_colloc = F points per sample
    inp = wl.make_inputs(cfgF, bias_std=bias_std)
    S = cfg.S
    disc_shape = (2 * S + 3 * F, cfg.LD, cfg.HD)
    inp["theta_D"] = wl.round_to_precision(wl.xavier_params(np.random.default_rng(1000 * cfg.index + 2), *disc_shape, bias_std=bias_std), cfg.precision)
    xy_free = wl.free_sensor_points(cfg, F); xy_real = wl.free_sensor_points(cfg, F, real=True)
    # "real" snapshots: the teacher pair at the sensors, f = 0 at that realization's free sensors (the paper's data solve Eq. 1 with f = 0)
    Xr, _ = orc.free_snapshot_ref(cfg.gen_shape, inp["teacher_Y"], inp["teacher_u"], xy_real, inp["xy_sensors"], inp["z_real"])
    Xr[:, 2 * S:2 * S + F] = 0.0
    return inp, disc_shape, xy_free, Xr.astype(np.float32)


def free_score_sensitivity(cfg, F, inp, disc_shape, xy_free):
    """(B, grad_f, f): by the fp64 oracle, grad_f = d mean D(X_fake) / d f [N][F] and B = max|f| * sum|grad_f|, the first-order bound
    on the change of mean D(fake) per unit RELATIVE (to max|f|) perturbation of the f entries of the snapshot."""
    S = cfg.S
    X, _ = orc.free_snapshot_ref(cfg.gen_shape, inp["theta_Y"], inp["theta_u"], xy_free, inp["xy_sensors"], inp["z"])
    lay = orc.unpack_params(inp["theta_D"], *disc_shape)
    g, _ = orc._disc_forward(lay, X)
    dX = orc._disc_backward(lay, g, np.full(X.shape[0], 1.0 / X.shape[0]), None)
    f, gf = X[:, 2 * S:2 * S + F], dX[:, 2 * S:2 * S + F]
    return float(np.abs(f).max() * np.abs(gf).sum()), gf, f


def free_step_parity(cfg, F, bias_std=0.1, loss_scale=1.0, chunk_rows=0, pde_weight=0.0):
    """Returns (errors, losses_gpu, losses_ref, found_inf, B) with B from free_score_sensitivity."""
    import torch
    from paper_1910_13444_b200 import PiGan
    inp, disc_shape, xy_free, real = free_case(cfg, F, bias_std)
    S = cfg.S
    gY, gu, gD, losses = orc.train_step_grads_free_ref(cfg.gen_shape, disc_shape, inp["theta_Y"], inp["theta_u"], inp["theta_D"], xy_free,
                                                       inp["xy_sensors"], inp["z"], real, inp["eps"], 10.0, pde_weight)
    B = free_score_sensitivity(cfg, F, inp, disc_shape, xy_free)[0]
    dev = "cuda:0"
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    pg = PiGan(latent_dim=cfg.m, gen_hidden=cfg.L, gen_width=cfg.H, disc_hidden=cfg.LD, disc_width=cfg.HD, n_samples=cfg.N, n_colloc=F,
               n_sensors=S, precision=cfg.precision, pde_weight=pde_weight, chunk_rows=chunk_rows, n_free=F)
    out = pg.train_step_grads(t(inp["theta_Y"]), t(inp["theta_u"]), t(inp["theta_D"]), t(xy_free), None, t(inp["xy_sensors"]), t(inp["z"]), t(real),
                              t(inp["eps"]), loss_scale)
    torch.cuda.synchronize()
    errs = {}
    for name, g_gpu, g_ref, shape in (("gY", out[0], gY, cfg.gen_shape), ("gu", out[1], gu, cfg.gen_shape), ("gD", out[2], gD, disc_shape)):
        a = per_layer(g_gpu.cpu().numpy(), shape); b = per_layer(g_ref, shape)
        for k in a:
            errs[f"{name}.{k}"] = rel_err(a[k], b[k])
    lg = out[3].cpu().numpy().astype(np.float64)
    fi = int(out[4].item())
    pg.close()
    return errs, lg, losses, fi, B
