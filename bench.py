#!/usr/bin/env python
"""bench.py -- PI-GAN train-step throughput on B200 (metric of BASELINE.json).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config c5] [--impl pigan|reference] [--all-configs]

A "step" is one pass of the whole hot path: pigan_train_step_grads on one batch of synthetic
input followed by the three pigan_adam_update calls.  The headline workload is config c5 (the largest; DESIGN.md
section 6 says why); --all-configs adds a short run of every other config to the same JSON line.  N > 1 runs N
independent replicas (the path does not shard: north_star says no collectives), one process per GPU under torchrun.
`--impl reference` times the fp64 oracle (oracle/) on the host cores on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
import workloads as wl  # noqa: E402

METRIC = "PI-GAN train-step sample*collocation-points/s"
UNIT = "sample*collocation-points/s"
ADAM = dict(lr=1e-4, beta1=0.5, beta2=0.9, adam_eps=1e-8)          # reading G3
PROFILE_CSVS = [os.path.join(ROOT, "profiles", n) for n in ("r03_step_dram_bytes.csv", "r02_step_dram_bytes.csv")]   # newest first
NCU_METRICS = ("dram__bytes_read.sum", "dram__bytes_write.sum", "gpu__time_duration.sum", "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_elapsed")


def library_srchash():
    """Content hash of the library's sources (what paper_1910_13444_b200/build.py stamps into libpigan.so.srchash)."""
    from paper_1910_13444_b200.build import source_hash
    return source_hash()


def ncu_profile(cfg_name):
    """Per kernel class of `cfg_name`: launches, DRAM bytes and tensor-pipe-active % of ONE timed step, as measured by the ncu
    pass recorded under profiles/ (not by this run); taken from the newest summary that has rows for the config.  Returns
    (rows, source file, stale): stale = the summary carries no source hash or was taken on other library sources than the
    ones in the tree, i.e. a kernel may have changed since."""
    import csv
    for path in PROFILE_CSVS:
        if not os.path.exists(path):
            continue
        out, hashes = {}, set()
        for r in csv.DictReader(open(path)):
            if r["config"] == cfg_name:
                out[r["kernel_class"]] = {"launches": int(r["launches"]), "dram_bytes": int(r["dram_bytes_read"]) + int(r["dram_bytes_write"]),
                                          "tensor_pct": float(r["tensor_pipe_active_pct_time_weighted"] or 0.0)}
                hashes.add(r.get("srchash") or "")
        if out:
            return out, os.path.relpath(path, ROOT), hashes != {library_srchash()}
    return {}, None, None


def kernel_class(name):
    """ncu's demangled kernel name -> the class names of pigan_profile_report where a class spans several kernels, else the function name."""
    import re
    m = re.match(r"(?:void )?(?:\(anonymous namespace\)::|<unnamed>::|pigan::)*([A-Za-z_0-9]+)(?:<([^>]*)>)?", name)
    fn, targs = m.group(1), [a.strip() for a in (m.group(2) or "").split(",")]
    ints = [int(a) for a in targs if re.fullmatch(r"-?\d+", a)]
    if fn in ("jet2_layer_kernel", "jet_layer_kernel") and len(ints) >= 2:
        C, mode = ints[0], ints[1]
        return {0: f"jet_layer_fwd(C={C})", 4: f"jet_layer_fwd(C={C})", 2: f"jet_layer_fwd_split(C={C})", 5: f"jet_layer_fwd_split(C={C})",
                1: f"jet_layer_bwd(C={C})", 3: f"jet_layer_bwd(C={C})"}.get(mode, fn)
    if fn in ("wgrad2_kernel", "wgrad_kernel"):
        return "wgrad"
    if fn in ("fused_bwd256_kernel", "fused_bwd128_kernel") and ints:
        return f"jet_layer_bwd_wgrad(C={ints[0]})"
    if fn == "fused_fwd128_kernel" and ints:
        return f"gen_fwd_fused(C={ints[0]})"
    return fn


def ncu_summary(path, cfg_name, out=sys.stdout):
    """Sums a per-launch ncu CSV (--csv --metrics NCU_METRICS, one timed step in the NVTX range) per kernel class and prints the
    rows of profiles/rNN_step_dram_bytes.csv for `cfg_name`, stamped with the hash of the library sources in the tree."""
    import csv
    import io
    lines = [l for l in open(path) if l.startswith('"')]
    per = {}                                                   # launch id -> {kernel, metric: value}
    for r in csv.DictReader(io.StringIO("".join(lines))):
        d = per.setdefault(r["ID"], {"kernel": r["Kernel Name"]})
        v = float(r["Metric Value"].replace(",", ""))
        unit = r["Metric Unit"]
        if r["Metric Name"].startswith("dram__bytes"):
            v *= {"byte": 1, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(unit, 1)
        if r["Metric Name"] == "gpu__time_duration.sum":
            v *= {"ns": 1e-3, "us": 1, "usecond": 1, "ms": 1e3, "msecond": 1e3, "nsecond": 1e-3, "second": 1e6}.get(unit, 1)     # -> us
        d[r["Metric Name"]] = v
    agg = {}
    for d in per.values():
        for cls in (kernel_class(d["kernel"]), "WHOLE_STEP"):
            a = agg.setdefault(cls, [0, 0.0, 0.0, 0.0, 0.0])
            t = d.get(NCU_METRICS[2], 0.0)
            a[0] += 1; a[1] += t; a[2] += d.get(NCU_METRICS[0], 0.0); a[3] += d.get(NCU_METRICS[1], 0.0); a[4] += t * d.get(NCU_METRICS[3], 0.0)
    h = library_srchash()
    w = csv.writer(out)
    w.writerow(["config", "kernel_class", "launches", "kernel_time_us_under_ncu", "dram_bytes_read", "dram_bytes_write",
                "tensor_pipe_active_pct_time_weighted", "srchash"])
    for cls, a in sorted(agg.items(), key=lambda kv: -kv[1][1]):
        w.writerow([cfg_name, cls, a[0], round(a[1], 1), int(a[2]), int(a[3]), round(a[4] / a[1], 1) if a[1] > 0 else 0.0, h])


# ----------------------------------------------------------------------------------------------------------------
def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "tflops_burst": d["bf16_tflops"], "tflops_sustained": d["bf16_tflops_sustained"], "source": "measured"}
    return {"hbm_gbs": 6650.0, "tflops_burst": 1590.0, "tflops_sustained": 1400.0, "source": "fallback"}


def max_over_ranks(t_ms: float, dist=None, device=None) -> float:
    """Max of a per-rank time over all ranks (the only exchange of the replicas-only multi-GPU mode).  Works on any
    torch.distributed backend: NCCL with a CUDA device in bench runs, gloo with CPU tensors in the CPU tests."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(t_ms)
    import torch
    t = torch.tensor([t_ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.barrier()
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank: int, world: int, t_max_ms: float) -> float:
    """Whole-job throughput of `world` independent replicas: all ranks' units over the slowest rank's time (weak scaling)."""
    return world * units_per_rank / (t_max_ms * 1e-3)


def hbm_class_bytes(cfg) -> dict:
    """Algorithmic bytes per step of the HBM-bound kernel classes: one pass over the C planes they
    read / write for the collocation rows of both nets (C = 3 + 5) and the sensor rows (C = 1 per net; the snapshot
    forward carries 2 planes), 28 B per parameter for Adam, 16 floats per row for the residual."""
    e = 4 if cfg.precision == "fp32" else 2
    rows, srows, H = cfg.N * cfg.P, cfg.N * cfg.S, cfg.H
    plane = H * e
    two = cfg.variant == "two_mlps"
    col = ((3 + 5) if two else 5) * rows * plane            # one pass over the C planes of the net(s), collocation rows
    sen = (2 if two else 1) * srows * plane                 # one pass over the value plane of the net(s), sensor rows
    n_par = (2 if two else 1) * wl.param_count(*cfg.gen_shape) + wl.param_count(*cfg.disc_shape)
    fused_fwd = e == 2 and two and H == 128 and cfg.P % 64 == 0 and 2 <= cfg.L <= 5     # tc_fused_fwd.cu computes the first layer of the collocation rows
    return {"first_layer_fwd": (0 if fused_fwd else col) + sen * (1 + (2 if e == 2 else 1)),   # writes h^1: collocation, sensor pass with stash, snapshot pass (hi, lo)
            "out_fwd": (0 if fused_fwd else col) + sen * (1 + (2 if e == 2 else 1)),           # reads h^L (the fused forward reduces the output dot itself)
            "jet_act_bwd": 2 * (col + sen),                               # top layer: reads h^L, writes ahat^L
            "first_layer_bwd": sen + (0 if (e == 2 and cfg.H % 256 == 0 and cfg.P % 64 == 0) else col),   # collocation part fused into the layer-2 dgrad when it can be
            "adam": 28 * n_par, "residual": 16 * 4 * rows}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index=0, period=0.1):
        super().__init__(daemon=True)
        self.index, self.period, self.samples, self.reasons, self.max_mhz = index, period, [], set(), None
        self._stop_evt = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if not self.nv:
            return
        nv = self.nv
        names = {"hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown if hasattr(nv, "nvmlClocksEventReasonHwSlowdown") else nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0)),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0)),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0))}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if bit and (r & bit):
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop_evt.wait(self.period)

    def finish(self):
        self._stop_evt.set()
        self.join(timeout=2)
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ----------------------------------------------------------------------------------------------------------------
def cpu_sample_config(cfg, flop_budget=1.5e12):
    """Bounded sample of cfg for the oracle (about 10-30 s of fp64 numpy work): full generator dimensions, a 32x32
    grid, N' samples chosen from a flop budget, sensors scaled to keep the config's P:S ratio (so that the cost per
    (sample x point) is representative of the full workload)."""
    if wl.step_flops(cfg)["total"] <= flop_budget:
        return cfg, "whole workload"
    Gp = min(cfg.G, 32)
    per_row = 3 * wl.jet_flops_per_point(cfg.L, cfg.H)
    Np = int(min(cfg.N, max(1, round(flop_budget / per_row / (Gp * Gp)))))
    Sp = max(2, int(round(cfg.S * (Gp * Gp) / cfg.P)))
    s = dataclasses.replace(cfg, name=cfg.name + "-cpu-sample", N=Np, G=Gp, S=Sp)
    return s, f"N={Np} samples x {Gp}x{Gp} grid, S={Sp} sensors (same P:S ratio), full generator dims {cfg.L}x{cfg.H}, m={cfg.m}"


def time_oracle(cfg, steps=1, warmup=0):
    """Times oracle.train_step_grads_ref (+ Adam) as it stands on the host cores.  Returns (units/s, seconds per step, cores, sample)."""
    from oracle import pigan_oracle as orc
    scfg, sample = cpu_sample_config(cfg)
    inp = wl.make_inputs(scfg)
    Ys = orc.gen_jet_forward_ref(inp["teacher_Y"], *scfg.gen_shape, inp["xy_sensors"], inp["z_real"], 0)[0]
    Us = orc.gen_jet_forward_ref(inp["teacher_u"], *scfg.gen_shape, inp["xy_sensors"], inp["z_real"], 0)[0]
    real = np.concatenate([Ys, Us], axis=1)
    th = [inp["theta_Y"].astype(np.float64), inp["theta_u"].astype(np.float64), inp["theta_D"].astype(np.float64)]
    mom = [(np.zeros_like(t), np.zeros_like(t)) for t in th]
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        g = orc.train_step_grads_ref(scfg.gen_shape, scfg.disc_shape, th[0], th[1], th[2], inp["xy_colloc"], inp["f"], inp["xy_sensors"],
                                     inp["z"], real, inp["eps"], 10.0, 1.0)
        for k in range(3):
            th[k], m, v = orc.adam_update_ref(th[k], g[k], mom[k][0], mom[k][1], it + 1, ADAM["lr"], ADAM["beta1"], ADAM["beta2"], ADAM["adam_eps"])
            mom[k] = (m, v)
        dt = time.perf_counter() - t0
        if it >= warmup:
            times.append(dt)
    sec = float(np.mean(times))
    try:
        from threadpoolctl import threadpool_info
        cores = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        cores = os.cpu_count()
    return scfg.N * scfg.P / sec, sec, cores, sample


# ----------------------------------------------------------------------------------------------------------------
class GpuWorkload:
    """Device-resident synthetic inputs + state of one config."""

    def __init__(self, cfg, device, seed_shift=0, chunk_rows=0):
        import torch
        from paper_1910_13444_b200 import PiGan
        self.cfg, self.device, self.torch = cfg, device, torch
        inp = wl.make_inputs(cfg)
        if seed_shift:      # data-parallel ranks are REPLICAS: identical parameters (and teachers), their own latent / real / eps streams
            own = wl.make_inputs(dataclasses.replace(cfg, index=cfg.index + 10 * seed_shift))
            for k in ("z", "z_real", "eps"):
                inp[k] = own[k]
        self.trunk = cfg.variant != "two_mlps"
        self.pg = PiGan.from_config(cfg, device=device, chunk_rows=chunk_rows, gen_variant=cfg.variant)
        d = {k: torch.from_numpy(np.ascontiguousarray(v)).to(device) for k, v in inp.items()}
        # "real" snapshots: the frozen teacher evaluated at the sensors by the GPU library, outside any timed region
        if self.trunk:
            J = self.pg.trunk_jet_forward(d["teacher_G"], d["xy_sensors"], d["z_real"], 0)
            Ys, Us = J[0][0], J[1][0]
        else:
            Ys = self.pg.gen_jet_forward(d["teacher_Y"], d["xy_sensors"], d["z_real"], 0)[0]
            Us = self.pg.gen_jet_forward(d["teacher_u"], d["xy_sensors"], d["z_real"], 0)[0]
        d["real"] = torch.cat([Ys, Us], dim=1).contiguous()
        self.d = d
        self.params = [d["theta_G"].clone(), d["theta_D"].clone()] if self.trunk else [d["theta_Y"].clone(), d["theta_u"].clone(), d["theta_D"].clone()]
        self.mom = [(torch.zeros_like(p), torch.zeros_like(p)) for p in self.params]
        if self.trunk:
            self.out = (torch.empty_like(self.params[0]), None, torch.empty_like(self.params[1]),
                        torch.empty(6, device=device), torch.zeros(1, dtype=torch.int32, device=device))
        else:
            self.out = (torch.empty_like(self.params[0]), torch.empty_like(self.params[1]), torch.empty_like(self.params[2]),
                        torch.empty(6, device=device), torch.zeros(1, dtype=torch.int32, device=device))
        self.loss_scale = 1024.0 if cfg.precision == "fp16" else 1.0
        self.step_no = 0
        # pinned host copies of the per-step inputs for the end-to-end leg
        self.host = {k: inp_k.cpu().pin_memory() for k, inp_k in (("z", d["z"]), ("real", d["real"]), ("eps", d["eps"]))}
        self.host_out = torch.empty(6, dtype=torch.float32).pin_memory()
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=device) if cfg.N * cfg.P < 400000 else None

    def step(self):
        d, pg = self.d, self.pg
        self.step_no += 1
        if self.trunk:
            pg.train_step_grads(self.params[0], None, self.params[1], d["xy_colloc"], d["f"], d["xy_sensors"], d["z"], d["real"],
                                d["eps"], self.loss_scale, out=self.out)
            grads = (self.out[0], self.out[2])
        else:
            pg.train_step_grads(self.params[0], self.params[1], self.params[2], d["xy_colloc"], d["f"], d["xy_sensors"], d["z"], d["real"],
                                d["eps"], self.loss_scale, out=self.out)
            grads = self.out[:3]
        if getattr(self, "dp_dist", None) is not None:
            self.dp_out.all_reduce_mean(self.dp_dist, self.dp_world)
        for k in range(len(self.params)):
            pg.adam_update(self.params[k], grads[k], self.mom[k][0], self.mom[k][1], self.step_no, skip_flag=self.out[4], **ADAM)

    def enable_dp(self, dist):
        """NEXT-4: this rank's context holds N / W samples; the three gradient vectors live in ONE flat buffer that is
        all-reduced (NCCL) right behind the step, then every rank applies the same Adam update."""
        from paper_1910_13444_b200.dp import FlatGrads
        self.dp_dist, self.dp_world = dist, dist.get_world_size()
        self.dp_out = FlatGrads([p.numel() for p in self.params], self.device)
        if self.trunk:
            self.out = (self.dp_out.grads[0], None, self.dp_out.grads[1], self.dp_out.losses, self.dp_out.found_inf)
        else:
            self.out = (self.dp_out.grads[0], self.dp_out.grads[1], self.dp_out.grads[2], self.dp_out.losses, self.dp_out.found_inf)

    def step_e2e(self):
        """Same step with the per-step inputs coming from pinned host memory and the losses read back."""
        d = self.d
        for k in ("z", "real", "eps"):
            d[k].copy_(self.host[k], non_blocking=True)
        self.step()
        self.host_out.copy_(self.out[3], non_blocking=True)
        self.torch.cuda.current_stream(self.device).synchronize()   # the host holds this step's losses before the next step is issued

    def jet_pass(self):
        """The jet evaluation alone (a1-a4 forward): G_u at order 2 and G_logk at order 1 on every (sample, point)."""
        d, pg = self.d, self.pg
        if not hasattr(self, "jet_out"):
            n = self.cfg.N * self.cfg.P
            self.jet_out = (self.torch.empty(5 * n, device=self.device), self.torch.empty(3 * n, device=self.device))
            self.jet_out2 = self.torch.empty(2, 5, self.cfg.N, self.cfg.P, device=self.device) if self.trunk else None
        if self.trunk:
            pg.trunk_jet_forward(self.params[0], d["xy_colloc"], d["z"], 2, out=self.jet_out2)
            return
        pg.gen_jet_forward(self.params[1], d["xy_colloc"], d["z"], 2, out=self.jet_out[0].view(5, self.cfg.N, self.cfg.P))
        pg.gen_jet_forward(self.params[0], d["xy_colloc"], d["z"], 1, out=self.jet_out[1].view(3, self.cfg.N, self.cfg.P))

    def e2e_bytes(self):
        return sum(int(v.numel() * 4) for v in self.host.values()), 6 * 4

    def timed(self, fn, steps, warmup, tag="timed_step"):
        """Per-step CUDA-event timing on the launch stream; L2 is flushed between steps for the small configs.  Every timed call
        sits in an NVTX range `tag` (ncu --nvtx --nvtx-include "timed_step/" profiles exactly the timed train steps)."""
        torch = self.torch
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize(self.device)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in ev:
            if self.flush is not None:
                self.flush.fill_(1)
            a.record()
            torch.cuda.nvtx.range_push(tag)
            fn()
            torch.cuda.nvtx.range_pop()
            b.record()
        torch.cuda.synchronize(self.device)
        return [a.elapsed_time(b) for a, b in ev]


def run_config(cfg, device, steps, warmup, rank, world, with_roofline=True, seed_shift=0, chunk_rows=0, dp=None):
    import torch
    w = GpuWorkload(cfg, device, seed_shift, chunk_rows)
    if dp is not None:
        w.enable_dp(dp)
    peaks = measured_peaks()
    flops = wl.step_flops(cfg)
    res = {}
    sampler = ClockSampler(index=torch.cuda.current_device()); sampler.start()
    # Large configs (seconds of tensor-core work per step): per-launch CUDA events are recorded INSIDE the timed region, so
    # the roofline durations and `value` come from the same steps (the library runs eagerly while profiling).  Small
    # configs are launch-latency bound: their timed region replays the step's CUDA graph (what a user gets), and the
    # per-kernel durations come from a separate eager pass right after it.
    in_region = cfg.N * cfg.P > 1000000
    for _ in range(warmup):
        w.step()
    torch.cuda.synchronize(device)
    if in_region:
        w.pg.profile_enable(True)
    l0 = w.pg.launch_count
    ms = w.timed(w.step, steps, 0)
    launches = w.pg.launch_count - l0
    if not in_region:
        w.pg.profile_enable(True)
        for _ in range(steps):
            w.step()
    prof = w.pg.profile_report()
    w.pg.profile_enable(False)
    res["clocks"] = sampler.finish()
    res["ms_steps"] = ms
    res["launches"] = launches
    res["found_inf"] = int(w.out[4].item())
    res["losses"] = [float(x) for x in w.out[3].cpu()]
    # end-to-end leg: host buffers in, losses out, copies inside the timed region
    ms_e2e = w.timed(w.step_e2e, max(2, steps // 2), 1, tag="timed_e2e")
    res["ms_e2e"] = ms_e2e
    res["h2d"], res["d2h"] = w.e2e_bytes()
    # jet evaluations/s (north_star's second throughput figure): forward jets of both nets, no residual, no backward
    res["ms_jet"] = w.timed(w.jet_pass, max(2, steps // 2), 1, tag="timed_jet")
    del w.jet_out, w.jet_out2
    # roofline of the dominant kernel class (the tcgen05 jet GEMMs: forward, dgrad+adjoint, wgrad)
    if with_roofline:
        tc = {k: v for k, v in prof.items() if k in ("jet_layer_fwd", "jet_layer_bwd", "wgrad", "jet_layer_bwd_wgrad", "gen_fwd_fused")}
        per_step = {k: [v[0] / steps, v[1] / steps] for k, v in prof.items()}
        tc_ms = sum(v[1] for v in tc.values()) / steps
        total_ms = sum(v[1] for v in prof.values()) / steps
        res["kernel_ms_per_step"] = {k: round(v[1], 4) for k, v in sorted(per_step.items(), key=lambda kv: -kv[1][1])}
        res["kernel_launches_per_step"] = {k: v[0] for k, v in per_step.items()}
        if tc_ms > 0:
            # algorithmic flops of the hidden jet layers of the collocation + sensor rows: 3 GEMMs (fwd, dgrad, wgrad) per layer
            sens_gemm = cfg.N * 3 * cfg.S * (2 if cfg.variant == "two_mlps" else 1) * (cfg.L - 1) * 2 * cfg.H * cfg.H
            alg = flops["jet_gemm"] + sens_gemm
            ach = alg / (tc_ms * 1e-3) / 1e12
            peak = peaks["tflops_sustained"]
            # per kernel class: its own roofline = max(flops / sustained tensor rate, algorithmic plane bytes / copy bandwidth).
            # plane bytes per row and hidden layer (16-bit): forward reads C + writes C planes, dgrad reads 2C (ahat^l, h^{l-1}) + writes C
            # (nothing for the fused layer-2 dgrad), wgrad reads 2C; C summed over the nets' collocation channels, sensors add 1 (2 split) per net
            chan = 8 if cfg.variant == "two_mlps" else 5
            nets = 2 if cfg.variant == "two_mlps" else 1
            rowsC = cfg.N * cfg.P * chan + cfg.N * cfg.S * nets
            pb = 2 * cfg.H                                        # bytes of one row of one 16-bit plane
            Lh = cfg.L - 1
            # width 256: dgrad and wgrad of a layer are ONE kernel (jet_layer_bwd_wgrad): two of the three GEMMs, planes read once
            # width 128: the whole forward of the collocation rows is ONE kernel (gen_fwd_fused): it writes h^1 .. h^L and reads no planes
            # Each class is credited the rows it actually processes: where the fused forward exists it does the collocation rows and
            # the layer-by-layer forward (jet_layer_fwd) only the sensor rows; every other class sees both.
            col, sen = flops["jet_gemm"] / 3, sens_gemm / 3      # one GEMM type (fwd, dgrad or wgrad) over the collocation / sensor rows
            fwd_rows_sens_only = "gen_fwd_fused" in tc
            rowsS = cfg.N * cfg.S * nets
            cls_bytes = {"jet_layer_fwd": 2 * (rowsS if fwd_rows_sens_only else rowsC) * pb * Lh, "jet_layer_bwd": rowsC * pb * (3 * Lh - 1),
                         "wgrad": 2 * rowsC * pb * Lh, "jet_layer_bwd_wgrad": rowsC * pb * (3 * Lh - 1), "gen_fwd_fused": cfg.N * cfg.P * chan * pb * cfg.L}
            cls_flops = {"jet_layer_fwd": sen if fwd_rows_sens_only else col + sen, "jet_layer_bwd": col + sen, "wgrad": col + sen,
                         "jet_layer_bwd_wgrad": 2 * (col + sen), "gen_fwd_fused": col}
            prof_ncu, prof_src, prof_stale = ncu_profile(cfg.name)
            per_kernel = {}
            for k, v in tc.items():
                if v[1] <= 0:
                    continue
                t_ms = v[1] / steps
                alg_k = cls_flops[k]
                t_tensor = alg_k / (peak * 1e12) * 1e3
                t_hbm = cls_bytes[k] / (peaks["hbm_gbs"] * 1e9) * 1e3
                pct = [d["tensor_pct"] for kk, d in prof_ncu.items() if kk.startswith(k + "(C=5") or kk == k]
                per_kernel[k] = {"tflops": round(alg_k / (t_ms * 1e-3) / 1e12, 1), "gbs_algorithmic": round(cls_bytes[k] / (t_ms * 1e-3) / 1e9, 1),
                                 "bound": "tensor" if t_tensor >= t_hbm else "hbm", "frac": round(max(t_tensor, t_hbm) / t_ms, 4),
                                 "tensor_pipe_active_pct_ncu": pct[0] if pct else None}
            dom = max(tc, key=lambda k: tc[k][1])
            dom_ncu = next((d for kk, d in prof_ncu.items() if kk.startswith(dom + "(C=5") or kk == dom), None)
            whole = prof_ncu.get("WHOLE_STEP")
            res["roofline"] = {"bound": "tensor", "achieved": round(ach, 2), "peak": peak, "unit": "TFLOP/s", "frac": round(ach / peak, 4),
                               "traffic": (dom_ncu["dram_bytes"] / dom_ncu["launches"]) if dom_ncu else None,
                               "traffic_kernel": f"{dom} (C=5), DRAM read+write bytes per launch" if dom_ncu else None,
                               "traffic_whole_step": whole["dram_bytes"] if whole else None,
                               "traffic_source": f"{prof_src} (an ncu pass recorded under profiles/, not this run)" if prof_ncu else None,
                               "traffic_stale": prof_stale,      # true: the library sources changed since that pass (or it carries no source hash)
                               "kernel": " + ".join(sorted(tc)) + " (tcgen05)", "peak_source": peaks["source"] + " sustained bf16",
                               "frac_of_burst": round(ach / peaks["tflops_burst"], 4), "frac_of_nominal_2250": round(ach / 2250.0, 4),
                               "share_of_step": round(tc_ms / total_ms, 4) if total_ms > 0 else None,
                               "profile_pass": ("in the timed region: one CUDA event is recorded after every launch inside the timed steps, so `value` carries that "
                                                "(~1 %) overhead") if in_region else "separate eager pass after the timed region (the timed region replays a CUDA graph)",
                               "per_kernel": per_kernel,
                               "per_kernel_frac_le_1": all(v["frac"] <= 1.0 for v in per_kernel.values())}
        else:
            # fp32 mode (c1): plain FP32 FMA path; report against the fp32 ALU peak (148 SMs x 128 lanes x 2 flop x clock)
            mhz = res["clocks"]["sm_mhz"] or 1965.0
            peak = 148 * 128 * 2 * mhz * 1e6 / 1e12
            ach = flops["total"] / (np.mean(ms) * 1e-3) / 1e12
            res["roofline"] = {"bound": "alu", "achieved": round(ach, 4), "peak": round(peak, 1), "unit": "TFLOP/s", "frac": round(ach / peak, 5),
                               "traffic": None, "kernel": "whole fp32 step (launch-latency bound at this size)"}
    # whole step against its roofline: t_roof = sum over kernel classes of max(flops / tensor peak, bytes / HBM peak)
    if with_roofline and prof:
        hb = hbm_class_bytes(cfg)
        t_roof = 0.0
        if cfg.precision != "fp32":
            sens_gemm = cfg.N * 3 * cfg.S * (2 if cfg.variant == "two_mlps" else 1) * (cfg.L - 1) * 2 * cfg.H * cfg.H
            t_roof += (flops["jet_gemm"] + sens_gemm) / (peaks["tflops_sustained"] * 1e12) * 1e3
        hk = {}
        for k, b in hb.items():
            if k in prof and prof[k][1] > 0:
                ms_k = prof[k][1] / steps
                t_roof += b / (peaks["hbm_gbs"] * 1e9) * 1e3
                hk[k] = {"gbs": round(b / (ms_k * 1e-3) / 1e9, 1), "frac": round(b / (ms_k * 1e-3) / 1e9 / peaks["hbm_gbs"], 3), "ms": round(ms_k, 4)}
        res["step_roofline"] = {"t_roof_ms": round(t_roof, 4), "frac": round(t_roof / float(np.mean(ms)), 4), "hbm_peak_gbs": peaks["hbm_gbs"],
                                "hbm_kernels": hk, "note": "tensor classes at the measured sustained bf16 rate + HBM-bound classes at the measured copy bandwidth; "
                                "critic, z-part and launch latency count as zero in t_roof"}
    w.pg.close()
    return res


def run_next_rows(device, steps=10, warmup=3):
    """NEXT-2 and NEXT-3 timed on c2's networks: the step with f at per-sample free sensors fed to the critic,
    and the step with a two-level hierarchy of 20 critics.  Device-resident inputs, CUDA events, eager launches."""
    import torch
    from paper_1910_13444_b200 import PiGan
    cfg = wl.CONFIGS["c2"]
    out = {}
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(device)

    def timed(fn):
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize(device)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in ev:
            a.record(); fn(); b.record()
        torch.cuda.synchronize(device)
        return float(np.mean([a.elapsed_time(b) for a, b in ev]))

    inp = wl.make_inputs(cfg)
    # NEXT-2: F = 2000 free sensors per sample (the paper's count for the top-level subdomain), critic input 2S + 3F
    F = 2000
    d_in = 2 * cfg.S + 3 * F
    thD = wl.round_to_precision(wl.xavier_params(np.random.default_rng(2002), d_in, cfg.LD, cfg.HD), cfg.precision)
    xy_free = wl.free_sensor_points(cfg, F)
    real = np.random.default_rng(2003).normal(size=(cfg.N, d_in)).astype(np.float32)
    real[:, 2 * cfg.S:2 * cfg.S + F] = 0.0
    pg = PiGan(latent_dim=cfg.m, gen_hidden=cfg.L, gen_width=cfg.H, disc_hidden=cfg.LD, disc_width=cfg.HD, n_samples=cfg.N, n_colloc=F,
               n_sensors=cfg.S, precision=cfg.precision, pde_weight=0.0, n_free=F, device=device)
    a = [t(inp["theta_Y"]), t(inp["theta_u"]), t(thD), t(xy_free), t(inp["xy_sensors"]), t(inp["z"]), t(real), t(inp["eps"])]
    o = pg.train_step_grads(a[0], a[1], a[2], a[3], None, a[4], a[5], a[6], a[7], 1.0)
    ms = timed(lambda: pg.train_step_grads(a[0], a[1], a[2], a[3], None, a[4], a[5], a[6], a[7], 1.0, out=o))
    out["next2_free_sensors"] = {"workload": f"c2 networks, {cfg.N} samples x {F} free sensors each, critic input {d_in}", "ms_per_step": ms,
                                 "value": cfg.N * F / (ms * 1e-3), "unit": "sample*free-sensor-points/s", "found_inf": int(o[4].item())}
    pg.close()
    # NEXT-3: levels of 1 and 19 subdomains, 10 sensors per critic
    levels, per = [1, 19], 10
    K = sum(levels)
    rng = np.random.default_rng(2004)
    sens = np.stack([np.sort(rng.choice(cfg.S, size=per, replace=False)) for _ in range(K)])
    subsets = np.concatenate([sens, cfg.S + sens], axis=1).astype(np.int32)
    thDs = np.stack([wl.round_to_precision(wl.xavier_params(np.random.default_rng(2100 + k), 2 * per, cfg.LD, cfg.HD), cfg.precision) for k in range(K)])
    w = np.concatenate([np.full(n, 1.0 / (len(levels) * n)) for n in levels])
    real = np.random.default_rng(2005).normal(size=(cfg.N, 2 * cfg.S)).astype(np.float32)
    pg = PiGan.from_config(cfg, n_critics=K, critic_inputs=2 * per, device=device)
    a = [t(inp["theta_Y"]), t(inp["theta_u"]), t(thDs), t(subsets), t(inp["xy_colloc"]), t(inp["f"]), t(inp["xy_sensors"]), t(inp["z"]), t(real), t(inp["eps"])]
    ms = timed(lambda: pg.train_step_grads_hier(a[0], a[1], a[2], a[3], w, a[4], a[5], a[6], a[7], a[8], a[9], 1.0))
    out["next3_hierarchical_critics"] = {"workload": f"c2, {K} critics in levels {levels}, {per} sensors each", "ms_per_step": ms,
                                         "value": cfg.N * cfg.P / (ms * 1e-3), "unit": UNIT}
    pg.close()
    return out


def summarize(cfg, res, n_gpus, steps, warmup, t_max_ms):
    units = cfg.N * cfg.P
    value = whole_job_value(units, n_gpus, t_max_ms)
    e2e_ms = float(np.mean(res["ms_e2e"]))
    return {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": n_gpus, "steps": steps, "warmup": warmup, "ms_per_step": t_max_ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        # the arithmetic type of the tensor-core operands: both 16-bit modes compute with fp16 operands and fp32 accumulation (R1)
        "dtype": "fp32" if cfg.precision == "fp32" else "fp16", "precision_mode": cfg.precision, "data": "synthetic",
        "config": {"workload": f"{cfg.name}: {cfg.L}x{cfg.H} tanh generators (m={cfg.m}), {cfg.G}x{cfg.G} grid x {cfg.N} samples, {cfg.S} sensors, "
                               f"critic {cfg.LD}x{cfg.HD}", "rows_per_step": units, "parallelism": f"replicas x{n_gpus}" if n_gpus > 1 else "single GPU",
                   "l2": "per-step working set >> L2" if cfg.N * cfg.P >= 400000 else "256 MiB L2 flush between timed steps",
                   "loss_scale": 1024.0 if cfg.precision == "fp16" else 1.0},
        "train_steps_per_s": 1e3 / t_max_ms,
        "jet_evals_per_s": n_gpus * units / (float(np.mean(res["ms_jet"])) * 1e-3),
        "step_tflops": wl.step_flops(cfg)["total"] / (t_max_ms * 1e-3) / 1e12,
        "e2e": {"value": n_gpus * units / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": res["h2d"], "d2h_bytes_per_step": res["d2h"]},
        "gpu_launches": res["launches"], "clocks": res["clocks"], "roofline": res.get("roofline"), "step_roofline": res.get("step_roofline"),
        "kernel_ms_per_step": res.get("kernel_ms_per_step"), "losses": res["losses"], "found_inf": res["found_inf"],
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="c5", choices=list(wl.CONFIGS) + ["t2"],
                    help="c1..c5 = BASELINE.json configs; t2 = the paper's Table II generator-worker workload on its own 21x1024 shared-trunk generator (NEXT-1)")
    ap.add_argument("--impl", default="pigan", choices=["pigan", "reference"])
    ap.add_argument("--all-configs", action="store_true", default=True, help="also run the other configs briefly and attach them as per_config (default)")
    ap.add_argument("--headline-only", dest="all_configs", action="store_false", help="time only --config")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--samples", type=int, default=None, help="override N (latent samples per step): a smaller job for ncu captures; "
                    "the line then says so in config.workload and is not a benchmark value")
    ap.add_argument("--dp", action="store_true", help="NEXT-4: with --gpus N > 1, shard the N latent samples of the step over the ranks and all-reduce "
                    "the gradients (strong scaling) instead of running N independent replicas")
    ap.add_argument("--chunk-rows", type=int, default=0, help="rows per chunk of the generator passes (0 = library default); sweeps only")
    ap.add_argument("--ncu-summary", default=None, metavar="CSV", help="no benchmark: sum the per-launch ncu CSV of one timed step of --config per kernel "
                    "class and print the rows of profiles/rNN_step_dram_bytes.csv (needs no GPU)")
    args = ap.parse_args()
    if args.ncu_summary:
        ncu_summary(args.ncu_summary, args.config)
        return 0
    cfg = wl.TABLE2 if args.config == "t2" else wl.CONFIGS[args.config]
    if args.samples:
        args.all_configs = False
        cfg = dataclasses.replace(cfg, name=f"{cfg.name}[N={args.samples} profiling subset]", N=args.samples)
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    warmup = max(3, args.warmup) if args.impl == "pigan" else args.warmup
    steps = args.steps if args.steps is not None else (5 if cfg.N * cfg.P > 1000000 else 20)

    if args.impl == "reference":
        # the oracle, as it stands, on the host cores; rank 0 alone works
        if rank != 0:
            return 0
        val, sec, cores, sample = time_oracle(cfg, steps=max(1, min(steps, 3)), warmup=min(args.warmup, 1))
        line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": max(1, min(steps, 3)),
                "warmup": min(args.warmup, 1), "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic", "config": {"workload": f"{cfg.name} (bounded sample: {sample})"},
                "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
                "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
        print(json.dumps(line))
        return 0

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl pigan needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    device = torch.device(f"cuda:{local_rank}")
    if world > 1:
        dist.init_process_group("nccl", device_id=device)
        dist.barrier()
    units_global = cfg.N * cfg.P
    if args.dp and world > 1:
        if cfg.N % world:
            raise SystemExit(f"--dp needs N = {cfg.N} divisible by the world size {world}")
        cfg = dataclasses.replace(cfg, N=cfg.N // world)      # this rank's shard; inputs are drawn per rank (seed_shift)
    res = run_config(cfg, device, steps, warmup, rank, world, seed_shift=rank, chunk_rows=args.chunk_rows, dp=dist if (args.dp and world > 1) else None)
    t_ms = float(np.mean(res["ms_steps"]))
    if world > 1:
        t_ms = max_over_ranks(t_ms, dist, device)           # max over ranks; the replicas exchange nothing else
    if rank == 0:
        line = summarize(cfg, res, world, steps, warmup, t_ms)
        if args.dp and world > 1:
            line["scaling"] = "strong"
            line["config"]["parallelism"] = f"data-parallel x{world}: {cfg.N} of {cfg.N * world} samples per rank, one fp32 all-reduce of the gradients per step"
            line["config"]["rows_per_step"] = units_global
        if args.all_configs:
            per = {}
            for name, c in wl.CONFIGS.items():
                if name == cfg.name:
                    continue
                r = run_config(c, device, 5 if c.N * c.P > 1000000 else 20, 3, rank, world)
                s = summarize(c, r, 1, len(r["ms_steps"]), 3, float(np.mean(r["ms_steps"])))
                per[name] = {k: s[k] for k in ("value", "ms_per_step", "dtype", "step_tflops", "jet_evals_per_s", "roofline", "step_roofline", "gpu_launches", "e2e", "kernel_ms_per_step")}
            # NEXT-1: the paper's Table II workload on its own generator (21 x 1024 shared trunk with skips)
            r = run_config(wl.TABLE2, device, 20, 3, rank, world)
            s2 = summarize(wl.TABLE2, r, 1, len(r["ms_steps"]), 3, float(np.mean(r["ms_steps"])))
            per["t2"] = {k: s2[k] for k in ("value", "ms_per_step", "dtype", "step_tflops", "jet_evals_per_s", "roofline", "step_roofline", "gpu_launches", "e2e", "kernel_ms_per_step")}
            per["t2"]["paper_table2"] = {"flop_per_step_paper": 12.3e12, "flop_per_step_8_channel_model": 6 * (2000 * 8 + 200) * 20 * 2 * 1024 * 1024 * 3,
                                         "flop_per_step_this_build": wl.step_flops(wl.TABLE2)["total"], "paper_step_s_v100": 12.3e12 / 38.6e12,
                                         "note": "the shared trunk needs 5 jet channel passes where the paper's TF autodiff graph counts 8; 2025 grid points stand in for the 2000 f sensors"}
            per.update(run_next_rows(device))
            line["per_config"] = per
        if not args.no_cpu_baseline:
            val, sec, cores, sample = time_oracle(cfg)
            line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "seconds": sec}
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
