"""NEXT-4: data-parallel training step and a minimal loop with the paper's sequential and
parallel schedules.

The path shards naturally: (sample, point) rows are independent and every loss is a MEAN over the latent samples, so with
the N samples of a step split evenly over W ranks the global gradient is the mean of the ranks' gradients ("the
gradient ... is the sum of the gradients of the local batches").  Each rank runs pigan_train_step_grads on its N / W samples
with its three gradient vectors laid out in ONE flat fp32 buffer, so the exchange is ONE all-reduce per step (NCCL over
NVLink / NVSwitch on GPUs; c5: 34.2 M floats = 137 MB, ~0.3 ms against a ~1 s step), issued on the step's stream right behind
the last weight-gradient chunk; then every rank applies the identical Adam update.

Schedules (Fig. 4):
  parallel    generator and critic gradients are both taken at the SAME current weights (what one pigan_train_step_grads call
              returns), then all networks are updated: one step call per iteration.
  sequential  the critic is updated first, the generator's gradient is then taken against the UPDATED critic: two step
              calls per iteration (the critic half of the first, the generator half of the second).

Only plumbing lives here (sharding, the flat buffer, torch.distributed, the update order); every gradient comes from the
CUDA library.  `step_fn` / `adam_fn` are injectable so that the host logic can be exercised on CPU ranks (gloo) in the tests.
"""
from __future__ import annotations

from typing import Callable, Sequence

import torch

__all__ = ["shard_bounds", "FlatGrads", "DataParallelTrainer"]


def shard_bounds(n_samples: int, world: int, rank: int) -> tuple[int, int]:
    """Rows [lo, hi) of the global batch that `rank` owns.  The means only commute with the all-reduce for EQUAL shards."""
    if n_samples % world != 0:
        raise ValueError(f"n_samples = {n_samples} is not divisible by the world size {world}")
    per = n_samples // world
    return rank * per, (rank + 1) * per


class FlatGrads:
    """The gradient vectors of one step as views of ONE flat fp32 buffer [g_0 | g_1 | ... | losses(6) | found_inf], every
    view 16-byte aligned (the library's requirement), so that a single all-reduce covers them all."""

    def __init__(self, sizes: Sequence[int], device):
        self.sizes = list(sizes)
        offs, off = [], 0
        for n in self.sizes + [6, 1]:
            offs.append(off)
            off += (n + 3) // 4 * 4
        self.flat = torch.zeros(off, dtype=torch.float32, device=device)
        self.grads = [self.flat[o:o + n] for o, n in zip(offs[:len(self.sizes)], self.sizes)]
        self.losses = self.flat[offs[-2]:offs[-2] + 6]
        self.flag = self.flat[offs[-1]:offs[-1] + 1]          # found_inf as a float, so that it rides in the same all-reduce
        self.found_inf = torch.zeros(1, dtype=torch.int32, device=device)

    def all_reduce_mean(self, dist, world: int):
        """Sum over ranks, then 1/W: gradients and losses become the global means; flag > 0 iff any rank overflowed.

        Stream order: the library's step -- eager launches or the replay of its CUDA graph -- is enqueued on
        the context's stream, which is torch's current stream of the device (PiGan takes it at creation).  torch.distributed's
        collective waits on an event recorded on torch's current stream before it starts on the backend's own stream, and the
        synchronous form used here makes the current stream wait for its completion; the library's private capture stream and
        side streams are joined back into the context's stream before a step call returns.  So the collective reads finished
        gradients and Adam reads reduced ones, as long as the caller keeps ONE current stream around step, collective and update.
        The collective is issued whenever a process group exists (also for a single rank: that keeps the one-rank path identical
        to the many-rank path, and lets a one-GPU box execute it)."""
        self.flag.copy_(self.found_inf.to(torch.float32))
        if dist is not None:
            dist.all_reduce(self.flat, op=dist.ReduceOp.SUM)
        if world > 1:
            self.flat.mul_(1.0 / world)
        self.found_inf.copy_((self.flag > 0).to(torch.int32))


class DataParallelTrainer:
    """step_fn(params, z, real, eps, out) fills out.grads / out.losses / out.found_inf with the LOCAL shard's step;
    adam_fn(param, grad, m, v, step_no, skip_flag) updates in place.  params: list of flat fp32 tensors, the critic last."""

    def __init__(self, step_fn: Callable, adam_fn: Callable, params: Sequence[torch.Tensor], schedule: str = "parallel", dist=None):
        if schedule not in ("parallel", "sequential"):
            raise ValueError("schedule must be 'parallel' or 'sequential' (P:179)")
        self.step_fn, self.adam_fn, self.schedule = step_fn, adam_fn, schedule
        self.dist = dist if (dist is not None and dist.is_available() and dist.is_initialized()) else None
        self.world = self.dist.get_world_size() if self.dist else 1
        self.rank = self.dist.get_rank() if self.dist else 0
        self.params = list(params)
        dev = self.params[0].device
        self.out = FlatGrads([p.numel() for p in self.params], dev)
        self.mom = [(torch.zeros_like(p), torch.zeros_like(p)) for p in self.params]
        # Adam step counters.  They count ATTEMPTED updates: found_inf lives on the device and reading it back every step would
        # serialise host and GPU, so a step that pigan_adam_update skips (overflow) still advances t.  Parameters and moments
        # stay bit-identical on a skipped step; only the bias correction 1 - beta^t runs one step ahead per skipped step,
        # which vanishes as t grows (with beta2 = 0.9: below 1e-4 after ~90 steps).
        self.t = [0] * len(self.params)
        self.step_calls = 0

    def _grads(self, z, real, eps):
        self.step_fn(self.params, z, real, eps, self.out)
        self.step_calls += 1
        self.out.all_reduce_mean(self.dist, self.world)

    def _update(self, which):
        for k in which:
            self.t[k] += 1
            self.adam_fn(self.params[k], self.out.grads[k], self.mom[k][0], self.mom[k][1], self.t[k], self.out.found_inf)

    def train_step(self, z, real, eps):
        """One iteration on this rank's shard (z [N/W][m], real [N/W][d], eps [N/W]).  Returns the global-mean losses (a view)."""
        gen, critic = list(range(len(self.params) - 1)), [len(self.params) - 1]
        if self.schedule == "parallel":
            self._grads(z, real, eps)
            self._update(critic + gen)
        else:
            self._grads(z, real, eps)
            self._update(critic)                                # critic first ...
            self._grads(z, real, eps)
            self._update(gen)                                   # ... then the generator against the updated critic
        return self.out.losses


def pigan_step_fns(pg, xy_colloc, f, xy_sensors, loss_scale=1.0, adam=None):
    """(step_fn, adam_fn) that drive a PiGan context (two-MLP generator): the product path of DataParallelTrainer."""
    adam = adam or dict(lr=1e-4, beta1=0.5, beta2=0.9, adam_eps=1e-8)

    def step_fn(params, z, real, eps, out):
        pg.train_step_grads(params[0], params[1], params[2], xy_colloc, f, xy_sensors, z, real, eps, loss_scale,
                            out=(out.grads[0], out.grads[1], out.grads[2], out.losses, out.found_inf))

    def adam_fn(p, g, m, v, t, skip):
        pg.adam_update(p, g, m, v, t, skip_flag=skip, **adam)

    return step_fn, adam_fn
