"""NEXT-4: host logic of the data-parallel step (paper_1910_13444_b200/dp.py) on CPU ranks: world_size-2 gloo processes with
the fp64 oracle standing in for the CUDA library (tests may use oracle/).  Checks that the sharded, all-reduced gradients are
the full-batch gradients, and that the two schedules of P:179 update in the stated order."""
import os
import sys

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _problem():
    import workloads as wl
    cfg = wl.Config("dp", 7, "fp32", m=3, L=2, H=6, G=3, N=4, S=3, LD=2, HD=5)
    inp = wl.make_inputs(cfg, bias_std=0.2)
    rng = np.random.default_rng(77)
    inp["real"] = rng.normal(size=(cfg.N, 2 * cfg.S)).astype(np.float32)
    return cfg, inp


def _oracle_fns(cfg, inp, lr=1e-2):
    from oracle import pigan_oracle as orc

    def step_fn(params, z, real, eps, out):
        gY, gu, gD, losses = orc.train_step_grads_ref(cfg.gen_shape, cfg.disc_shape, params[0].numpy(), params[1].numpy(), params[2].numpy(),
                                                      inp["xy_colloc"], inp["f"], inp["xy_sensors"], z.numpy(), real.numpy(), eps.numpy(), 10.0, 1.0)
        for dst, src in zip(out.grads, (gY, gu, gD)):
            dst.copy_(torch.from_numpy(src).float())
        out.losses.copy_(torch.from_numpy(losses).float())
        out.found_inf.zero_()

    def adam_fn(p, g, m, v, t, skip):
        if int(skip.item()):
            return
        th, mm, vv = orc.adam_update_ref(p.numpy(), g.numpy(), m.numpy(), v.numpy(), t, lr, 0.5, 0.9, 1e-8)
        p.copy_(torch.from_numpy(th).float()); m.copy_(torch.from_numpy(mm).float()); v.copy_(torch.from_numpy(vv).float())

    return step_fn, adam_fn


def _worker(rank, world, port, schedule, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1910_13444_b200.dp import DataParallelTrainer, shard_bounds
    cfg, inp = _problem()
    step_fn, adam_fn = _oracle_fns(cfg, inp)
    params = [torch.from_numpy(inp[k].copy()) for k in ("theta_Y", "theta_u", "theta_D")]
    tr = DataParallelTrainer(step_fn, adam_fn, params, schedule=schedule, dist=dist)
    lo, hi = shard_bounds(cfg.N, world, rank)
    t = lambda k: torch.from_numpy(np.ascontiguousarray(inp[k][lo:hi]))
    losses = tr.train_step(t("z"), t("real"), t("eps")).clone()
    q.put((rank, [g.clone().numpy() for g in tr.out.grads], losses.numpy(), [p.numpy().copy() for p in tr.params], tr.step_calls))
    dist.barrier()
    dist.destroy_process_group()


def _run_world(schedule, world=2):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29600 + (os.getpid() % 200) + (0 if schedule == "parallel" else 1)
    procs = [ctx.Process(target=_worker, args=(r, world, port, schedule, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=120) for _ in range(world)], key=lambda x: x[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    return res


def _single(schedule):
    from paper_1910_13444_b200.dp import DataParallelTrainer
    cfg, inp = _problem()
    step_fn, adam_fn = _oracle_fns(cfg, inp)
    params = [torch.from_numpy(inp[k].copy()) for k in ("theta_Y", "theta_u", "theta_D")]
    tr = DataParallelTrainer(step_fn, adam_fn, params, schedule=schedule)
    t = lambda k: torch.from_numpy(np.ascontiguousarray(inp[k]))
    losses = tr.train_step(t("z"), t("real"), t("eps")).clone()
    return [g.clone().numpy() for g in tr.out.grads], losses.numpy(), [p.numpy().copy() for p in tr.params], tr.step_calls


@pytest.mark.parametrize("schedule", ["parallel", "sequential"])
def test_two_ranks_reproduce_the_full_batch_step(schedule):
    g1, l1, p1, calls1 = _single(schedule)
    res = _run_world(schedule)
    for rank, g2, l2, p2, calls2 in res:
        assert calls2 == calls1 == (1 if schedule == "parallel" else 2)
        for a, b in zip(g1, g2):
            assert np.allclose(a, b, rtol=2e-5, atol=1e-7), (schedule, rank)            # mean of the shard means = the full-batch mean
        assert np.allclose(l1, l2, rtol=2e-5, atol=1e-7)
        for a, b in zip(p1, p2):
            assert np.allclose(a, b, rtol=1e-5, atol=1e-7)                               # identical updates on every rank
    assert all(np.array_equal(res[0][3][k], res[1][3][k]) for k in range(3))


def test_sequential_schedule_takes_the_generator_gradient_against_the_updated_critic():
    from oracle import pigan_oracle as orc
    cfg, inp = _problem()
    gpar, _, ppar, _ = _single("parallel")
    gseq, _, pseq, _ = _single("sequential")
    # by hand: critic step first, then the generator gradient at the new critic
    a = [inp[k].astype(np.float64) for k in ("theta_Y", "theta_u", "theta_D")]
    args = (inp["xy_colloc"], inp["f"], inp["xy_sensors"], inp["z"], inp["real"], inp["eps"], 10.0, 1.0)
    _, _, gD, _ = orc.train_step_grads_ref(cfg.gen_shape, cfg.disc_shape, a[0], a[1], a[2], *args)
    thD, _, _ = orc.adam_update_ref(a[2], gD, np.zeros_like(gD), np.zeros_like(gD), 1, 1e-2, 0.5, 0.9, 1e-8)
    gY, gu, _, _ = orc.train_step_grads_ref(cfg.gen_shape, cfg.disc_shape, a[0], a[1], thD.astype(np.float32), *args)
    assert np.allclose(gseq[0], gY, rtol=1e-4, atol=1e-7) and np.allclose(gseq[1], gu, rtol=1e-4, atol=1e-7)
    assert np.allclose(pseq[2], ppar[2], rtol=1e-6)                                       # the critic update is the same in both schedules
    assert np.abs(gseq[0] - gpar[0]).max() > 1e-6                                         # and the generator gradients do differ


def test_shard_bounds_and_flat_buffer_layout():
    from paper_1910_13444_b200.dp import FlatGrads, shard_bounds
    assert [shard_bounds(8, 4, r) for r in range(4)] == [(0, 2), (2, 4), (4, 6), (6, 8)]
    with pytest.raises(ValueError):
        shard_bounds(6, 4, 0)
    fg = FlatGrads([2369, 2369, 2817], "cpu")
    for v in fg.grads + [fg.losses, fg.flag]:
        assert v.data_ptr() % 16 == 0 and v.is_contiguous()
    assert fg.flat.numel() >= 2369 * 2 + 2817 + 7
