"""Host-side logic of bench.py that needs no GPU: the multi-GPU mode is "replicas only", so the
N > 1 path is the max-over-ranks reduction of the step time, the whole-job throughput formula and the launch contract
(rank 0 alone prints one JSON line).  Covered here with world_size-2 gloo process groups on the CPU."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    t_local = 10.0 + 5.0 * rank                       # rank 1 is the slow replica
    t = bench.max_over_ranks(t_local, dist, None)
    q.put((rank, t, bench.whole_job_value(1000, world, t)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # every rank sees the slowest rank's time; value = units of ALL ranks / that time
    assert [g[1] for g in got] == [15.0, 15.0]
    assert got[0][2] == pytest.approx(2 * 1000 / 15e-3)


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.whole_job_value(4194304, 1, 1000.0) == pytest.approx(4194304.0)


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    """`bench.py --impl reference` under torchrun with 2 ranks: rank 0 times the oracle on the host and prints the one
    JSON line, rank 1 exits 0 without work (config c1 is small enough for the oracle to finish in a second)."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--config", "c1",
           "--steps", "1", "--warmup", "0"]
    out = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["value"] > 0 and d["unit"] == "sample*collocation-points/s"


def test_ncu_summary_groups_launches_into_the_library_s_kernel_classes():
    """bench.py --ncu-summary on a committed per-launch ncu CSV: kernel names map to the classes of pigan_profile_report, the
    whole-step row counts every launch, and every row carries the hash of the library sources in the tree (traffic_stale's key)."""
    import csv
    import io
    import bench
    assert bench.kernel_class("void jet2_layer_kernel<__half, 5, 1>(CUtensorMap_st, CUtensorMap_st, CUtensorMap_st, Jet2Params)") == "jet_layer_bwd(C=5)"
    assert bench.kernel_class("void jet2_layer_kernel<__half, 3, 4>(CUtensorMap_st)") == "jet_layer_fwd(C=3)"
    assert bench.kernel_class("void jet_layer_kernel<__half, 2, 5>(CUtensorMap_st)") == "jet_layer_fwd_split(C=2)"
    assert bench.kernel_class("void wgrad2_kernel<__half>(CUtensorMap_st, CUtensorMap_st, Wgrad2Params)") == "wgrad"
    assert bench.kernel_class("void fused_bwd256_kernel<__half, 5, 0>(CUtensorMap_st)") == "jet_layer_bwd_wgrad(C=5)"
    assert bench.kernel_class("void fused_fwd128_kernel<__half, 3>(FusedFwdMaps, FusedFwdParams)") == "gen_fwd_fused(C=3)"
    assert bench.kernel_class("void <unnamed>::critic_fused_kernel<4>(int)") == "critic_fused_kernel"
    assert bench.kernel_class("adam_kernel(float *, const float *)") == "adam_kernel"
    buf = io.StringIO()
    bench.ncu_summary(os.path.join(bench.ROOT, "profiles", "r02_launches_c5n2.csv"), "c5", out=buf)
    rows = {r["kernel_class"]: r for r in csv.DictReader(io.StringIO(buf.getvalue()))}
    assert int(rows["WHOLE_STEP"]["launches"]) == 188 and int(rows["wgrad"]["launches"]) == 20
    assert sum(int(r["launches"]) for k, r in rows.items() if k != "WHOLE_STEP") == 188
    assert abs(float(rows["WHOLE_STEP"]["kernel_time_us_under_ncu"]) - 27903.6) < 1.0
    assert {r["srchash"] for r in rows.values()} == {bench.library_srchash()}
    prof, src, stale = bench.ncu_profile("c5")
    assert prof and src.startswith("profiles/") and stale in (True, False)
