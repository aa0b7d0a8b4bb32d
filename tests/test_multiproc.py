"""The N > 1 path of bench.py on CPU (gloo, world_size 2).  The hot path does not shard ("replicas only", DESIGN.md
section 9): every rank runs the same workload on its own GPU and the only cross-rank logic is the barrier, the
max-over-ranks timing and the whole-job value -- that logic is what runs here, plus the rank-0-only reference arm under
torchrun."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import bench

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group(backend="gloo", rank=rank, world_size=world)
    ms_local = 10.0 + 5.0 * rank  # rank 1 is the slow one
    dist.barrier()
    ms = bench.max_over_ranks(ms_local, dist, "cpu")
    value = bench.job_value(1000, 2, world, ms)
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, ms, value))


def test_max_over_ranks_and_job_value_gloo_world2():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # both ranks see the slow rank's time; the job value counts both replicas over that time
    for rank, ms, value in got:
        assert ms == 15.0
        assert value == pytest.approx(2 * 1000 * 3 * 2 / 15.0e-3 / 1e9)


def test_single_rank_helpers():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.max_over_ranks(3.5) == 3.5
    # board energy per point-stage from the sampled mean power: 1000 W x 20 steps of 11.8 ms over 256^3 x 3 x 20 updates
    assert bench.energy_nj_per_point_stage({"power_w_mean": 1000.0}, 20 * 11.8, 256 ** 3, 20) == pytest.approx(234.445, rel=1e-5)
    assert bench.energy_nj_per_point_stage({"sm_mhz": None, "reasons": ["nvidia-smi unavailable"]}, 1.0, 10, 1) is None
    assert bench.job_value(16777216, 10, 1, 130.0) == pytest.approx(16777216 * 30 / 0.130 / 1e9)


def test_reference_arm_under_torchrun_prints_one_line_on_rank0():
    """`bench.py --impl reference` launched the way the driver launches N > 1: rank 0 times the oracle and prints ONE
    JSON line, the other rank exits 0 without work."""
    port = 31500 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--workload", "c1"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["unit"] == "Gpts/s"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["value"] > 0
