"""Host logic of bench.py that needs no GPU: the replicas-only multi-rank arithmetic over a world_size-2 gloo group
(no data-path collective; the only exchange is the MAX of the device times) and the reference arm
(the CPU oracle; ranks other than 0 exit without work)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world)          # rank 1 is the slow one
    out.put((rank, ms, bench.whole_job_rate(world, 2.0, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_rate_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, rate in got:
        assert ms == 15.0                                          # every rank reports the slowest rank's time
        assert rate == pytest.approx(2 * 2.0 / 15.0e-3)            # units of both replicas / max time


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.whole_job_rate(1, 8.0, 4.0) == pytest.approx(2000.0)


def _run_reference(env_extra):
    env = dict(os.environ, **env_extra)
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "tiny", "--steps", "1",
                           "--warmup", "0", "--cpu-seconds", "2"], capture_output=True, text=True, env=env, timeout=600)


def test_reference_arm_prints_the_contract_line_on_rank0():
    r = _run_reference({"RANK": "0", "WORLD_SIZE": "1"})
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "MP/s" and line["higher_is_better"] is True
    assert line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] == 1
    assert line["e2e"] == {"value": line["value"], "unit": "MP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["config"]["workload"] == "tiny" and line["vs_baseline"] is None
    # ms_per_step is what one step of this arm actually timed (a bounded sample), the extrapolation sits in cpu_baseline
    cb = line["cpu_baseline"]
    assert line["ms_per_step"] == pytest.approx(cb["sample_seconds_median"] * 1e3, rel=1e-2, abs=1.0)
    assert cb["nproc"] >= 1 and isinstance(cb["cpu_model"], str) and cb["scale_gaussians"] >= 1 and cb["scale_tiles"] >= 1
    assert cb["full_view_seconds_extrapolated"] > 0


def test_reference_arm_slices_gaussians_and_tiles_on_a_larger_scene():
    """With a small time budget the sample takes a slice of the Gaussians and every k-th tile; the extrapolated
    full-view time stays within a factor of the time of running the whole view."""
    import bench
    smp = bench.OracleSampler("object", 20_000, 0.5)
    assert smp.kt > 1 and smp.n_slice <= smp.N
    wall, t, full = smp.sample(0)
    assert set(t) == {"project_fwd", "bin_tiles", "raster_fwd", "raster_bwd", "project_bwd"}
    assert full > wall > 0


def test_reference_arm_other_ranks_exit_without_work():
    r = _run_reference({"RANK": "1", "WORLD_SIZE": "2"})
    assert r.returncode == 0 and r.stdout.strip() == ""
