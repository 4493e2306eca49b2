"""Host-side logic of bench.py that needs no GPU: the multi-rank (replicas-only) aggregation over gloo with
world_size 2, the reference arm's rank gating and JSON contract, and the clock-sample parser."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist

    import bench

    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r needs (1 + r) seconds for 1000 units: the job did 2000 units in max = 2 s
    slow = bench.max_over_ranks(1.0 + rank, world)
    rate = bench.whole_job_rate(1000.0, 1.0 + rank, world)
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, slow, rate))


def test_replica_aggregation_over_gloo_world2():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, slow, rate in res:
        assert slow == 2.0          # every rank sees the slowest rank's time
        assert rate == 1000.0       # 2 ranks x 1000 units / 2 s


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.whole_job_rate(10.0, 2.0, 1) == 5.0


def _run_reference(env_extra):
    env = dict(os.environ, **env_extra)
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "lj864",
                           "--steps", "1", "--warmup", "0", "--inner", "5"], capture_output=True, text=True, env=env,
                          timeout=600)


def test_reference_arm_prints_the_contract_line_on_rank0_only():
    r0 = _run_reference({"RANK": "0", "WORLD_SIZE": "2"})
    assert r0.returncode == 0, r0.stderr
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "timesteps/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert line["gpu_launches"] == 0 and line["higher_is_better"] is True
    r1 = _run_reference({"RANK": "1", "WORLD_SIZE": "2"})
    assert r1.returncode == 0 and r1.stdout.strip() == ""


def test_clock_sampler_parses_nvidia_smi_lines():
    sys.path.insert(0, ROOT)
    import bench

    c = bench.ClockSampler(0)
    c.proc = type("P", (), {"terminate": lambda self: None, "wait": lambda self, timeout=None: 0,
                            "kill": lambda self: None})()
    c.lines = ["1965, 1965, 250.1, Not Active, Not Active, Not Active, Not Active",
               "1900, 1965, 900.0, Not Active, Not Active, Not Active, Active",
               "garbage"]
    out = c.stop(0)
    assert out["sm_mhz"] == 1932.5 and out["sm_max_mhz"] == 1965.0 and out["reasons"] == ["sw_power_cap"]


def test_bench_refuses_to_run_without_a_gpu():
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1"], capture_output=True, text=True,
                       timeout=300)
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)


def test_traffic_profiles_named_by_bench_exist_and_name_their_command():
    """`roofline.traffic` is null with a pointer to an ncu capture under profiles/ (`traffic_source`): every file
    bench.py can point at is committed and states the command that made it."""
    import bench

    for name, rel in bench.TRAFFIC_PROFILES.items():
        path = os.path.join(ROOT, rel)
        assert os.path.exists(path), (name, rel)
        txt = open(path).read()
        assert "ncu --set full" in txt and "bench.py" in txt and "dram__bytes_read.sum" in txt, rel
