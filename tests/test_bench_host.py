"""Host logic of bench.py that needs no GPU: the N > 1 path (replicas only: the single collective is the max over
ranks of the elapsed time) with world_size 2 over gloo, the reference arm's JSON line, and the clock-sample parser."""
import json
import os
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, "cpu")          # rank 1 is the slower replica
    if rank == 0:
        with open(out, "w") as f:
            json.dump({"ms": ms, "rate": bench.aggregate_rate(1000, 4, world, ms * 1e-3)}, f)
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_time_is_max_over_ranks_gloo(tmp_path):
    out = str(tmp_path / "r.json")
    mp.spawn(_worker, args=(2, 29533, out), nprocs=2, join=True)
    r = json.load(open(out))
    assert r["ms"] == 15.0
    assert r["rate"] == 1000 * 4 * 2 / 15e-3          # all ranks' cell-updates over the slowest rank's time


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(3.5, 1, "cpu") == 3.5
    assert bench.aggregate_rate(8, 2, 1, 0.5) == 32.0


def test_reference_arm_prints_contract_line():
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=300)
    assert p.returncode == 0, p.stderr
    d = json.loads(p.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["unit"] == "cell-updates/s" and d["value"] > 1e4
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["gpu_launches"] == 0 and d["vs_baseline"] is None


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       capture_output=True, text=True, timeout=60, env=env)
    assert p.returncode == 0 and p.stdout.strip() == ""


def test_clock_sampler_parses_nvidia_smi_lines():
    import bench
    s = bench.ClockSampler(0)
    s.proc = type("P", (), {"terminate": lambda self: None, "wait": lambda self, timeout=None: 0})()
    s.lines = ["0, 1965, 1965, 512.3, Not Active, Not Active, Not Active, Not Active",
               "0, 1740, 1965, 1003.1, Not Active, Not Active, Not Active, Active",
               "0, 1725, 1965, 998.0, Not Active, Not Active, Not Active, Active"]
    r = s.stop()
    assert r["sm_mhz"] == 1740 and r["sm_max_mhz"] == 1965 and r["reasons"] == ["sw_power_cap"] and r["samples"] == 3
