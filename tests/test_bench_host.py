"""Host-side logic of bench.py on CPU: the N > 1 timing aggregation (max over ranks of the time, sum of the
units) over a world-size-2 gloo group, the `--impl reference` arm (rank 0 prints one JSON line, other ranks
print nothing), and the clock-sampler parser."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
rank = int(os.environ["RANK"])
dist.init_process_group(backend="gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=2)
bench.barrier()
t, u = bench.dist_max_sum(1.0 + rank, 100.0 * (rank + 1), torch.device("cpu"))
bench.barrier()
print(json.dumps({{"rank": rank, "t": t, "u": u}}))
dist.destroy_process_group()
"""


def test_dist_max_sum_world_size_2_gloo(tmp_path):
    port = 29500 + os.getpid() % 2000
    script = tmp_path / "w.py"
    script.write_text(_WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script)], env={**os.environ, "RANK": str(r), "WORLD_SIZE": "1"},
                              stdout=subprocess.PIPE, text=True) for r in range(2)]
    outs = [json.loads(p.communicate(timeout=240)[0].strip().splitlines()[-1]) for p in procs]
    for o in outs:
        assert o["t"] == 2.0 and o["u"] == 300.0     # max of (1, 2), sum of (100, 200)


def test_dist_max_sum_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.dist_max_sum(3.5, 7.0, None) == (3.5, 7.0)
    bench.barrier()


def test_reference_arm_prints_contract_line_on_rank0_only():
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "c1_64sq", "--steps", "2",
           "--warmup", "1", "--gpus", "2"]
    r0 = subprocess.run(cmd, env={**os.environ, "RANK": "0"}, capture_output=True, text=True, timeout=600)
    r1 = subprocess.run(cmd, env={**os.environ, "RANK": "1"}, capture_output=True, text=True, timeout=600)
    assert r0.returncode == 0 and r1.returncode == 0 and r1.stdout.strip() == ""
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "MLUPS" and line["unit"] == "MLUPS" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == {"value": line["value"], "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["config"]["workload"] == "c1_64sq" and line["higher_is_better"] is True


def test_clock_sampler_parses_nvidia_smi_lines(monkeypatch):
    sys.path.insert(0, ROOT)
    import bench

    class FakeProc:
        def terminate(self): pass
        def communicate(self, timeout=None):
            return ("1965, 1965, Not Active, Not Active, Not Active, Active\n"
                    "1800, 1965, Not Active, Not Active, Not Active, Not Active\n"
                    "garbage\n1700, 1965, Not Active, Active, Not Active, Not Active\n", "")
    s = bench.ClockSampler.__new__(bench.ClockSampler)
    s.proc = FakeProc()
    out = s.stop()
    assert out["sm_mhz"] == 1800 and out["sm_max_mhz"] == 1965
    assert out["reasons"] == ["hw_thermal_slowdown", "sw_power_cap"]


def test_full_mode_times_the_step_counts_baseline_json_states():
    """bench.py --full: configs 2-5 (and their uniform counterparts) at the step counts BASELINE.json states."""
    import re
    sys.path.insert(0, ROOT)
    import bench
    from paper_2509_01099_b200 import inputs
    cfgs = json.load(open(os.path.join(ROOT, "BASELINE.json")))["configs"]
    stated = [int(re.search(r"(\d+) steps timed", c).group(1)) for c in cfgs[1:]]
    assert stated == [20000, 50000, 5000, 10000]
    names = [n for n, _ in bench.FULL_RUNS]
    for key, steps in zip(("c2_512sq", "c3_1024sq", "c4_128cu", "c5_256cu"), stated):
        assert key in names
        assert inputs.workload(key).steps == steps and steps % 100 == 0        # sampled every 100 steps (A20)
    for key in ("c2_512sq", "c3_1024sq", "c5_256cu"):                          # the configs that ask for a uniform counterpart
        assert key + "_uniform" in names
        assert inputs.workload(key + "_uniform").steps == inputs.workload(key).steps
    assert ("c3_1024sq", 1) in bench.FULL_RUNS and ("c5_256cu", 1) in bench.FULL_RUNS   # "fp64 and fp32 storage"
