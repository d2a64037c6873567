"""-m "not gpu": bench.py's host logic -- launch/pass bookkeeping, clock-line parsing, the replicas-only
aggregation over ranks (world_size 2, gloo, on CPU) and the bounded oracle sample used by cpu_baseline /
--impl reference."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_pass_and_launch_counts():
    import bench
    # SURVEY.md §8 size table: 1650 passes at configs[2..4], 33 at configs[0..1]
    assert bench.passes_per_interval(50, 3, 10) == 1650
    assert bench.passes_per_interval(1, 3, 10) == 33
    # prep + predict + initial residual + 2 norm kernels + per (em,k): 2 corrupts + 11 x (pass, reduce, control)
    assert bench.expected_launches(50, 3, 10, True) == 5 + 150 * (2 + 33)
    # cluster by cluster: per (em,k) one write-back/statistics kernel + one cooperative M-step kernel, + last write-back
    assert bench.expected_launches(50, 3, 10, True, "percluster") == 5 + 150 * 2 + 1
    # compressed, cluster groups of 4 (13 groups at K=50, the last of 2): per EM iteration 13 write-back/statistics
    # kernels (which take the cross grams as well in the first one) + 50 M-step kernels + (12*3 + 1) correction kernels,
    # + last write-back
    assert bench.expected_launches(50, 3, 10, True, "compressed", "scalar") == 5 + 3 * (13 + 50 + 37) + 1
    assert bench.expected_launches(50, 3, 10, True, "compressed", "full") == 5 + 3 * (13 + 50 + 37) + 1
    per = bench.wbgroup_bytes_per_sample(50, 3, "full")
    assert len(per) == 40 and per[0] == 64 + 4 * 64 and per[1] == 128 + 8 * 64 and per[-1] == 128 + 2 * 64
    assert bench.wbgroup_bytes_per_sample(1, 1, "scalar") == [64 + 16, 128 + 16]
    # n_lm = 25 re-centres twice more per M-step: 3 statistics kernels and 3 M-step kernels
    assert bench.expected_launches(1, 2, 25, False, "compressed") == 3 + 2 * 6 + 1
    assert bench.seconds_per_interval(2000.0, 1) == 2.0
    assert bench.seconds_per_interval(2000.0, 4) == 0.5          # replicas: 4 intervals per step time


def test_parse_clock_lines():
    import bench
    lines = ["0, 1965, 1965, 612.10, 0x0000000000000000, Not Active, Not Active, Not Active, Not Active\n",
             "0, 1410, 1965, 1001.50, 0x0000000000000004, Not Active, Not Active, Not Active, Active\n",
             "0, 1395, 1965, 998.00, 0x0000000000000004, Not Active, Not Active, Not Active, Active\n",
             "garbage\n"]
    c = bench.parse_clock_lines(lines)
    assert c["sm_mhz"] == 1410 and c["sm_max_mhz"] == 1965 and c["reasons"] == ["sw_power_cap"] and c["samples"] == 3
    assert bench.parse_clock_lines([])["sm_mhz"] is None


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
ms = bench.max_over_ranks(100.0 + 50.0 * rank, world)          # rank 1 is the slow one
dist.barrier()
if rank == 0:
    print("RESULT", ms, bench.seconds_per_interval(ms, world))
dist.destroy_process_group()
"""


def test_replicas_max_over_ranks_gloo_world2(tmp_path):
    """N>1 path: no data-path collective, the step time is the max over ranks, value = time / N intervals."""
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29531", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r), LOCAL_RANK=str(r)),
                              stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = [p.communicate(timeout=120) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    line = [l for l in outs[0][0].splitlines() if l.startswith("RESULT")][0].split()
    assert float(line[1]) == 150.0 and float(line[2]) == 0.075


def test_reference_arm_prints_contract_line():
    """bench.py --impl reference on configs[0] (the oracle, host cores): one JSON line with the contract's keys."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "s" and line["higher_is_better"] is False
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0
    # other ranks of a torchrun launch do no work
    out1 = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0"],
                          capture_output=True, text=True, timeout=60, env=dict(os.environ, RANK="1", WORLD_SIZE="2"))
    assert out1.returncode == 0 and out1.stdout.strip() == ""


def test_oracle_sample_scaling_is_exact_when_sample_is_whole_problem():
    """With the sample equal to the whole (tiny) problem both scale factors are 1: the reported time is the measured
    time of predict + calibrate, nothing extrapolated."""
    import bench
    from sagecal_inputs import make_config
    p = make_config(0)
    v, desc, parts = bench.oracle_sample(p, dict(T=p.T, K=p.K, n_em=p.n_em, n_lm=p.n_lm))
    assert parts["predict_scale"] == 1.0 and parts["calibrate_scale"] == 1.0
    assert abs(v - (parts["predict_s"] + parts["calibrate_s"])) < 1e-12
