"""Host logic of bench.py without a GPU: the reference arm prints a contract-shaped
JSON line, and the max/sum-over-ranks timing reduction works across 2 ranks (gloo)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_contract_line():
    env = dict(os.environ, PYTHONPATH=ROOT)
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "1"], capture_output=True, text=True, env=env, cwd=ROOT, timeout=600)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "interactions/s" and line["value"] > 1e6
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"], "h2d_bytes_per_step": 0,
                           "d2h_bytes_per_step": 0}
    assert line["config"]["workload"].startswith("config4") and line["higher_is_better"] is True


def test_own_arm_refuses_to_run_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, cwd=ROOT, timeout=600)
    assert out.returncode != 0 and "no CPU fallback" in (out.stderr + out.stdout)


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import bench
rank, world = bench.dist_init("gloo")
bench.barrier()
mx = bench.reduce_over_ranks(10.0 + 5.0 * rank, "max")
sm = bench.reduce_over_ranks(1.0 + rank, "sum")
print(f"RESULT {{rank}} {{world}} {{mx}} {{sm}}", flush=True)
# rank-0-only reference arm: other ranks exit 0 without work
if rank != 0:
    class A: gpus=2; steps=1; warmup=1; config=4
    assert bench.run_reference(A) == 0
import torch.distributed as dist
dist.destroy_process_group()
"""


def test_two_rank_gloo_timing_reduction(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT="29617")
        procs.append(subprocess.Popen([sys.executable, str(script)], stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True, env=env))
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (so, se) in zip(procs, outs):
        assert p.returncode == 0, se
    for r, (so, _) in enumerate(outs):
        res = [l for l in so.splitlines() if l.startswith("RESULT")][0].split()
        assert int(res[1]) == r and int(res[2]) == 2
        assert float(res[3]) == 15.0 and float(res[4]) == 3.0        # max over ranks, sum over ranks


def test_gpus_flag_starts_the_ranks_itself(capfd):
    """`python bench.py --gpus 2` with no launcher around it: bench.spawn_ranks starts two ranks (RANK / WORLD_SIZE /
    MASTER_* as torchrun would), they rendezvous (gloo here: the ranks run tests/bench_stub_rank.py, bench.py's timing
    path with the GPU taken out), the timing is the max over ranks, the units the sum, and rank 0 alone prints, with
    n_gpus = 2."""
    import argparse
    sys.path.insert(0, ROOT)
    import bench
    saved = {k: os.environ.pop(k) for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT") if k in os.environ}
    try:
        rc = bench.spawn_ranks(argparse.Namespace(gpus=2), ["--gpus", "2", "--steps", "4"],
                               script=os.path.join(ROOT, "tests", "bench_stub_rank.py"))
    finally:
        os.environ.update(saved)
    assert rc == 0
    lines = [l for l in capfd.readouterr().out.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                   # rank 0 only
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["steps"] == 4 and d["config"]["parallelism"] == "replicas only"
    assert d["ms_per_step"] >= 3.9                           # rank 1 sleeps 4 ms per step, rank 0 only 2: the max over ranks
    assert abs(d["value"] - 2 * 1000.0 / (d["ms_per_step"] * 1e-3)) < 1e-6 * d["value"]   # units of BOTH ranks / that time


def test_gpus_flag_must_agree_with_the_launcher():
    env = dict(os.environ, RANK="0", LOCAL_RANK="0", WORLD_SIZE="1", MASTER_ADDR="127.0.0.1", MASTER_PORT="29618")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2"],
                         capture_output=True, text=True, env=env, cwd=ROOT, timeout=600)
    assert out.returncode != 0 and "WORLD_SIZE=1" in (out.stderr + out.stdout)


def test_both_arms_print_the_same_config_object():
    """The driver compares the two arms' `config`: one function makes it for both."""
    sys.path.insert(0, ROOT)
    import bench
    from workloads import make_config, params_f32
    w = make_config(1)
    c = bench.workload_config(w, params_f32(w.params))
    assert c["workload"] == w.name and c["n"] == 2048 and c["parallelism"] == "replicas only" and "flushed" in c["l2"]
    src = open(os.path.join(ROOT, "bench.py")).read()
    assert src.count('"config": workload_config(w, p)') == 2
