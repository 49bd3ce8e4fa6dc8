"""Host-side logic of bench.py that has no GPU in it: the N > 1 aggregation (replicas only: max of
the ranks' times, sum of their work) over a world_size-2 gloo group on the CPU, and the reference
arm's rank handling under a multi-rank launch."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
rank = int(os.environ["RANK"])
dist.init_process_group("gloo", rank=rank, world_size=2)
ms = bench.max_over_ranks([7.0, 11.5][rank], 2, device="cpu")
dist.barrier()
assert ms == 11.5, ms
assert abs(bench.job_mlups(2, 1000, 50, ms) - 2 * 1000 * 50 / 11.5e-3 / 1e6) < 1e-9
print("rank", rank, "ok", ms)
dist.destroy_process_group()
"""


def test_two_rank_aggregation_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    port = 29500 + os.getpid() % 2000
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=240)[0] for p in procs]
    for rank, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, o
        assert "rank %d ok 11.5" % rank in o


def test_single_rank_aggregation_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.25, 1) == 3.25
    assert bench.job_mlups(1, 4063232, 1000, 1279.0) == pytest.approx(4063232 * 1000 / 1.279 / 1e6)


def test_reference_arm_rank_handling():
    """--impl reference: rank 0 alone runs the oracle and prints the line; other ranks exit 0 silently."""
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0", "--fd-ratio", "4",
           "--steps", "20", "--warmup", "3", "--gpus", "2"]
    r1 = subprocess.run(cmd, env=dict(os.environ, RANK="1", WORLD_SIZE="2"), capture_output=True, text=True, timeout=600)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    r0 = subprocess.run(cmd, env=dict(os.environ, RANK="0", WORLD_SIZE="2"), capture_output=True, text=True, timeout=600)
    assert r0.returncode == 0, r0.stderr
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "MLUPS" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert line["steps"] == 20 and line["warmup"] == 3 and line["n_gpus"] == 2
    # a step is counted as the GPU arm counts it (r LB steps + one director and force update), and the config dict is
    # the one the GPU arm prints for the same command line
    sys.path.insert(0, ROOT)
    import bench
    sys.argv, keep = ["bench.py"] + cmd[2:], sys.argv
    try:
        args = bench.parse()
    finally:
        sys.argv = keep
    p, d, desc = bench.workload(args)
    assert line["config"] == json.loads(json.dumps(bench.config_of(args, p, desc, 1)))
    assert line["config"]["lb_steps_per_step"] == 4 and "4 LB steps" in line["config"]["step"]
    nf = 16 * 16 * 6
    assert line["value"] == pytest.approx(nf * 4 / (line["ms_per_step"] * 1e-3) / 1e6, rel=1e-6)


def test_bench_source_has_one_config_builder():
    """Both arms take `config` from bench.config_of, so the driver's same_config comparison holds by construction."""
    src = open(os.path.join(ROOT, "bench.py")).read()
    assert src.count('"config": config_of(') == 2
