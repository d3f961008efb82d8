"""world_size-2 gloo tests (CPU): bench.py's multi-rank plumbing.  The path is "replicas only"
(DESIGN.md section 8): no data-path collective, one all_reduce(MAX) of the elapsed time."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_SCRIPT = r'''
import os, sys
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, ws = dist.get_rank(), dist.get_world_size()
assert bench.dist_info()[0] == rank and bench.dist_info()[2] == ws == 2
v = bench.max_over_ranks(10.0 + 5.0 * rank, ws)
assert v == 15.0, v
# replicas: every rank plans the same layers and generates its own (identical-recipe) inputs
plan = bench.step_plan("c1")
assert [a for a, _ in plan] == ["x"]
print("rank %%d ok" %% rank)
dist.destroy_process_group()
''' % ROOT


def _torchrun(args, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29731"] + args
    return subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, cwd=ROOT)


def test_max_over_ranks_gloo(tmp_path):
    script = tmp_path / "mr.py"
    script.write_text(_SCRIPT)
    r = _torchrun([str(script)])
    assert r.returncode == 0, r.stderr[-2000:]
    assert "rank 0 ok" in r.stdout and "rank 1 ok" in r.stdout


def test_reference_arm_under_torchrun_prints_one_line():
    r = _torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config",
                   "c1", "--steps", "2", "--warmup", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                   # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0
    assert d["metric"] == "fused W4A4 linear tokens/s" and d["unit"] == "tokens/s"
