"""N > 1 path of bench.py on CPU: two gloo ranks (replicas only -- DESIGN.md §8: the path has no
data-path collective; the only exchange is the max-over-ranks of the timed region)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["BRMPPI_ROOT"])
os.environ["BRMPPI_DIST_BACKEND"] = "gloo"
import bench, scenes
rank, world, local_rank, dist = bench.dist_setup(2)
assert world == 2 and dist is not None
# each rank reports its own time; every rank must see the slowest one
mine = 1.0 + rank
slowest = bench.max_over_ranks(mine, dist, "cpu")
assert slowest == 2.0, slowest
assert bench.whole_job_value(100.0, world, slowest) == 100.0
# rank r works on scene seed r: independent replicas with different inputs
a, _ = bench.workload("cfg1", 0)
b, _ = bench.workload("cfg1", rank)
assert (rank == 0) == bool((a.obstacles == b.obstacles).all())
dist.barrier()
dist.destroy_process_group()
sys.stdout.write(f"rank{rank}-ok\n")
"""


def _torchrun(args, env_extra, timeout=300):
    env = dict(os.environ, BRMPPI_ROOT=ROOT, **env_extra)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29613"] + args
    return subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, env=env, cwd=ROOT)


def test_two_gloo_ranks_reduce_the_timed_region(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    r = _torchrun([str(script)], {})
    assert r.returncode == 0, r.stdout + r.stderr
    assert "rank0-ok" in r.stdout and "rank1-ok" in r.stdout


def test_reference_arm_under_two_ranks_prints_one_line():
    r = _torchrun(["bench.py", "--gpus", "2", "--steps", "1", "--warmup", "0", "--impl", "reference",
                   "--workload", "cfg0"], {})
    assert r.returncode == 0, r.stdout + r.stderr
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    out = json.loads(lines[0])
    assert out["impl"] == "reference" and out["cpu_baseline"]["kind"] == "oracle"
    assert out["e2e"]["h2d_bytes_per_step"] == 0 and out["value"] > 0
