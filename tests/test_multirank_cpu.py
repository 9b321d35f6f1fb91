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


# K-sharded solve: every rank builds the record of ITS range of the samples from the oracle's
# costs and sampled controls, the records are all-gathered by the package's own exchange function over gloo, and
# the merge rule of the online softmax (any partition of the samples gives the two-pass result) is checked
# against the oracle's plain two-pass update.
SHARD_WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["BRMPPI_ROOT"])
import numpy as np, torch
import torch.distributed as dist
import scenes
from oracle import oracle as O
from paper_2508_05773_b200 import sharded
dist.init_process_group(backend="gloo")
rank, world = dist.get_rank(), dist.get_world_size()
sc = scenes.scene_cfg1(3)
p = sc.params.with_(K=301, T=12, n_iter=1, lam=7.0)
ref = O.iteration(p, 5, sc.x0, sc.goal, sc.obstacles, np.zeros((p.T, 2)), want_samples=True)
k0, Kr = sharded.shard_range(p.K, rank, world)
ranges = [sharded.shard_range(p.K, r, world) for r in range(world)]
assert ranges[0][0] == 0 and sum(n for _, n in ranges) == p.K and ranges[1][0] == ranges[0][1]
S, u = ref["S"][k0:k0 + Kr], ref["u"][k0:k0 + Kr]
# this rank's record: (m, argmin, eta, A[2T]) of its own samples, weights against its OWN minimum
m = S.min(); w = np.exp(-(S - m) / p.lam)
rec = np.concatenate([[m, k0 + int(np.argmin(S)), w.sum()], (w[:, None, None] * u).sum(axis=0).reshape(-1)])
records = sharded.gather_records(dist, torch.from_numpy(rec), world).numpy()
assert records.shape == (world, 3 + 2 * p.T)
assert records[rank, 1] == rec[1] and all(ranges[r][0] <= records[r, 1] < ranges[r][0] + ranges[r][1] for r in range(world))
# merge in rank order: m = min m_p, c_p = exp(-(m_p - m)/lambda), eta = sum c_p eta_p, U = sum c_p A_p / eta
mg = records[:, 0].min(); c = np.exp(-(records[:, 0] - mg) / p.lam)
eta = (c * records[:, 2]).sum()
U = (c[:, None] * records[:, 3:]).sum(axis=0).reshape(p.T, 2) / eta
assert np.abs(U - ref["U"]).max() <= 1e-12, np.abs(U - ref["U"]).max()
assert abs(eta - ref["eta"]) <= 1e-12 * ref["eta"]
assert int(records[np.argmin(records[:, 0]), 1]) == ref["argmin"]
dist.barrier()
dist.destroy_process_group()
sys.stdout.write(f"shard{rank}-ok\n")
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


def test_sharded_exchange_and_merge_rule_over_two_gloo_ranks(tmp_path):
    script = tmp_path / "shard_worker.py"
    script.write_text(SHARD_WORKER)
    r = _torchrun([str(script)], {})
    assert r.returncode == 0, r.stdout + r.stderr
    assert "shard0-ok" in r.stdout and "shard1-ok" in r.stdout
