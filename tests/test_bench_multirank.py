"""-m "not gpu": the N > 1 host logic of bench.py with world_size 2 on the gloo backend (the path does not shard:
replicas only, DESIGN.md section 7 -- the only cross-rank step is the MAX over the ranks' timings), and the
reference arm under a 2-process launch (rank 0 alone prints, the other rank exits 0 without work)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r'''
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
# each replica reports its own timings; every rank must end up with the slowest ones
red = bench.max_over_ranks([100.0 + 7.0 * rank, 3.0 - rank], device="cpu")
val = bench.whole_job_value(world, 10, 1.0e6, red[0])
open(os.path.join({out!r}, "rank%d.json" % rank), "w").write(json.dumps(dict(rank=rank, world=world, red=red, value=val)))
dist.destroy_process_group()
'''


def _torchrun(args, env_extra=None, timeout=300):
    env = dict(os.environ, PYTHONPATH=ROOT + os.pathsep + os.environ.get("PYTHONPATH", ""), OMP_NUM_THREADS="2")
    env.update(env_extra or {})
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", "29731"] + args
    return subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, env=env, cwd=ROOT)


def test_max_over_ranks_and_whole_job_value_gloo(tmp_path):
    worker = tmp_path / "worker.py"
    worker.write_text(_WORKER.format(root=ROOT, out=str(tmp_path)))
    res = _torchrun([str(worker)])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [json.loads((tmp_path / f"rank{r}.json").read_text()) for r in (0, 1)]   # one file per rank: stdout interleaves
    assert sorted(l["rank"] for l in lines) == [0, 1]
    for l in lines:
        assert l["world"] == 2 and l["red"] == [107.0, 3.0]               # MAX over ranks, on every rank
        assert abs(l["value"] - 2 * 10 * 1.0e6 / 0.107) < 1e-3          # two replicas in the slowest rank's time


def test_reference_arm_under_two_ranks_prints_once():
    res = _torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "0",
                     "--steps", "1", "--warmup", "0"])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [json.loads(l) for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    assert lines[0]["impl"] == "reference" and lines[0]["n_gpus"] == 2 and lines[0]["value"] > 0
    assert lines[0]["cpu_baseline"]["kind"] == "oracle" and lines[0]["e2e"]["h2d_bytes_per_step"] == 0
