"""The N > 1 path of bench.py on CPU: two gloo ranks (replicas only: the single cross-rank step
is the MAX over ranks of the timed durations; the reference arm prints on rank 0 only)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys
sys.path.insert(0, %r)
OUT = %r
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
r = dist.get_rank()
out = bench.max_over_ranks([1.0 + r, 10.0 - r, 5.0])
assert out == [2.0, 10.0, 5.0], out
assert bench.whole_job_value(100.0, dist.get_world_size(), out[0]) == 100.0
dist.barrier()
dist.destroy_process_group()
open(os.path.join(OUT, "rank%%d.ok" %% r), "w").write("ok")     # one file per rank: stdout of two ranks interleaves
'''


def _run(args, **kw):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    return subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                           "--master-addr", "127.0.0.1", "--master-port", "29517"] + args,
                          cwd=ROOT, env=env, capture_output=True, text=True, timeout=600, **kw)


def test_max_over_ranks_with_two_gloo_ranks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % (ROOT, str(tmp_path)))
    p = _run([str(script)])
    assert p.returncode == 0, p.stdout + p.stderr
    assert (tmp_path / "rank0.ok").exists() and (tmp_path / "rank1.ok").exists()


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    p = _run(["bench.py", "--impl", "reference", "--gpus", "2", "--config", "0", "--steps", "1", "--warmup", "0"])
    assert p.returncode == 0, p.stdout + p.stderr
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0


def test_single_rank_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([3.0, 4.0]) == [3.0, 4.0]
