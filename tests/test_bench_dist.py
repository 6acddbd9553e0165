"""N>1 plumbing of bench.py on CPU (gloo, world_size 2): the path does not shard ("replicas only", DESIGN.md
section 9), so what multi-rank runs need is the rendezvous, the max-over-ranks of the device time, the sum of the
sites, and that only rank 0 prints.  No GPU and no compute kernels are involved here."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import bench
rank, world, local = bench.dist_setup(2)
assert world == 2 and rank == int(os.environ["RANK"])
bench.barrier_all()
mx = bench.max_over_ranks(10.0 + rank)          # the slower rank decides
sm = bench.sum_over_ranks(100.0 * (rank + 1))
assert mx == 11.0 and sm == 300.0, (mx, sm)
bench.barrier_all()
if rank == 0:
    print("DIST_OK", mx, sm)
"""


def _torchrun(args, port):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port)] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)


def test_max_and_sum_over_ranks_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    r = _torchrun([str(script)], 29611)
    assert r.returncode == 0, r.stderr[-2000:]
    assert r.stdout.count("DIST_OK 11.0 300.0") == 1


def test_reference_arm_under_torchrun_prints_once():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "1"], 29613)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                               # rank 0 alone runs and prints
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["unit"] == "MLUPS" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
