"""The z-slab decomposition across PROCESSES: two and three ranks under torchrun, each owning a slab
of one global lattice on the same GPU, faces moved rank to rank by paper_2507_08820_b200.slab.FaceTransport (gloo through
pinned host buffers here; NCCL send/recv when every rank has its own GPU) must reproduce the undivided lattice bit for
bit.  tests/test_gpu_slab.py proves the same inside one process; tests/test_slab_host.py covers the host logic on the CPU."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("world,port", [(2, 29641), (3, 29643)])
def test_slab_ranks_equal_the_undivided_lattice(world, port):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "tests", "slab_dist_worker.py")]
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, (r.stdout[-2000:], r.stderr[-4000:])
    assert r.stdout.count(f"SLAB_DIST_OK {world}") == 1
