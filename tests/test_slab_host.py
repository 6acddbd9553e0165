"""Host logic of the z-slab runner (paper_2507_08820_b200/slab.py) on the CPU: who owns which
layers, who the neighbours are, and that the face transport delivers, over gloo with 2 and 3 ranks, the LOW pack of
the rank above to this rank's HIGH side and the HIGH pack of the rank below to its LOW side.  No GPU, no kernels."""
import os
import subprocess
import sys

import pytest

from paper_2507_08820_b200 import slab

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("nzg,world", [(8, 1), (8, 2), (9, 2), (7, 3), (256 * 5, 5), (5, 5), (100, 7)])
def test_slab_extent_partitions_the_layers(nzg, world):
    ext = [slab.slab_extent(r, world, nzg) for r in range(world)]
    assert ext[0][0] == 0 and sum(n for _, n in ext) == nzg
    for (z0, n), (z1, _) in zip(ext, ext[1:]):
        assert z0 + n == z1                                   # contiguous, in rank order
    sizes = [n for _, n in ext]
    assert min(sizes) >= 1 and max(sizes) - min(sizes) <= 1


def test_slab_extent_rejects_empty_slabs_and_bad_ranks():
    with pytest.raises(ValueError):
        slab.slab_extent(0, 4, 3)
    with pytest.raises(ValueError):
        slab.slab_extent(2, 2, 8)
    with pytest.raises(ValueError):
        slab.slab_extent(0, 0, 8)


def test_neighbours_are_periodic():
    assert slab.neighbours(0, 1) == (0, 0)
    assert slab.neighbours(0, 2) == (1, 1) and slab.neighbours(1, 2) == (0, 0)
    assert slab.neighbours(0, 4) == (3, 1) and slab.neighbours(3, 4) == (2, 0)


def test_single_rank_transport_hands_the_faces_across():
    import torch
    tr = slab.FaceTransport()
    lo, hi = torch.arange(6.0), torch.arange(6.0) + 10
    for_low, for_high = tr.exchange(lo, hi)
    assert for_low is hi and for_high is lo                   # the rank is its own neighbour: LOW pack -> HIGH side


WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_2507_08820_b200 import slab
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
tr = slab.FaceTransport()
assert (tr.rank, tr.world) == (rank, world)
below, above = slab.neighbours(rank, world)
for rep in range(3):                                          # buffers are reused from call to call
    lo = torch.full((9, 3, 5), 100.0 * rank + 1 + rep, dtype=torch.float64)      # this rank's LOW pack
    hi = torch.full((9, 3, 5), 100.0 * rank + 2 + rep, dtype=torch.float64)      # this rank's HIGH pack
    for_low, for_high = tr.exchange(lo, hi)
    assert torch.all(for_high == 100.0 * above + 1 + rep), (rank, for_high[0, 0, 0])   # LOW pack of the rank above
    assert torch.all(for_low == 100.0 * below + 2 + rep), (rank, for_low[0, 0, 0])     # HIGH pack of the rank below
dist.barrier()
if rank == 0:
    print("TRANSPORT_OK", world)
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world,port", [(2, 29631), (3, 29633)])
def test_face_transport_over_gloo(tmp_path, world, port):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)]
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    assert r.stdout.count(f"TRANSPORT_OK {world}") == 1
