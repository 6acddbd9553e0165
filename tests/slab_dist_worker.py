"""Worker of tests/test_gpu_slab_dist.py: run under torchrun (gloo, every rank on cuda:0).  Every rank runs its slab of
the global lattice through paper_2507_08820_b200.slab.SlabLattice and, for comparison, the undivided lattice through one
plain handle; the gathered slabs must equal the undivided lattice bit for bit."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import numpy as np
import torch
import torch.distributed as dist

from paper_2507_08820_b200 import binding, slab, synthetic

CASES = [
    # nx, ny, nzg, precision, scheme, walls, force
    (40, 6, 9, binding.F64, binding.SCHEME_AB, False, None),
    (40, 6, 9, binding.F64, binding.SCHEME_AA, True, (1e-5, -2e-6, 3e-6)),
    (136, 4, 8, binding.F32, binding.SCHEME_AB, True, None),
    (33, 5, 7, binding.F32, binding.SCHEME_AA, False, (1e-6, 0.0, 0.0)),
]


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    tau, kT, seed = 0.8, 1e-4, 77
    for nx, ny, nzg, prec, scheme, walls, force in CASES:
        rho, u = synthetic.smooth_random_fields(nx, ny, nzg, 23)
        lat = slab.SlabLattice(nx, ny, nzg, tau, kT, 1.0, seed, prec, scheme=scheme, walls=walls, force=force)
        assert (lat.z0, lat.nz) == slab.slab_extent(rank, world, nzg)
        lat.init(rho, u)
        one = binding.Rflbm(nx, ny, nzg, tau, kT, 1.0, seed, prec, scheme=scheme)
        if walls:
            one.set_walls_z(True)
        if force is not None:
            one.set_force(*force)
        one.init(torch.from_numpy(rho), torch.from_numpy(u))
        done = 0
        for target in (0, 1, 2, 9):
            lat.step(target - done)
            one.step(target - done)
            done = target
            assert torch.equal(lat.gather(lat.get_populations(), 1), one.get_populations().cpu()), (rank, target)
            r1, u1 = one.moments()
            rs, us = lat.moments()
            assert torch.equal(lat.gather(rs, 0), r1.cpu()) and torch.equal(lat.gather(us, 1), u1.cpu())
            assert torch.equal(lat.gather(lat.stress(), 1), one.stress().cpu())
        d_all, d_one = np.array(lat.diagnostics()), np.array(one.diagnostics())
        tol = 1e-12 if prec == binding.F64 else 1e-6
        assert np.allclose(d_all[:7], d_one[:7], rtol=tol, atol=tol), (d_all, d_one)
        assert np.allclose(d_all[7:], d_one[7:], rtol=1e-6, atol=1e-14), (d_all, d_one)
        exchanges = 10 if scheme == binding.SCHEME_AB else 9                      # A-B also fills the ghost layers after init
        assert lat.sim.step_count == 9 and lat.bytes_sent == exchanges * 2 * lat.face_bytes
        # checkpoint / resume across decompositions: the global state gathered from the slabs restarts a fresh set of slabs
        f9 = lat.gather(lat.get_populations(), 1)
        lat2 = slab.SlabLattice(nx, ny, nzg, tau, kT, 1.0, seed, prec, scheme=scheme, walls=walls, force=force)
        lat2.set_populations(f9, step=9)
        lat2.step(3)
        one.step(3)
        assert torch.equal(lat2.gather(lat2.get_populations(), 1), one.get_populations().cpu()), rank
        lat2.close()
        lat.close()
        one.close()
    # uniform start (rho0, u = 0) without input fields
    lat = slab.SlabLattice(40, 6, 9, tau, kT, 1.0, seed, binding.F64)
    one = binding.Rflbm(40, 6, 9, tau, kT, 1.0, seed, binding.F64)
    lat.init()
    one.init()
    lat.step(5)
    one.step(5)
    assert torch.equal(lat.gather(lat.get_populations(), 1), one.get_populations().cpu()), rank
    dist.barrier()
    if rank == 0:
        print("SLAB_DIST_OK", world, len(CASES))
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
