"""z-slab decomposition (include/rflbm.h rflbm_set_slab / rflbm_halo_*) proved on ONE GPU: two or
three slab handles whose faces the TEST carries from handle to handle (device-to-device copies) must reproduce the
single handle of the undivided lattice BIT FOR BIT — populations, moments, stress — after 1, 2 and 41 steps, in the
A-B and the in-place AA scheme, periodic and with walls, fp64 and fp32 (the oracle's order/partition independence is
pin P13; the single handle is compared with the oracle once per case as well)."""
import numpy as np
import pytest

import oracle
from paper_2507_08820_b200 import binding, synthetic

pytestmark = pytest.mark.gpu
LOW, HIGH = binding.SIDE_LOW, binding.SIDE_HIGH


def torch_():
    import torch
    return torch


def exchange(slabs):
    """what a multi-GPU caller does between steps: pack both faces of every slab, move them to the neighbours
    (periodic along z), unpack.  The move is a plain device-to-device copy into a fresh receive buffer."""
    torch = torch_()
    pend = [s.halo_pending for s in slabs]
    assert all(pend) or not any(pend)                       # slabs advance in lock step
    if not pend[0]:
        return 0
    n = len(slabs)
    sent = [(s.halo_pack(LOW), s.halo_pack(HIGH)) for s in slabs]
    for k, s in enumerate(slabs):
        below, above = slabs[(k - 1) % n], slabs[(k + 1) % n]
        recv_lo = torch.empty_like(sent[k][0]); recv_lo.copy_(sent[k][0])        # D2D "transport"
        recv_hi = torch.empty_like(sent[k][1]); recv_hi.copy_(sent[k][1])
        below.halo_unpack(HIGH, recv_lo)
        above.halo_unpack(LOW, recv_hi)
    assert not any(s.halo_pending for s in slabs)
    return sent[0][0].numel() * sent[0][0].element_size()


def ghosted(a, z0, nz, nzg):
    """layers z0-1 .. z0+nz of a global field [..., nzg, ny, nx] (periodic)"""
    idx = [(z0 - 1 + i) % nzg for i in range(nz + 2)]
    return np.ascontiguousarray(a[..., idx, :, :])


CASES = [
    # nx, ny, nzg, split, precision, scheme, walls, force, kT
    (16, 6, 8, (4, 4), binding.F64, binding.SCHEME_AB, False, None, 1e-4),
    (16, 6, 8, (4, 4), binding.F64, binding.SCHEME_AA, False, None, 1e-4),
    (40, 5, 9, (3, 1, 5), binding.F64, binding.SCHEME_AB, True, (1e-5, -2e-6, 3e-6), 1e-4),
    (40, 5, 9, (3, 1, 5), binding.F64, binding.SCHEME_AA, True, (1e-5, -2e-6, 3e-6), 1e-4),
    (130, 5, 6, (1, 5), binding.F64, binding.SCHEME_AA, True, None, 1e-4),          # a slab that is only the wall
    (130, 5, 6, (2, 2, 2), binding.F32, binding.SCHEME_AB, True, (1e-6, 0.0, 0.0), 1e-4),
    (136, 4, 7, (3, 4), binding.F32, binding.SCHEME_AA, False, None, 1e-4),
    (9, 7, 5, (5,), binding.F64, binding.SCHEME_AB, False, None, 1e-4),             # one slab: its own neighbour
    (9, 7, 5, (5,), binding.F64, binding.SCHEME_AA, False, None, 0.0),
    (34, 3, 4, (1, 1, 1, 1), binding.F64, binding.SCHEME_AA, False, None, 1e-4),     # every slab a single layer
    (34, 3, 4, (1, 1, 1, 1), binding.F64, binding.SCHEME_AB, True, None, 1e-4),
]


@pytest.mark.parametrize("nx,ny,nzg,split,prec,scheme,walls,force,kT", CASES)
def test_slabs_equal_the_undivided_lattice_bit_for_bit(nx, ny, nzg, split, prec, scheme, walls, force, kT):
    torch = torch_()
    assert sum(split) == nzg
    tau, seed = 0.8, 77
    rho, u = synthetic.smooth_random_fields(nx, ny, nzg, 19)

    def configure(s):
        if walls:
            s.set_walls_z(True)
        if force is not None:
            s.set_force(*force)

    one = binding.Rflbm(nx, ny, nzg, tau, kT, 1.0, seed, prec, scheme=scheme)
    configure(one)
    one.init(torch.from_numpy(rho), torch.from_numpy(u))
    slabs, z0 = [], 0
    for nz in split:
        s = binding.Rflbm(nx, ny, nz, tau, kT, 1.0, seed, prec, scheme=scheme, slab=(z0, nzg))
        configure(s)
        s.init(torch.from_numpy(ghosted(rho, z0, nz, nzg)), torch.from_numpy(ghosted(u, z0, nz, nzg)))
        slabs.append(s)
        z0 += nz
    assert slabs[0].halo_bytes == 9 * nx * ny * (8 if prec == binding.F64 else 4)
    if scheme == binding.SCHEME_AB:                          # A-B pulls through the ghost layers from the start
        with pytest.raises(binding.RflbmError) as e:
            slabs[0].get_populations()
        assert e.value.code == binding.ESTATE
    exchange(slabs)

    def same():
        assert torch.equal(torch.cat([s.get_populations() for s in slabs], dim=1), one.get_populations())
        r1, u1 = one.moments()
        rs, us = zip(*[s.moments() for s in slabs])
        assert torch.equal(torch.cat(rs, dim=0), r1) and torch.equal(torch.cat(us, dim=1), u1)
        assert torch.equal(torch.cat([s.stress() for s in slabs], dim=1), one.stress())

    same()
    done = 0
    for target in (1, 2, 41):
        while done < target:
            one.step(1)
            for s in slabs:
                s.step(1)
            if done == 0:
                with pytest.raises(binding.RflbmError) as e:  # the next step needs the faces first
                    slabs[0].step(1)
                assert e.value.code == binding.ESTATE
            exchange(slabs)
            done += 1
        same()
    assert all(s.step_count == 41 for s in slabs)
    # conserved sums add up over the slabs (fluid sites only)
    d1 = one.diagnostics()
    ds = np.array([s.diagnostics() for s in slabs])
    assert np.allclose(ds[:, :4].sum(axis=0), d1[:4], rtol=1e-12 if prec == binding.F64 else 1e-6, atol=1e-12)
    # and the undivided lattice is the oracle's
    ref = oracle.Ref(nx, ny, nzg, tau, kT, 1.0, seed, prec, threads=min(8, oracle.max_threads()))
    if walls:
        ref.set_walls_z(True)
    if force is not None:
        ref.set_force(*force)
    ref.init(rho, u); ref.step(41)
    err = np.abs(one.get_populations().cpu().numpy().astype(np.float64) - ref.get_populations()).max()
    assert err < (1e-11 if prec == binding.F64 else 1e-5), err


def test_slab_resume_from_exported_state_and_set_populations():
    """checkpoint / resume across a decomposition change: the populations exported by two slabs, re-cut into three
    slabs (with their ghost layers) through rflbm_set_populations, continue bit for bit."""
    torch = torch_()
    nx, ny, nzg, tau, kT, seed = 33, 6, 9, 0.7, 1e-4, 5
    one = binding.Rflbm(nx, ny, nzg, tau, kT, 1.0, seed)
    one.init(); one.step(13)
    f = one.get_populations().cpu().numpy()
    slabs, z0 = [], 0
    for nz in (2, 3, 4):
        s = binding.Rflbm(nx, ny, nz, tau, kT, 1.0, seed, scheme=binding.SCHEME_AA, slab=(z0, nzg))
        s.set_populations(torch.from_numpy(ghosted(f, z0, nz, nzg)), 13)
        slabs.append(s); z0 += nz
    exchange(slabs)
    for _ in range(6):
        one.step(1)
        for s in slabs:
            s.step(1)
        exchange(slabs)
    assert torch.equal(torch.cat([s.get_populations() for s in slabs], dim=1), one.get_populations())
    assert slabs[0].last_kernel.startswith("step_kernel_tma<TX=64>") and one.last_kernel == slabs[0].last_kernel
    with pytest.raises(binding.RflbmError) as e:
        slabs[0].step(2)                                      # one step at a time in slab mode
    assert e.value.code == binding.EINVAL


@pytest.mark.parametrize("scheme,steps", [(binding.SCHEME_AA, 1), (binding.SCHEME_AA, 2), (binding.SCHEME_AB, 1)])
def test_second_unpack_of_a_finished_side_is_a_no_op(scheme, steps):
    """after the exchange a repeated rflbm_halo_unpack must not launch again.  In the AA scheme after an odd
    step (the faces carry populations HOME into the owned boundary layer) a second unpack would overwrite nine
    populations of that layer with whatever the buffer holds by then; the slab that owns only a wall layer also
    reports finite (zero) statistics instead of 0/0."""
    torch = torch_()
    nx, ny, nzg, split = 40, 5, 8, (1, 4, 3)
    rho, u = synthetic.smooth_random_fields(nx, ny, nzg, 19)
    slabs, z0 = [], 0
    for nz in split:
        s = binding.Rflbm(nx, ny, nz, 0.8, 1e-4, 1.0, 77, binding.F64, scheme=scheme, slab=(z0, nzg))
        s.set_walls_z(True)
        s.init(torch.from_numpy(ghosted(rho, z0, nz, nzg)), torch.from_numpy(ghosted(u, z0, nz, nzg)))
        slabs.append(s)
        z0 += nz
    exchange(slabs)
    for _ in range(steps):
        for s in slabs:
            s.step(1)
        exchange(slabs)
    before = [s.get_populations().clone() for s in slabs]
    launches = [s.launch_count for s in slabs]
    junk = torch.full((9, ny, nx), 123.0, dtype=torch.float64, device="cuda")
    for s in slabs:
        s.halo_unpack(LOW, junk)
        s.halo_unpack(HIGH, junk)
        assert not s.halo_pending
    assert [s.launch_count for s in slabs] == launches
    for s in slabs:
        s.step(1)
    assert all(s.halo_pending for s in slabs)
    exchange(slabs)
    # the junk never entered: the same three slabs stepped without the extra calls give the same bits
    again, z0 = [], 0
    for nz, f in zip(split, before):
        full = torch.cat(before, dim=1)
        idx = [(z0 - 1 + i) % nzg for i in range(nz + 2)]
        s = binding.Rflbm(nx, ny, nz, 0.8, 1e-4, 1.0, 77, binding.F64, scheme=scheme, slab=(z0, nzg))
        s.set_walls_z(True)
        s.set_populations(full[:, idx].contiguous(), steps)
        again.append(s)
        z0 += nz
    exchange(again)
    for s in again:
        s.step(1)
    exchange(again)
    for a, b in zip(again, slabs):
        assert torch.equal(a.get_populations(), b.get_populations())
    d = slabs[0].diagnostics()                                # global layer 0 only: solid, no fluid site
    assert d == [0.0] * 10
