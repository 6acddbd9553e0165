"""Element-wise parity AT FULL SIZE for the kernel instantiations that tests/test_gpu_parity.py proves only on lattices of
a few thousand sites ("prove at full size what is proved only small"):

  * BASELINE configs[4] at its own size: 256^3 channel, fp32 storage, walls, body force, through the AUTO kernel (TMA loads
    + bulk tensor stores) - the store path differs from fp64;
  * 512^3 fp64 (byte offsets beyond 2^31, 4 x 32 x 512 TMA blocks): BGK-FLBM, the general ghost rate, and the ODD phase of
    the in-place AA scheme (the push through the per-thread column pointers);
  * rflbm_run_host pipelined against its serial form in the 32-band regime bench.py's e2e number runs in.

Method (as test_config4_sampled_parity_and_conservation_512): take the pre-collision state before and after ONE step with
rflbm_get_populations; for a few hundred sampled fluid sites x the oracle's single-site collision of the 27 populations at x
must reappear, population by population, at x + c_i after the step (Eq.7, periodic wrap), or at the site itself in slot
opp(i) when x + c_i is a solid node (halfway bounce-back, R12).  The sample contains the warp-box, tile and block edges
of the kernels, the periodic seam and the wall-adjacent layers.
"""
import gc

import numpy as np
import pytest

import oracle
from paper_2507_08820_b200 import binding, synthetic

pytestmark = pytest.mark.gpu


def torch_():
    import torch
    return torch


def need_free(gb):
    torch = torch_()
    gc.collect(); torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < gb * 1e9:
        pytest.skip(f"needs {gb} GB of free device memory")


def sample_points(nx, ny, nz, walls, seed=5, nrand=160):
    rng = np.random.default_rng(seed)
    zlo, zhi = (1, nz - 2) if walls else (0, nz - 1)
    rz = lambda: int(rng.integers(zlo, zhi + 1))
    pts = [(int(rng.integers(0, nx)), int(rng.integers(0, ny)), rz()) for _ in range(nrand)]
    xe = sorted({x for x in (0, 1, 31, 32, 33, 63, 64, 126, 127, 128, 129, 255, 256, nx - 2, nx - 1) if 0 <= x < nx})
    pts += [(x, int(rng.integers(0, ny)), rz()) for x in xe]                         # warp boxes, tiles, the x seam
    ye = sorted({y for y in (0, 7, 8, 15, 16, 17, 31, 32, ny - 1) if 0 <= y < ny})
    pts += [(int(rng.integers(0, nx)), y, z) for y in ye for z in (zlo, zhi, (zlo + zhi) // 2)]   # block rows x z faces
    pts += [(x, y, z) for x in (0, nx - 1) for y in (0, ny - 1) for z in (zlo, zhi)]             # the eight corners
    return pts


def one_step_sampled_error(sim, shape, pts, collide, walls):
    """max |S_{t+1}[i](x + c_i) - collide(S_t[.](x))[i]| over the sample (bounce-back: slot opp(i) of x itself)"""
    torch = torch_()
    nx, ny, nz = shape
    c = np.array(oracle.tables()[0], dtype=np.int64)[:, :3]                       # canonical velocities
    opp = [int(np.where((c == -c[i]).all(axis=1))[0][0]) for i in range(27)]
    t = sim.step_count
    f0 = sim.get_populations()
    P = torch.tensor(pts, device="cuda")
    g_all = f0[:, P[:, 2], P[:, 1], P[:, 0]].T.double().cpu().numpy()             # [npts, 27]
    del f0
    sim.step(1)
    f1 = sim.get_populations()
    got = torch.empty((len(pts), 27), dtype=f1.dtype, device="cuda")
    for i in range(27):
        xs, ys, zs = (P[:, 0] + int(c[i][0])) % nx, (P[:, 1] + int(c[i][1])) % ny, P[:, 2] + int(c[i][2])
        if walls:
            solid = (zs == 0) | (zs == nz - 1)
            there = f1[i, zs.clamp(0, nz - 1), ys, xs]
            back = f1[opp[i], P[:, 2], P[:, 1], P[:, 0]]
            got[:, i] = torch.where(solid, back, there)
        else:
            got[:, i] = f1[i, zs % nz, ys, xs]
    del f1
    got = got.double().cpu().numpy()
    worst = 0.0
    for k, (x, y, z) in enumerate(pts):
        want = collide(g_all[k], site=x + nx * (y + ny * z), t=t)
        worst = max(worst, float(np.abs(got[k] - want).max()))
    return worst


def test_config5_channel_fp32_sampled_parity_at_256():
    """BASELINE configs[4] at its own size through the AUTO kernel: 256^3, fp32 storage, walls, g_x = 1e-6, tau = 0.9,
    kT = 1e-4, seed 5.  One step from a thermal state; tolerance: one fp32 collision against the fp64 oracle in its
    fp32 mode (24-bit uniforms, R14) differs by a few ulp of the largest population (8/27: ulp 3e-8) through the ~60-term
    back-transform - 1e-6; the 100-step bound of north_star is 1e-5."""
    n, tau, kT, seed, g = 256, 0.9, 1e-4, 5, (1e-6, 0.0, 0.0)
    need_free(8)
    sim = binding.Rflbm(n, n, n, tau, kT, 1.0, seed, binding.F32)
    sim.set_walls_z(True)
    sim.set_force(*g)
    sim.init()
    sim.step(3)
    assert sim.last_kernel.startswith("step_kernel_tma")
    pts = sample_points(n, n, n, walls=True)
    assert any(p[2] == 1 for p in pts) and any(p[2] == n - 2 for p in pts)
    collide = lambda gg, site, t: oracle.collide_site(gg, tau, kT, seed, precision=oracle.F32, gacc=g, site=site, t=t)
    worst = one_step_sampled_error(sim, (n, n, n), pts, collide, walls=True)
    assert worst < 1e-6, worst
    d = sim.diagnostics()
    assert abs(d[0] / (n * n * (n - 2)) - 1.0) < 1e-6


@pytest.mark.parametrize("case", ["bgk", "ghost", "aa_odd", "aa_even"])
def test_512_fp64_sampled_parity_of_the_other_kernels(case):
    """512^3 fp64, tau = 0.8, kT = 1e-4, seed 11 (the bench lattice) through the TMA kernel, for the instantiations the
    headline test does not cover: BGK-FLBM (Eq.11), the ghost rate tau_g = 1.6 (Eq.21), and both phases of the in-place
    AA scheme (the step taken from t = 3 is the odd one: it pulls slot 26-q from x - c_q and pushes slot q to x + c_q)."""
    n, tau, kT, seed = 512, 0.8, 1e-4, 11
    aa = case.startswith("aa")
    need_free(95 if aa else 125)
    sim = binding.Rflbm(n, n, n, tau, kT, 1.0, seed, scheme=binding.SCHEME_AA if aa else binding.SCHEME_AB)
    sim.set_kernel_variant(binding.KERNEL_TMA)
    if case == "bgk":
        sim.set_model(binding.MODEL_BGK)
        collide = lambda gg, site, t: oracle.collide_site_bgk(gg, tau, kT, seed, site=site, t=t)
    elif case == "ghost":
        sim.set_ghost_tau(1.6)
        collide = lambda gg, site, t: oracle.collide_site_ghost(gg, tau, 1.6, kT, seed, site=site, t=t)
    else:
        collide = lambda gg, site, t: oracle.collide_site(gg, tau, kT, seed, site=site, t=t)
    sim.init()
    sim.step(4 if case == "aa_even" else 3)          # AA: steps 0, 2, 4 are the in-place (even) ones, 1, 3 the odd ones
    pts = sample_points(n, n, n, walls=False)
    worst = one_step_sampled_error(sim, (n, n, n), pts, collide, walls=False)
    assert worst < 1e-13, (case, worst)
    assert sim.last_kernel.startswith("step_kernel_tma")
    d = sim.diagnostics()
    assert abs(d[0] / n ** 3 - 1.0) < 1e-12 and max(abs(v) for v in d[1:4]) / n ** 3 < 1e-14


@pytest.mark.parametrize("shape,K,bands", [((256, 256, 512), 30, 10), ((512, 512, 512), 20, 32)])
def test_run_host_pipelined_equals_serial_at_bench_scale(shape, K, bands):
    """rflbm_run_host pipelined against its serial form where bench.py's e2e number runs: 512^3 fp64, K = 20 - 32 bands of 16
    layers, one skewed pass - and 256 x 256 x 512, K = 30 - 10 bands of 56 layers, skewed ends around whole-lattice
    launches.  Moments on the host and the final populations of the handle must equal those of the serial form bit for
    bit (the serial form is what the small tests tie to the oracle), and what came back must be the moments of the state
    the job left on the device."""
    torch = torch_()
    nx, ny, nz = shape
    need_free(130 if nx == 512 else 50)
    rho, u = synthetic.taylor_green_fields(nx, ny, nz, u0=0.02)
    rho_h = torch.from_numpy(rho).pin_memory(); u_h = torch.from_numpy(u).pin_memory()
    del rho, u
    outs = []
    for piped in (False, True):
        sim = binding.Rflbm(nx, ny, nz, 0.8, 1e-4, 1.0, 11)
        if piped:
            sim.set_copy_stream(torch.cuda.Stream())
        ro = torch.empty_like(rho_h).pin_memory(); uo = torch.empty_like(u_h).pin_memory()
        n0 = sim.launch_count
        sim.run_host(rho_h, u_h, K, ro, uo)
        launches = sim.launch_count - n0
        assert sim.step_count == K
        r_d, u_d = sim.moments()
        assert torch.equal(r_d.cpu(), ro) and torch.equal(u_d.cpu(), uo)          # what came back is the state's moments
        del r_d, u_d
        outs.append((ro, uo, sim.get_populations(), launches))
        sim.close()
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])
    assert torch.equal(outs[0][2], outs[1][2])
    # serial: init + K steps + moments; pipelined: every skewed level band by band (all K + 1 levels when K <= 24,
    # else 13 + 12 of them) plus the moments of every band
    assert outs[0][3] == K + 2 and outs[1][3] >= bands * (min(K, 24) + 1), outs[1][3]
