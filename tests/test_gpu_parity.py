"""GPU parity: the CUDA path through the C-ABI against the CPU oracle, element by element on identical
seeded inputs (configs[0] of BASELINE.json and ragged / walled / forced / fp32 variants)."""
import numpy as np
import pytest

import oracle
from paper_2507_08820_b200 import binding, synthetic

pytestmark = pytest.mark.gpu

TOL64 = 1e-11   # north_star: fp64 populations within 1e-11 max-abs after 100 steps
TOL32 = 1e-5    # north_star: fp32 storage within 1e-5
NT = min(8, oracle.max_threads())


def torch_():
    import torch
    return torch


def make_pair(nx, ny, nz, tau, kT, seed, precision=binding.F64, walls=False, force=None, rho0=1.0):
    sim = binding.Rflbm(nx, ny, nz, tau, kT, rho0, seed, precision)
    ref = oracle.Ref(nx, ny, nz, tau, kT, rho0, seed, precision, threads=NT)
    if walls:
        sim.set_walls_z(True); ref.set_walls_z(True)
    if force is not None:
        sim.set_force(*force); ref.set_force(*force)
    return sim, ref


def init_pair(sim, ref, fields=None):
    torch = torch_()
    if fields is None:
        sim.init(); ref.init()
    else:
        rho, u = fields
        sim.init(torch.from_numpy(rho), torch.from_numpy(u)); ref.init(rho, u)


def pops(sim):
    return sim.get_populations().cpu().numpy().astype(np.float64)


def test_config1_rng_stream_bit_exact_and_normals():
    sim, ref = make_pair(16, 16, 16, 1.0, 1e-4, 42)
    for step in (0, 1, 99, 2 ** 32 + 5):
        w_g, n_g = sim.debug_rng(step)
        w_r, n_r = ref.debug_rng(step)
        assert np.array_equal(w_g.cpu().numpy().view(np.uint32), w_r)          # bit exact
        d = np.abs(n_g.cpu().numpy() - n_r)
        assert d.max() < 2e-14, d.max()                                         # libm vs CUDA math: a few ulp of 6.8


def test_config1_populations_100_steps():
    sim, ref = make_pair(16, 16, 16, 1.0, 1e-4, 42)
    init_pair(sim, ref)
    assert np.abs(pops(sim) - ref.get_populations()).max() < 1e-16
    for chunk in (1, 9, 90):
        sim.step(chunk); ref.step(chunk)
        err = np.abs(pops(sim) - ref.get_populations()).max()
        assert err < TOL64, (sim.step_count, err)
    assert sim.step_count == 100 == ref.step_count
    # conservation and equipartition (config 1 checks)
    d = sim.diagnostics()
    n = 16 ** 3
    assert abs(d[0] - n) < 1e-13 * n * 10
    assert max(abs(v) for v in d[1:4]) / n < 1e-15
    dr = ref.diagnostics()
    assert np.abs(np.array(d) - dr).max() < 1e-9                              # mass sum of 4096 sites
    rho, u = sim.moments()
    u = u.cpu().numpy()
    assert np.abs((u ** 2).mean(axis=(1, 2, 3)) / 1e-4 - 1.0).max() < 0.05
    rr, ur = ref.moments()
    assert np.abs(rho.cpu().numpy() - rr).max() < 1e-11 and np.abs(u - ur).max() < 1e-11


@pytest.mark.parametrize("shape,tau,kT", [((5, 7, 9), 0.7, 1e-4), ((130, 6, 5), 0.51, 1e-4), ((40, 9, 4), 50.0, 1e-4),
                                          ((1, 1, 1), 0.8, 1e-4), ((33, 33, 2), 0.9, 0.0), ((300, 3, 3), 1.5, 1e-3)])
def test_ragged_shapes_smooth_init(shape, tau, kT):
    """several blocks plus a ragged tail in x and y, non-trivial (rho,u) through rflbm_init"""
    nx, ny, nz = shape
    sim, ref = make_pair(nx, ny, nz, tau, kT, 7)
    init_pair(sim, ref, synthetic.smooth_random_fields(nx, ny, nz, 5))
    assert np.abs(pops(sim) - ref.get_populations()).max() < 1e-15
    sim.step(30); ref.step(30)
    assert np.abs(pops(sim) - ref.get_populations()).max() < TOL64


def test_walls_and_force_fp64():
    nx, ny, nz = 12, 10, 11
    sim, ref = make_pair(nx, ny, nz, 0.9, 1e-4, 5, walls=True, force=(1e-5, -2e-6, 3e-6))
    init_pair(sim, ref, synthetic.smooth_random_fields(nx, ny, nz, 9))
    assert np.abs(pops(sim) - ref.get_populations()).max() < 1e-15
    sim.step(60); ref.step(60)
    assert np.abs(pops(sim) - ref.get_populations()).max() < TOL64
    rho, u = sim.moments()
    rr, ur = ref.moments()
    assert np.abs(rho.cpu().numpy() - rr).max() < 1e-11 and np.abs(u.cpu().numpy() - ur).max() < 1e-11
    assert (rho.cpu().numpy()[0] == 0).all() and (rho.cpu().numpy()[-1] == 0).all()
    assert np.abs(np.array(sim.diagnostics()) - ref.diagnostics()).max() < 1e-10


def test_walls_minimal_nz3_and_force_only_periodic():
    sim, ref = make_pair(6, 5, 3, 0.8, 1e-4, 3, walls=True)
    init_pair(sim, ref)
    sim.step(20); ref.step(20)
    assert np.abs(pops(sim) - ref.get_populations()).max() < TOL64
    sim, ref = make_pair(6, 5, 4, 0.8, 0.0, 3, force=(1e-6, 0.0, -2e-6))
    init_pair(sim, ref)
    sim.step(10); ref.step(10)
    assert np.abs(pops(sim) - ref.get_populations()).max() < 1e-14
    d = sim.diagnostics()
    assert abs(d[1] / (120 * 1e-6 * 10.5) - 1) < 1e-11                       # momentum grows by N rho0 g per step


def test_fp32_channel_parity_100_steps():
    """config 5 at test size: 16x16x18 channel, fp32 storage, walls, body force, 100 steps."""
    nx, ny, nz = 16, 16, 18
    sim, ref = make_pair(nx, ny, nz, 0.9, 1e-4, 5, precision=binding.F32, walls=True, force=(1e-6, 0.0, 0.0))
    init_pair(sim, ref)
    sim.step(100); ref.step(100)
    err = np.abs(pops(sim) - ref.get_populations()).max()
    assert err < TOL32, err
    w_g, n_g = sim.debug_rng(17)
    w_r, n_r = ref.debug_rng(17)
    assert np.array_equal(w_g.cpu().numpy().view(np.uint32), w_r)
    nerr = np.abs(n_g.cpu().numpy().astype(np.float64) - n_r).max()
    # R14: the fp32 Box-Muller runs on the special-function unit; DESIGN.md states 1e-5 on a normal (derived bound
    # 4e-6: lg2.approx 2^-22 absolute at the radius R = 0.044 where the series takes over, sin/cos.approx 2^-21.4
    # times |R| <= 5.9; measured 1.8e-6 over 5.6e6 draws).  A population sees sqrt(3 kT rho) w_i/b_k times that.
    print(f"fp32 parity after 100 steps: max|f_gpu - f_oracle| = {err:.3e} (tolerance {TOL32:g}); "
          f"max|normal_gpu - normal_oracle| = {nerr:.3e} (tolerance 1e-5)")
    assert nerr < 1e-5, nerr


def test_fp32_periodic_parity():
    sim, ref = make_pair(20, 12, 7, 0.7, 1e-4, 8, precision=binding.F32)
    init_pair(sim, ref, synthetic.smooth_random_fields(20, 12, 7, 2))
    sim.step(100); ref.step(100)
    err = np.abs(pops(sim) - ref.get_populations()).max()
    print(f"fp32 periodic parity after 100 steps: max|f_gpu - f_oracle| = {err:.3e} (tolerance {TOL32:g})")
    assert err < TOL32, err


def test_set_get_roundtrip_and_resume_bit_exact():
    torch = torch_()
    c, w = oracle.tables()[:2]
    for walls in (False, True):
        nx, ny, nz = 9, 6, 5
        f = synthetic.random_population_field(nx, ny, nz, 4, w)
        sim, ref = make_pair(nx, ny, nz, 0.8, 1e-4, 11, walls=walls)
        sim.set_populations(torch.from_numpy(f), 17)
        ref.set_populations(f, 17)
        assert np.array_equal(pops(sim), f)                                    # import -> export is the identity
        sim.step(25); ref.step(25)
        assert sim.step_count == 42
        assert np.abs(pops(sim) - ref.get_populations()).max() < TOL64
    # step(50)+step(50) == step(100), and resume from an exported state, bit for bit
    a = binding.Rflbm(16, 8, 8, 0.8, 1e-4, 1.0, 3); a.init(); a.step(100)
    b = binding.Rflbm(16, 8, 8, 0.8, 1e-4, 1.0, 3); b.init(); b.step(50); b.step(50)
    c2 = binding.Rflbm(16, 8, 8, 0.8, 1e-4, 1.0, 3); c2.set_populations(b.get_populations() * 0 + 1, 0)
    c2.init(); c2.step(50)
    d = binding.Rflbm(16, 8, 8, 0.8, 1e-4, 1.0, 3); d.set_populations(c2.get_populations(), c2.step_count); d.step(50)
    fa = a.get_populations()
    assert torch.equal(fa, b.get_populations()) and torch.equal(fa, d.get_populations())


def test_kT0_equilibrium_fixed_point_and_error_codes():
    torch = torch_()
    sim = binding.Rflbm(8, 8, 8, 0.6, 0.0)
    rho, u = synthetic.uniform_fields(8, 8, 8, 1.2, (0.05, -0.02, 0.08))
    sim.init(torch.from_numpy(rho), torch.from_numpy(u))
    f0 = sim.get_populations().clone()
    sim.step(5)
    assert (sim.get_populations() - f0).abs().max().item() < 1e-15
    with pytest.raises(binding.RflbmError) as e:
        sim.set_walls_z(True)                                                  # after init
    assert e.value.code == binding.ESTATE
    with pytest.raises(binding.RflbmError) as e:
        sim.step(-1)
    assert e.value.code == binding.EINVAL
    fresh = binding.Rflbm(4, 4, 4, 1.0, 0.0)
    with pytest.raises(binding.RflbmError) as e:
        fresh.moments()
    assert e.value.code == binding.ESTATE


def test_run_host_matches_device_path():
    torch = torch_()
    nx, ny, nz = 24, 10, 6
    rho, u = synthetic.smooth_random_fields(nx, ny, nz, 12)
    sim, ref = make_pair(nx, ny, nz, 0.8, 1e-4, 21)
    rho_h = torch.from_numpy(rho).pin_memory(); u_h = torch.from_numpy(u).pin_memory()
    ro = torch.empty_like(rho_h).pin_memory(); uo = torch.empty_like(u_h).pin_memory()
    sim.run_host(rho_h, u_h, 20, ro, uo)
    ref.init(rho, u); ref.step(20)
    rr, ur = ref.moments()
    assert np.abs(ro.numpy() - rr).max() < 1e-11 and np.abs(uo.numpy() - ur).max() < 1e-11
    assert sim.launch_count == 22                                             # init + 20 steps + moments


@pytest.mark.parametrize("shape,prec,walls,force,nsteps", [
    ((24, 10, 6), binding.F64, False, None, 20), ((40, 6, 70), binding.F64, True, (1e-5, 0.0, 2e-6), 9),
    ((130, 5, 33), binding.F32, False, None, 13), ((9, 4, 3), binding.F64, False, None, 5),
    ((36, 4, 40), binding.F64, False, None, 0), ((36, 4, 40), binding.F64, True, None, 1),
    ((40, 6, 70), binding.F64, True, (1e-5, 0.0, 2e-6), 30), ((36, 4, 40), binding.F64, False, None, 25),
    ((9, 4, 5), binding.F64, False, None, 40), ((130, 5, 200), binding.F32, False, None, 26),
    ((33, 4, 64), binding.F64, False, None, 24), ((32, 3, 129), binding.F64, True, None, 31)])
def test_run_host_pipelined_is_bit_identical_to_serial(shape, prec, walls, force, nsteps):
    """rflbm_run_host with a copy stream (time-skewed along z: every band of uploaded layers advances every level, the
    ring's seam is closed at the end, moments leave behind the last level; more than 24 steps: skewed ends around
    whole-lattice launches) against the serial form of the same call: bit-identical moments AND bit-identical final
    state of the handle; bands of 1..7 layers with a ragged last band, walls, force, fp32, 0 and 1 steps, more steps
    than layers."""
    torch = torch_()
    nx, ny, nz = shape
    dt = torch.float64 if prec == binding.F64 else torch.float32
    rho, u = synthetic.smooth_random_fields(nx, ny, nz, 12)
    rho_h = torch.from_numpy(rho).to(dt).pin_memory(); u_h = torch.from_numpy(u).to(dt).pin_memory()
    outs = []
    for piped in (False, True):
        sim = binding.Rflbm(nx, ny, nz, 0.8, 1e-4, 1.0, 21, prec)
        if walls:
            sim.set_walls_z(True)
        if force is not None:
            sim.set_force(*force)
        if piped:
            sim.set_copy_stream(torch.cuda.Stream())
        ro = torch.empty_like(rho_h).pin_memory(); uo = torch.empty_like(u_h).pin_memory()
        sim.run_host(rho_h, u_h, nsteps, ro, uo)
        assert sim.step_count == nsteps
        sim.step(3)                                           # the handle continues from the state the job left
        outs.append((ro.clone(), uo.clone(), sim.get_populations().clone(), sim.launch_count))
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])
    assert torch.equal(outs[0][2], outs[1][2])
    if nz >= 3:
        assert outs[1][3] > outs[0][3]                        # the pipelined job really ran chunk by chunk
    # uniform start without upload
    a = binding.Rflbm(nx, ny, nz, 0.8, 1e-4, 1.0, 21, prec); b = binding.Rflbm(nx, ny, nz, 0.8, 1e-4, 1.0, 21, prec)
    b.set_copy_stream(torch.cuda.Stream())
    res = []
    for sim in (a, b):
        ro = torch.empty_like(rho_h).pin_memory(); uo = torch.empty_like(u_h).pin_memory()
        sim.run_host(None, None, nsteps, ro, uo)
        res.append((ro, uo))
    assert torch.equal(res[0][0], res[1][0]) and torch.equal(res[0][1], res[1][1])


@pytest.mark.parametrize("shape,walls,force,kT", [((128, 4, 3), False, None, 1e-4), ((256, 5, 4), True, (1e-5, 2e-6, -3e-6), 1e-4),
                                                 ((300, 3, 3), False, None, 1e-4), ((130, 18, 5), True, None, 0.0),
                                                 ((384, 20, 2), False, (1e-6, 0.0, 0.0), 1e-3),
                                                 ((129, 7, 5), False, None, 1e-4), ((131, 19, 4), True, (1e-5, 0.0, 0.0), 1e-4),
                                                 ((32, 9, 4), False, None, 1e-4), ((33, 35, 3), True, None, 1e-4),
                                                 ((64, 17, 3), False, (1e-6, 1e-6, 0.0), 1e-4), ((100, 6, 5), True, None, 1e-4),
                                                 ((127, 33, 2), False, None, 1e-4),
                                                 ((128, 1, 1), False, None, 1e-4), ((64, 2, 1), False, None, 1e-4),
                                                 ((33, 1, 2), False, (1e-6, 0.0, 1e-6), 1e-4), ((32, 1, 3), True, None, 1e-4)])
def test_tma_kernel_matches_plain_kernel_and_oracle(shape, walls, force, kT):
    """The TMA-staged step kernel (fp64; tiles of 128, 64 or 32 sites; any nx >= 32, odd ones included: the internal
    row pitch is padded) against the plain kernel (bit for bit: same arithmetic) and the oracle; shapes span several
    x tiles, a ragged last tile, > rows_per_block rows, ragged row groups of the narrow tiles, walls."""
    torch = torch_()
    nx, ny, nz = shape
    fields = synthetic.smooth_random_fields(nx, ny, nz, 13)
    outs = {}
    for variant in (binding.KERNEL_TMA, binding.KERNEL_PLAIN):
        sim, ref = make_pair(nx, ny, nz, 0.8, kT, 17, walls=walls, force=force)
        sim.set_kernel_variant(variant)
        init_pair(sim, ref, fields)
        sim.step(12)
        outs[variant] = sim.get_populations()
    ref.step(12)
    assert torch.equal(outs[binding.KERNEL_TMA], outs[binding.KERNEL_PLAIN])
    assert np.abs(outs[binding.KERNEL_TMA].cpu().numpy() - ref.get_populations()).max() < TOL64


@pytest.mark.parametrize("shape,walls,force,kT", [((128, 5, 4), False, None, 1e-4), ((260, 18, 5), True, (1e-5, 2e-6, -3e-6), 1e-4),
                                                 ((384, 3, 3), False, (1e-6, 0.0, 0.0), 0.0), ((130, 7, 5), False, None, 1e-4),
                                                 ((131, 6, 4), True, None, 1e-4), ((33, 19, 3), False, None, 1e-4),
                                                 ((66, 9, 5), True, (1e-6, 0.0, 0.0), 1e-4)])
def test_tma_kernel_fp32_matches_plain_kernel_and_oracle(shape, walls, force, kT):
    """fp32 instantiation of the TMA kernel (any nx >= 32): 136-float boxes at TX = 128, 4-element halo."""
    torch = torch_()
    nx, ny, nz = shape
    fields = synthetic.smooth_random_fields(nx, ny, nz, 14)
    outs = {}
    for variant in (binding.KERNEL_TMA, binding.KERNEL_PLAIN):
        sim, ref = make_pair(nx, ny, nz, 0.8, kT, 19, precision=binding.F32, walls=walls, force=force)
        sim.set_kernel_variant(variant)
        init_pair(sim, ref, fields)
        sim.step(40)
        outs[variant] = sim.get_populations()
    ref.step(40)
    assert torch.equal(outs[binding.KERNEL_TMA], outs[binding.KERNEL_PLAIN])
    assert np.abs(outs[binding.KERNEL_TMA].cpu().numpy().astype(np.float64) - ref.get_populations()).max() < TOL32


def test_tma_variant_rejected_only_below_32_and_auto_never_takes_the_plain_kernel_with_noise():
    for nx, prec in ((31, binding.F64), (8, binding.F32)):       # shorter than the narrowest tile
        sim = binding.Rflbm(nx, 4, 4, 0.8, 1e-4, precision=prec)
        sim.set_kernel_variant(binding.KERNEL_TMA)
        sim.init()
        with pytest.raises(binding.RflbmError) as e:
            sim.step(1)
        assert e.value.code == binding.EINVAL
    # AUTO with noise: every lattice with nx >= 32 runs the TMA kernel (the internal row pitch is padded, so odd nx
    # qualifies); kT = 0 keeps the plain kernel (pure streaming, where it is the faster one)
    # tile width: fewest idle threads on the ragged last tile, widest on a tie
    for nx, prec, name in ((32, binding.F64, "TX=32"), (33, binding.F32, "TX=64"), (64, binding.F64, "TX=64"),
                           (96, binding.F64, "TX=32"), (127, binding.F32, "TX=128"), (129, binding.F64, "TX=32"),
                           (130, binding.F32, "TX=32"), (200, binding.F64, "TX=32"), (320, binding.F64, "TX=64"), (511, binding.F64, "TX=128")):
        sim = binding.Rflbm(nx, 3, 3, 0.8, 1e-4, precision=prec)
        assert sim.last_kernel == ""
        sim.init(); sim.step(2)
        assert sim.last_kernel == f"step_kernel_tma<{name}>", (nx, sim.last_kernel)
    sim = binding.Rflbm(16, 3, 3, 0.8, 1e-4); sim.init(); sim.step(1)
    assert sim.last_kernel == "step_kernel"
    sim = binding.Rflbm(256, 3, 3, 0.8, 0.0); sim.init(); sim.step(1)
    assert sim.last_kernel == "step_kernel"


@pytest.mark.parametrize("shape,prec,walls,kT,tau", [((16, 16, 16), binding.F64, False, 1e-4, 1.0), ((5, 7, 9), binding.F64, False, 1e-4, 0.55),
                                                    ((132, 6, 5), binding.F64, True, 1e-4, 0.8), ((256, 4, 3), binding.F64, False, 0.0, 3.0),
                                                    ((20, 12, 7), binding.F32, False, 1e-4, 0.7), ((136, 5, 6), binding.F32, True, 1e-4, 0.9)])
def test_bgk_flbm_model_matches_oracle(shape, prec, walls, kT, tau):
    """BGK-FLBM (Eq.11), the paper's comparison model: GPU mode-space form against the oracle's population-space
    form, 100 steps, plain and (where the lattice allows) TMA kernel bit-identical."""
    torch = torch_()
    nx, ny, nz = shape
    fields = synthetic.smooth_random_fields(nx, ny, nz, 23)
    outs = []
    variants = [binding.KERNEL_PLAIN] + ([binding.KERNEL_TMA] if nx >= 32 else [])
    for variant in variants:
        sim, ref = make_pair(nx, ny, nz, tau, kT, 29, precision=prec, walls=walls)
        sim.set_model(binding.MODEL_BGK); ref.set_model(oracle.MODEL_BGK)
        sim.set_kernel_variant(variant)
        init_pair(sim, ref, fields)
        sim.step(100)
        outs.append(sim.get_populations())
    ref.step(100)
    if len(outs) == 2:
        assert torch.equal(outs[0], outs[1])
    err = np.abs(outs[0].cpu().numpy().astype(np.float64) - ref.get_populations()).max()
    assert err < (TOL64 if prec == binding.F64 else TOL32), err
    d = sim.diagnostics()
    assert abs(d[0] - ref.diagnostics()[0]) < (1e-9 if prec == binding.F64 else 1e-2)


def test_bgk_model_refuses_force_and_differs_from_reg():
    sim = binding.Rflbm(8, 8, 8, 0.8, 1e-4, 1.0, 3)
    sim.set_model(binding.MODEL_BGK)
    with pytest.raises(binding.RflbmError) as e:
        sim.set_force(1e-6, 0.0, 0.0)
    assert e.value.code == binding.EINVAL
    with pytest.raises(binding.RflbmError):
        sim.set_model(5)
    sim.init(); sim.step(20)
    reg = binding.Rflbm(8, 8, 8, 0.8, 1e-4, 1.0, 3)
    reg.init(); reg.step(20)
    assert (sim.get_populations() - reg.get_populations()).abs().max().item() > 1e-6


@pytest.mark.parametrize("prec,walls", [(binding.F64, False), (binding.F64, True), (binding.F32, True)])
def test_stress_observable_matches_oracle(prec, walls):
    nx, ny, nz = 40, 9, 6
    sim, ref = make_pair(nx, ny, nz, 0.8, 1e-4, 13, precision=prec, walls=walls, force=(1e-6, 0.0, 0.0) if walls else None)
    init_pair(sim, ref, synthetic.smooth_random_fields(nx, ny, nz, 6))
    sim.step(15); ref.step(15)
    d = np.abs(sim.stress().cpu().numpy().astype(np.float64) - ref.stress()).max()
    assert d < (1e-12 if prec == binding.F64 else 1e-5), d


@pytest.mark.parametrize("shape,prec,scheme,walls,steps", [
    ((40, 9, 6), binding.F64, binding.SCHEME_AB, False, 15), ((130, 7, 5), binding.F64, binding.SCHEME_AA, True, 3),
    ((130, 7, 5), binding.F32, binding.SCHEME_AA, True, 4), ((33, 33, 3), binding.F32, binding.SCHEME_AB, True, 6),
    ((5, 3, 2), binding.F64, binding.SCHEME_AB, False, 2)])
def test_snapshot_equals_moments_plus_stress_bit_for_bit(shape, prec, scheme, walls, steps):
    """rflbm_snapshot (rho, rho u and Pi_ab saved together) is one gather with ten stores; it must write
    exactly what rflbm_moments and rflbm_stress write - which the tests above tie to the oracle - in both schemes and AA
    phases, with walls (solid layers: zeros) and a body force (u carries g/2), and launch one kernel."""
    torch = torch_()
    nx, ny, nz = shape
    sim = binding.Rflbm(nx, ny, nz, 0.8, 1e-4, 1.0, 13, prec, scheme=scheme)
    if walls:
        sim.set_walls_z(True)
        sim.set_force(1e-6, -3e-6, 0.0)
    rho, u = synthetic.smooth_random_fields(nx, ny, nz, 6)
    sim.init(torch.from_numpy(rho), torch.from_numpy(u))
    sim.step(steps)
    r1, u1 = sim.moments()
    p1 = sim.stress()
    n0 = sim.launch_count
    r2, u2, p2 = sim.snapshot()
    assert sim.launch_count == n0 + 1
    assert torch.equal(r1, r2) and torch.equal(u1, u2) and torch.equal(p1, p2)
    if walls:
        assert float(r2[0].abs().max()) == 0.0 and float(p2[:, -1].abs().max()) == 0.0
    fresh = binding.Rflbm(4, 4, 4, 1.0, 0.0)
    with pytest.raises(binding.RflbmError) as e:
        fresh.snapshot()
    assert e.value.code == binding.ESTATE


@pytest.mark.parametrize("shape,prec,walls,force,kT,variant", [
    ((16, 16, 16), binding.F64, False, None, 1e-4, binding.KERNEL_AUTO),
    ((5, 7, 9), binding.F64, True, (1e-5, -2e-6, 3e-6), 1e-4, binding.KERNEL_AUTO),
    ((33, 6, 5), binding.F32, True, (1e-6, 0.0, 0.0), 1e-4, binding.KERNEL_AUTO),
    ((1, 1, 1), binding.F64, False, None, 1e-4, binding.KERNEL_AUTO),
    ((130, 18, 5), binding.F64, True, (1e-5, 2e-6, -3e-6), 1e-4, binding.KERNEL_TMA),
    ((256, 20, 3), binding.F64, False, None, 1e-4, binding.KERNEL_TMA),
    ((300, 3, 4), binding.F64, False, None, 0.0, binding.KERNEL_TMA),
    ((136, 5, 6), binding.F32, True, None, 1e-4, binding.KERNEL_TMA),
    ((256, 4, 3), binding.F64, False, None, 1e-4, binding.KERNEL_PLAIN)])
def test_aa_in_place_scheme_is_bit_identical_to_ab_and_matches_oracle(shape, prec, walls, force, kT, variant):
    """AA (one buffer, in place) against A-B: same arithmetic, so bit-identical observable state after even AND
    odd step counts (the export gathers differently in the two AA phases), moments and stress included."""
    torch = torch_()
    nx, ny, nz = shape
    fields = synthetic.smooth_random_fields(nx, ny, nz, 31)
    sims = {}
    for scheme in (binding.SCHEME_AB, binding.SCHEME_AA):
        sim = binding.Rflbm(nx, ny, nz, 0.8, kT, 1.0, 37, prec, scheme=scheme)
        if walls:
            sim.set_walls_z(True)
        if force is not None:
            sim.set_force(*force)
        sim.set_kernel_variant(variant)
        sim.init(torch.from_numpy(fields[0]), torch.from_numpy(fields[1]))
        sims[scheme] = sim
    ab, aa = sims[binding.SCHEME_AB], sims[binding.SCHEME_AA]
    assert aa.workspace.numel() < 0.52 * ab.workspace.numel() + 40000
    assert torch.equal(ab.get_populations(), aa.get_populations())
    ref = oracle.Ref(nx, ny, nz, 0.8, kT, 1.0, 37, prec, threads=NT)
    if walls:
        ref.set_walls_z(True)
    if force is not None:
        ref.set_force(*force)
    ref.init(*fields)
    for n in (1, 1, 5, 12, 21):                       # odd and even totals: 1, 2, 7, 19, 40
        ab.step(n); aa.step(n); ref.step(n)
        assert torch.equal(ab.get_populations(), aa.get_populations()), ab.step_count
        ra, ua = aa.moments(); rb, ub = ab.moments()
        assert torch.equal(ra, rb) and torch.equal(ua, ub) and torch.equal(aa.stress(), ab.stress())
        assert np.allclose(aa.diagnostics(), ab.diagnostics(), rtol=1e-12, atol=1e-12)   # atomics: order varies
    err = np.abs(aa.get_populations().cpu().numpy().astype(np.float64) - ref.get_populations()).max()
    assert err < (TOL64 if prec == binding.F64 else TOL32), err


def test_aa_set_get_roundtrip_resume_and_bgk():
    torch = torch_()
    w = oracle.tables()[1]
    nx, ny, nz = 9, 6, 5
    f = synthetic.random_population_field(nx, ny, nz, 4, w)
    for walls in (False, True):
        sim = binding.Rflbm(nx, ny, nz, 0.8, 1e-4, 1.0, 11, scheme=binding.SCHEME_AA)
        ref = oracle.Ref(nx, ny, nz, 0.8, 1e-4, 1.0, 11, threads=NT)
        if walls:
            sim.set_walls_z(True); ref.set_walls_z(True)
        sim.set_populations(torch.from_numpy(f), 17); ref.set_populations(f, 17)
        assert np.array_equal(pops(sim), f)
        sim.step(7); ref.step(7)                      # odd phase
        assert np.abs(pops(sim) - ref.get_populations()).max() < TOL64
        mid = sim.get_populations().clone()
        sim.step(6); ref.step(6)
        assert np.abs(pops(sim) - ref.get_populations()).max() < TOL64
        # resume from the odd-phase export in a fresh handle: bit exact
        sim2 = binding.Rflbm(nx, ny, nz, 0.8, 1e-4, 1.0, 11, scheme=binding.SCHEME_AA)
        if walls:
            sim2.set_walls_z(True)
        sim2.set_populations(mid, 24); sim2.step(6)
        assert torch.equal(sim2.get_populations(), sim.get_populations())
    a = binding.Rflbm(20, 8, 6, 0.7, 1e-4, 1.0, 3, scheme=binding.SCHEME_AA); a.set_model(binding.MODEL_BGK); a.init(); a.step(15)
    b = binding.Rflbm(20, 8, 6, 0.7, 1e-4, 1.0, 3); b.set_model(binding.MODEL_BGK); b.init(); b.step(15)
    assert torch.equal(a.get_populations(), b.get_populations())


@pytest.mark.parametrize("shape,prec,walls,kT,tau,tau_g,scheme", [
    ((16, 16, 16), binding.F64, False, 1e-4, 0.8, 1.6, binding.SCHEME_AB), ((5, 7, 9), binding.F64, True, 1e-4, 0.55, 0.7, binding.SCHEME_AA),
    ((132, 6, 5), binding.F64, True, 1e-4, 3.0, 0.6, binding.SCHEME_AB), ((256, 4, 3), binding.F64, False, 0.0, 0.9, 2.5, binding.SCHEME_AA),
    ((136, 5, 6), binding.F32, False, 1e-4, 0.8, 1.3, binding.SCHEME_AB)])
def test_general_ghost_rate_matches_oracle(shape, prec, walls, kT, tau, tau_g, scheme):
    """omega_g != 1 (Eq.21 live): GPU closed-form pair sums against the oracle's literal tensor recursion."""
    torch = torch_()
    nx, ny, nz = shape
    fields = synthetic.smooth_random_fields(nx, ny, nz, 41)
    sim = binding.Rflbm(nx, ny, nz, tau, kT, 1.0, 43, prec, scheme=scheme)
    ref = oracle.Ref(nx, ny, nz, tau, kT, 1.0, 43, prec, threads=NT)
    if walls:
        sim.set_walls_z(True); ref.set_walls_z(True)
    sim.set_ghost_tau(tau_g); ref.set_ghost_tau(tau_g)
    init_pair(sim, ref, fields)
    sim.step(61); ref.step(61)
    err = np.abs(pops(sim) - ref.get_populations()).max()
    assert err < (TOL64 if prec == binding.F64 else TOL32), err
    with pytest.raises(binding.RflbmError):
        sim.set_force(1e-6, 0.0, 0.0)
    # tau_g = 1 is the default path bit for bit
    a = binding.Rflbm(12, 6, 5, 0.8, 1e-4, 1.0, 3); a.set_ghost_tau(1.0); a.init(); a.step(9)
    b = binding.Rflbm(12, 6, 5, 0.8, 1e-4, 1.0, 3); b.init(); b.step(9)
    assert torch.equal(a.get_populations(), b.get_populations())


def test_two_handles_on_their_own_streams_do_not_interfere():
    """Every call enqueues on the stream given to the handle (rflbm_set_stream): two simulations stepped in an
    interleaved fashion on two non-default streams give the same bits as each one alone."""
    torch = torch_()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    solo = []
    for seed in (5, 6):
        sim = binding.Rflbm(140, 9, 7, 0.8, 1e-4, 1.0, seed)
        sim.init(); sim.step(24)
        solo.append(sim.get_populations().clone())
    torch.cuda.synchronize()
    a = binding.Rflbm(140, 9, 7, 0.8, 1e-4, 1.0, 5, stream=s1)
    b = binding.Rflbm(140, 9, 7, 0.8, 1e-4, 1.0, 6, stream=s2, scheme=binding.SCHEME_AA)
    with torch.cuda.stream(s1):
        a.init()
    with torch.cuda.stream(s2):
        b.init()
    for _ in range(8):
        a.step(3); b.step(3)
    with torch.cuda.stream(s1):
        fa = a.get_populations()
    with torch.cuda.stream(s2):
        fb = b.get_populations()
    torch.cuda.synchronize()
    assert torch.equal(fa, solo[0]) and torch.equal(fb, solo[1])
    assert a.launch_count == 26 and b.step_count == 24


@pytest.mark.parametrize("nth", [1, 5, 8, 11, 29, 31, 40])
def test_run_host_pipelined_failure_leaves_no_state(nth):
    """ADVICE r2 / VERDICT r2 item 6: every CUDA call of the pipelined rflbm_run_host is checked; a job in which one of
    them fails (event creation, the first record, an upload, a wait, the download side: rflbm_debug_inject_failure makes
    the nth checked call report an error) returns ECUDA with the text of that first failure and leaves the handle
    WITHOUT a state (ESTATE on the next rflbm_step) instead of claiming t = nsteps; both streams are quiet and no
    sticky error is left, and the same handle then runs a proper job to the result a fresh handle gives."""
    torch = torch_()
    nx, ny, nz = 36, 4, 40
    sim = binding.Rflbm(nx, ny, nz, 0.8, 1e-4, 1.0, 21)
    sim.set_copy_stream(torch.cuda.Stream())
    sim.init()
    sim.step(2)
    rho, u = synthetic.smooth_random_fields(nx, ny, nz, 12)
    rho_h = torch.from_numpy(rho).pin_memory(); u_h = torch.from_numpy(u).pin_memory()
    ro = torch.empty(nz, ny, nx, dtype=torch.float64).pin_memory(); uo = torch.empty(3, nz, ny, nx, dtype=torch.float64).pin_memory()
    sim.debug_inject_failure(nth)
    with pytest.raises(binding.RflbmError) as e:
        sim.run_host(rho_h, u_h, 5, ro, uo)
    assert e.value.code == binding.ECUDA and "unknown error" in str(e.value).lower()
    with pytest.raises(binding.RflbmError) as e:
        sim.step(1)
    assert e.value.code == binding.ESTATE
    with pytest.raises(binding.RflbmError) as e:
        sim.moments()
    assert e.value.code == binding.ESTATE
    assert sim.step_count == 0
    torch.cuda.synchronize()                                                   # no sticky error left behind
    sim.run_host(rho_h, u_h, 5, ro, uo)                                        # the hook disarmed itself
    fresh = binding.Rflbm(nx, ny, nz, 0.8, 1e-4, 1.0, 21)
    ro2 = torch.empty_like(ro).pin_memory(); uo2 = torch.empty_like(uo).pin_memory()
    fresh.run_host(rho_h, u_h, 5, ro2, uo2)
    assert torch.equal(ro, ro2) and torch.equal(uo, uo2) and sim.step_count == 5
