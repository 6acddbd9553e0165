"""GPU runs of BASELINE.json configs[1..4] through the C-ABI (configs[0] is tests/test_gpu_parity.py).

configs[1] 64^3 equipartition + flat structure factor, configs[2] 256^3 Taylor-Green decay, configs[3] 512^3 in the
launch configuration bench.py times (TMA kernel): sampled outputs against the oracle's single-site collision plus
conservation, configs[4] 256^3 fp32 channel against the start-up series of the oracle pin P12.
Statistics are computed test-side (numpy / torch on the downloaded moments); the expected values are the closed
forms that also pin the oracle."""
import numpy as np
import pytest

import oracle
from analysis import fit_decay_rate, shell_spectrum
from paper_2507_08820_b200 import binding, synthetic

pytestmark = pytest.mark.gpu


def torch_():
    import torch
    return torch


@pytest.mark.parametrize("tau", [0.6, 1.0])
def test_config2_equipartition_and_structure_factor_64(tau):
    """<u_a^2> rho0/kT = 1 +- 0.005 and S_rho(k), S_j(k) = 1 shell by shell within 4 sigma + 0.5 % (R11, P10), where
    sigma = 1/sqrt(n_eff cnt/2): |X_k|^2 of a complex Gaussian mode has relative spread 1, k and -k are the same
    mode, and of the 91 snapshots taken 20 steps apart only n_eff = min(91, 1800 nu k^2) are independent (the
    variance of a mode decorrelates at rate 2 nu k^2).  That is +-1.5 % on the well-populated shells.
    The run starts cold (no fluctuations), so a mode of wavenumber k reaches its stationary variance as
    1 - exp(-2 nu k^2 t); averaged over the sampling window [200, 2000] that leaves a deficit of
    exp(-2 nu k^2 200) / (2 nu k^2 1800).  Shells where this exceeds 0.2 % (|k| L/2pi < 5 at tau=0.6, < 3 at
    tau=1.0) are reported only: they are slow, not wrong (measured: 0.96 and 0.98 on shells 3, 4 at tau=0.6)."""
    n, kT, rho0 = 64, 1e-4, 1.0
    sim = binding.Rflbm(n, n, n, tau, kT, rho0, 7)
    sim.init()
    sim.step(200)
    u2, acc, cnt = [], {}, None
    while sim.step_count <= 2000:
        rho, u = sim.moments()
        rho, u = rho.cpu().numpy(), u.cpu().numpy()
        u2.append((u ** 2).mean(axis=(1, 2, 3)))
        for name, fld, norm in [("rho", rho, 3 * rho0 * kT)] + [(f"j{a}", rho * u[a], rho0 * kT) for a in range(3)]:
            tot, cnt = shell_spectrum(fld)
            acc.setdefault(name, []).append(tot / norm)
        sim.step(20)
    u2 = np.mean(u2, axis=0) * rho0 / kT
    assert np.abs(u2 - 1.0).max() < 0.005, u2
    nu = (tau - 0.5) / 3.0
    shells = np.arange(len(cnt))
    k2 = (2 * np.pi * shells / n) ** 2
    rate = np.maximum(2 * nu * k2, 1e-300)
    gate = (np.exp(-rate * 200) / (rate * 1800) < 0.002) & (cnt >= 30) & (shells >= 1)
    assert gate.sum() >= 40 and gate[5:30].all()
    for name in ("rho", "j0", "j1", "j2"):
        s = np.mean(acc[name], axis=0)
        assert abs(s[1:].sum() / cnt[1:].sum() - 1.0) < 0.005, name
        sk = s[gate] / cnt[gate]
        n_eff = np.minimum(len(acc[name]), 1800 * nu * k2[gate])
        tol = 4.0 / np.sqrt(n_eff * cnt[gate] / 2.0) + 0.005
        assert (np.abs(sk - 1.0) < tol).all(), (name, tau, np.abs(sk - 1.0) / tol)
        assert tol[20:40].max() < 0.02
    d = sim.diagnostics()
    assert abs(d[0] / n ** 3 - rho0) < 1e-12 and max(abs(v) for v in d[1:4]) / n ** 3 < 1e-14


@pytest.mark.parametrize("tau,kT,tol", [(0.51, 0.0, 0.03), (0.8, 0.0, 0.005), (1.5, 0.0, 0.005),
                                        (0.51, 1e-5, 0.25), (0.8, 1e-5, 0.02), (1.5, 1e-5, 0.02)])
def test_config3_taylor_green_decay_256(tau, kT, tol):
    """Decay rate of the R15 vortex = 2 nu k^2, nu = (tau - 1/2)/3, with and without thermal noise.
    tau = 0.51: the amplitude decays by only 0.16 % over the fit window, and the weak sound wave radiated by the
    uniform-density start (R15: an O(u0^2) = 1e-4 pressure mismatch, one acoustic period = 443 steps, barely damped
    at this viscosity) modulates it at the 1e-5 level: 3 % on the rate without noise (measured 1.8 %), 25 % with."""
    torch = torch_()
    n, nz = 256, 256
    sim = binding.Rflbm(n, n, nz, tau, kT, 1.0, 3)
    rho0, u0 = synthetic.taylor_green_fields(n, n, nz, u0=0.01)
    sim.init(torch.from_numpy(rho0), torch.from_numpy(u0))
    x = torch.arange(n, device="cuda", dtype=torch.float64)
    shape = (torch.sin(2 * np.pi * x / n)[None, None, :] * torch.cos(2 * np.pi * x / n)[None, :, None])
    rho = torch.empty((nz, n, n), dtype=torch.float64, device="cuda")
    u = torch.empty((3, nz, n, n), dtype=torch.float64, device="cuda")
    sim.step(100)
    ts, amps = [], []
    while sim.step_count <= 500:
        sim.moments(rho, u)
        ts.append(sim.step_count)
        amps.append(4.0 * float((u[0] * shape).mean()))
        sim.step(10)
    k2 = 2 * (2 * np.pi / n) ** 2
    nu = (tau - 0.5) / 3.0
    assert abs(fit_decay_rate(ts, amps) / (nu * k2) - 1.0) < tol, (fit_decay_rate(ts, amps), nu * k2)


def test_config4_sampled_parity_and_conservation_512():
    """512^3 fp64 through the TMA kernel (the bench configuration): one step of sampled sites against the oracle's
    single-site collision (exact neighbours through the periodic wrap), then conservation over the run."""
    torch = torch_()
    n, tau, kT, seed = 512, 0.8, 1e-4, 11
    import gc
    gc.collect(); torch.cuda.empty_cache()                     # earlier tests' cached blocks do not count as free
    free, _ = torch.cuda.mem_get_info()
    if free < 125e9:
        pytest.skip("needs 125 GB of free device memory")
    sim = binding.Rflbm(n, n, n, tau, kT, 1.0, seed)
    sim.set_kernel_variant(binding.KERNEL_TMA)
    sim.init()
    sim.step(3)                                                # a thermal, site-dependent state
    f0 = sim.get_populations()
    sim.step(1)
    f1 = sim.get_populations()
    c = oracle.tables()[0]
    rng = np.random.default_rng(5)
    pts = rng.integers(0, n, size=(160, 3)).tolist()
    edge = [0, 1, 126, 127, 128, 129, 255, 256, 510, 511]      # tile boundaries of the TMA kernel and the wrap
    pts += [(x, int(rng.integers(0, n)), int(rng.integers(0, n))) for x in edge]
    pts += [(int(rng.integers(0, n)), y, z) for y in (0, 15, 16, 511) for z in (0, 511, 200)]
    pts += [(0, 0, 0), (511, 511, 511), (0, 511, 0), (511, 0, 511)]
    P = torch.tensor(pts, device="cuda")
    g_all = f0[:, P[:, 2], P[:, 1], P[:, 0]].T.cpu().numpy()   # [npts, 27]
    got = torch.empty((len(pts), 27), dtype=torch.float64, device="cuda")
    for i in range(27):
        xs, ys, zs = (P[:, 0] + int(c[i][0])) % n, (P[:, 1] + int(c[i][1])) % n, (P[:, 2] + int(c[i][2])) % n
        got[:, i] = f1[i, zs, ys, xs]
    got = got.cpu().numpy()
    worst = 0.0
    for k, (x, y, z) in enumerate(pts):
        want = oracle.collide_site(g_all[k], tau, kT, seed, site=x + n * (y + n * z), t=3)
        worst = max(worst, float(np.abs(got[k] - want).max()))
    assert worst < 1e-13, worst
    del f0, f1
    d0 = sim.diagnostics()
    sim.step(20)
    d1 = sim.diagnostics()
    N = n ** 3
    assert abs(d1[0] - d0[0]) / N < 1e-13 and abs(d0[0] / N - 1.0) < 1e-12
    assert max(abs(v) for v in d1[1:4]) / N < 1e-14
    assert np.abs(np.array(d1[7:10]) / kT - 1.0).max() < 0.01   # <u_a^2> = kT/rho0 (thermalised within ~10 steps)


def test_config5_channel_fp32_startup_profile_256():
    """256^3 channel, fp32 storage, walls z=0,255, g_x=1e-6, tau=0.9, kT=1e-4, 5000 steps: the plane-averaged
    u_x(z) follows the start-up series of P12 (5000 steps = 1 % of H^2/nu: a plug with boundary layers), and the
    bulk velocity variance is kT/rho0.  Near-wall variance is reported, not gated (parity unpinned)."""
    n, nz, tau, g, kT = 256, 256, 0.9, 1e-6, 1e-4
    sim = binding.Rflbm(n, n, nz, tau, kT, 1.0, 5, binding.F32)
    sim.set_walls_z(True)
    sim.set_force(g, 0.0, 0.0)
    sim.init()
    d0 = sim.diagnostics()
    sim.step(4000)
    prof, var, ts = [], [], []
    while sim.step_count <= 5000:
        rho, u = sim.moments()
        ud = u.double()
        prof.append(ud[0].mean(dim=(1, 2)).cpu().numpy())
        var.append(((ud - ud.mean(dim=(2, 3), keepdim=True)) ** 2).mean(dim=(2, 3)).cpu().numpy())
        ts.append(sim.step_count)
        sim.step(100)
    H = nz - 2
    nu = (tau - 0.5) / 3.0
    z = np.arange(1, nz - 1)
    lam = (tau - 0.5) / 2.0

    def series(t):
        steady = g / (2 * nu) * ((z - 0.5) * (nz - 1.5 - z) + 4 * lam / 3 - 0.25)
        ser = sum(4 * g * H ** 2 / (nu * np.pi ** 3 * m ** 3) * np.sin(m * np.pi * (z - 0.5) / H)
                  * np.exp(-m ** 2 * np.pi ** 2 * nu * t / H ** 2) for m in range(1, 4000, 2))
        return steady - ser

    want = np.mean([series(t) for t in ts], axis=0)
    got = np.mean(prof, axis=0)[1:-1]
    umax = want.max()
    assert 4.0e-3 < umax < 5.0e-3                                   # ~ g t: still a plug
    assert np.abs(got - want).max() < 0.03 * umax, np.abs(got - want).max() / umax
    v = np.mean(var, axis=0)[:, 1:-1] / kT                           # [3, fluid layers]
    assert np.abs(v[:, 20:-20].mean(axis=1) - 1.0).max() < 0.02, v[:, 20:-20].mean(axis=1)
    print("near-wall <du^2>/kT (layers 1..3):", v[:, :3])
    d1 = sim.diagnostics()
    assert abs(d1[0] / d0[0] - 1.0) < 1e-5                           # fp32 storage: mass drift reported and bounded


def _equilibration_ratios(sim, c, kT, until, every):
    """ER of rho, momentum, diagonal and off-diagonal Hermite stress over the lattice:
    variance / (rho0 kT b_k / cs2), averaged over snapshots taken `every` steps apart."""
    torch = torch_()
    er = []
    while sim.step_count <= until:
        f = sim.get_populations().reshape(27, -1)
        rho = f.sum(0)
        j = c.T @ f
        pd = torch.stack([((c[:, a] ** 2 - 1.0 / 3.0)[:, None] * f).sum(0) for a in range(3)])
        po = torch.stack([((c[:, a] * c[:, b])[:, None] * f).sum(0) for a, b in ((0, 1), (0, 2), (1, 2))])
        er.append([float(rho.var(unbiased=False)) / (3 * kT), float(j.var(dim=1, unbiased=False).mean()) / kT,
                   float(pd.var(dim=1, unbiased=False).mean()) / (2.0 / 3.0 * kT),
                   float(po.var(dim=1, unbiased=False).mean()) / (1.0 / 3.0 * kT)])
        sim.step(every)
    return np.mean(er, axis=0)


def _thermal_populations(n, kT, seed):
    """independent Gaussian populations of variance 3 kT rho0 w_i around w_i: the equilibrium measure of the
    fluctuating model (P8), so that the slow hydrodynamic modes of a tau -> 1/2 run start thermalised"""
    torch = torch_()
    w = torch.tensor(oracle.tables()[1], dtype=torch.float64, device="cuda").reshape(27, 1, 1, 1)
    gen = torch.Generator(device="cuda").manual_seed(seed)
    return w + torch.sqrt(3.0 * kT * w) * torch.randn((27, n, n, n), dtype=torch.float64, device="cuda", generator=gen)


def test_table_III_reduced_sweep_regflbm_all_14_tau(golden_dir):
    """Reduced Table III: all 14 relaxation times of the Reg-FLBM column at 64^3 and 2e4 steps
    instead of 256^3 and 5e5, kT = 1/3000 (:254), from a thermal start, printed beside the paper's row
    (tests/golden/table_III_regflbm.txt).  Gated: only what the paper states in words -
      * "within 0.5 %" of 1 for 0.51 <~ tau <~ 100 (:260): |ER - 1| < 0.005 for 0.55 <= tau <= 100, and < 0.016 at
        tau = 0.505 and 0.51, where Table III itself prints up to 1.016;
      * stable down to tau = 0.5001 with the errors GROWING as tau -> 1/2 (:268), and of the printed sign (ER > 1).
    The distance to the printed values is reported and bracketed at 0.03 (this build's bracket: the lattice is 64
    times smaller and the run 25 times shorter than the paper's)."""
    torch = torch_()
    n, kT = 64, 1.0 / 3000.0
    c = torch.tensor(oracle.tables()[0], dtype=torch.float64, device="cuda")
    rows = [[float(v) for v in ln.split()] for ln in open(golden_dir + "/table_III_regflbm.txt")
            if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 14
    got = {}
    print("\n   tau    ER(rho, j, Pi_aa, Pi_ab) here (64^3, 2e4 steps)   |  Table III (256^3, 5e5 steps)")
    for tau, *paper in rows:
        sim = binding.Rflbm(n, n, n, tau, kT, 1.0, 9)
        sim.set_populations(_thermal_populations(n, kT, 99), 0)
        sim.step(2000)
        er = _equilibration_ratios(sim, c, kT, 20000, 200)
        got[tau] = er
        print(f"{tau:8.4f}  " + "  ".join(f"{v:6.4f}" for v in er) + "   |  " + "  ".join(f"{v:5.3f}" for v in paper))
        assert np.isfinite(er).all(), tau                                   # stable (:268)
        assert np.abs(er - np.array(paper)).max() < 0.03, (tau, er, paper)  # reported distance, this build's bracket
        if tau >= 0.55:
            assert np.abs(er - 1.0).max() < 0.005, (tau, er)                # :260
        elif tau >= 0.505:
            assert np.abs(er - 1.0).max() < 0.016, (tau, er)
        else:
            assert (er > 1.005).all(), (tau, er)                            # the printed sign of the excess
    # errors grow as tau -> 1/2 (:268): momentum and both stress ratios are ordered like the printed column
    for k in (1, 2, 3):
        col = [got[t][k] for t in (0.5001, 0.5005, 0.501, 0.505, 0.51, 0.55)]
        assert all(a > b for a, b in zip(col, col[1:])), (k, col)


@pytest.mark.parametrize("tau", [1.0, 50.0])
def test_table_III_bgk_flbm_reading_R19_64(tau):
    """BGK-FLBM with reading R19 (all 23 modes thermalised at the one omega) ALSO equilibrates to 1.000 at tau = 50;
    the paper's BGK column (0.953 / 0.930 at tau >= 50) is not reproduced by Eq.11 as printed — DESIGN.md section 10."""
    torch = torch_()
    n, kT = 64, 1.0 / 3000.0
    c = torch.tensor(oracle.tables()[0], dtype=torch.float64, device="cuda")
    sim = binding.Rflbm(n, n, n, tau, kT, 1.0, 9)
    sim.set_model(binding.MODEL_BGK)
    sim.init()
    sim.step(4000)
    er = _equilibration_ratios(sim, c, kT, 20000, 200)
    print("bgk", tau, "ER(rho, j, Pi_aa, Pi_ab) =", np.round(er, 4))
    assert np.abs(er - 1.0).max() < 0.005, er


def test_largest_lattice_768_in_place_sampled_against_oracle():
    """Maximum size on a 180 GB part: 768^3 fp64 in the AA scheme (97.8 GB in one buffer; site indices up to 4.5e8,
    byte offsets up to 9.8e10).  After ONE step from the uniform start the state at a site is fully determined by
    the 27 neighbouring collisions of f = w (each with its own Philox counter), which the oracle evaluates one by one:
    S_1[q](x) = collide(w; site = x - c_q, t = 0)[q].  rho and u of sampled sites (corners, tile edges, the last
    site) are compared through rflbm_moments; then a second (odd-phase) step must conserve mass and momentum."""
    torch = torch_()
    n, tau, kT, seed = 768, 0.8, 1e-4, 11
    import gc
    gc.collect(); torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 120e9:
        pytest.skip("needs 120 GB of free device memory")
    sim = binding.Rflbm(n, n, n, tau, kT, 1.0, seed, scheme=binding.SCHEME_AA)
    assert sim.workspace.numel() < 99e9
    sim.init()
    sim.step(1)
    rho, u = sim.moments()
    c, w = oracle.tables()[:2]
    rng = np.random.default_rng(8)
    pts = rng.integers(0, n, size=(40, 3)).tolist()
    pts += [(0, 0, 0), (n - 1, n - 1, n - 1), (0, n - 1, 0), (127, 5, 767), (128, 767, 3), (767, 0, 400), (640, 15, 16)]
    worst = 0.0
    for x, y, z in pts:
        s1 = np.zeros(27)
        for q in range(27):
            xs, ys, zs = (x - c[q][0]) % n, (y - c[q][1]) % n, (z - c[q][2]) % n
            s1[q] = oracle.collide_site(w, tau, kT, seed, site=int(xs + n * (ys + n * zs)), t=0)[q]
        r = s1.sum()
        uu = (s1 @ c) / r
        worst = max(worst, abs(float(rho[z, y, x]) - r), float(np.abs(u[:, z, y, x].cpu().numpy() - uu).max()))
    assert worst < 1e-14, worst
    del rho, u
    d1 = sim.diagnostics()
    sim.step(1)                                                  # odd phase: pushes to the neighbours
    d2 = sim.diagnostics()
    N = n ** 3
    # sums of 4.5e8 terms through fp64 atomics: rounding of the accumulation itself is ~1e-13 relative
    assert abs(d1[0] / N - 1.0) < 1e-12 and abs(d2[0] - d1[0]) / N < 1e-12
    assert max(abs(v) for v in d2[1:4]) / N < 1e-14


@pytest.mark.parametrize("tau", [0.51, 50.0])
def test_fig1_fig2_fluctuation_spectra_256(tau):
    """The paper's spectral check (Fig.1 c-d, Fig.2) at its own lattice size, 256^3, kT = 1/3000:
    spherically averaged ER spectra of rho, momentum, diagonal and off-diagonal stress for 4 <= |k| <= 64 stay at 1 for
    Reg-FLBM at tau = 0.51 and tau = 50.  The run starts from an already thermal state (independent Gaussian
    populations of variance 3 kT rho0 w_i, the equilibrium measure P8) because at tau = 0.51 the |k| = 4 shell would
    need ~1.5e4 steps to thermalise from a cold start; what is tested is that the scheme KEEPS every shell at its
    equipartition value.  FFTs run on the GPU (torch.fft), test-side."""
    from analysis import shell_spectrum_torch
    torch = torch_()
    n, kT = 256, 1.0 / 3000.0
    w = torch.tensor(oracle.tables()[1], dtype=torch.float64, device="cuda").reshape(27, 1, 1, 1)
    c = torch.tensor(oracle.tables()[0], dtype=torch.float64, device="cuda")
    gen = torch.Generator(device="cuda").manual_seed(1234)
    f0 = w + torch.sqrt(3.0 * kT * w) * torch.randn((27, n, n, n), dtype=torch.float64, device="cuda", generator=gen)
    sim = binding.Rflbm(n, n, n, tau, kT, 1.0, 21, scheme=binding.SCHEME_AA)
    sim.set_populations(f0, 0)
    del f0
    acc = {}
    sim.step(200)
    rho = torch.empty((n, n, n), dtype=torch.float64, device="cuda")
    u = torch.empty((3, n, n, n), dtype=torch.float64, device="cuda")
    pi = torch.empty((6, n, n, n), dtype=torch.float64, device="cuda")
    nsamp = 0
    while sim.step_count <= 2000:
        sim.snapshot(rho, u, pi)                       # the paper's snapshot (:252) in one pass: = moments + stress bit for bit
        fields = [("rho", rho, 3 * kT)] + [("j", rho * u[a], kT) for a in range(3)] + \
                 [("pd", pi[a], 2.0 / 3.0 * kT) for a in range(3)] + [("po", pi[a], 1.0 / 3.0 * kT) for a in range(3, 6)]
        for name, fld, norm in fields:
            tot, cnt = shell_spectrum_torch(fld)
            acc[name] = acc.get(name, 0.0) + tot / norm
        nsamp += 1
        sim.step(100)
    sel = slice(4, 65)
    nu = (tau - 0.5) / 3.0
    k2 = (2 * np.pi * np.arange(len(cnt)) / n) ** 2
    n_eff = np.clip(nsamp * 100 * 2 * nu * k2 / 2, 1.0, nsamp)[sel]       # independent snapshots per shell
    bad = []
    for name, mult in (("rho", 1), ("j", 3), ("pd", 3), ("po", 3)):
        er = acc[name][sel] / (nsamp * mult * cnt[sel])
        # statistical tolerance (4 sigma) + a systematic bracket: 1 % at tau = 50; 6 % at tau = 0.51, where, next to the
        # stability limit, the mid-range shells sit a few per cent ABOVE 1 (the printed means over 24 <= |k| <= 64; rho:
        # 1.03): the direction of the excess Table III prints for tau = 0.51 (1.005 / 1.013 / 1.004 / 1.012 lattice-wide,
        # i.e. averaged up to the Nyquist corner).  Fig.1(c) itself is not in the container, so the 6 % is this build's
        # bracket, not the paper's.  That the excess is the METHOD's and not the kernel's is shown on the oracle:
        # tests/test_oracle_physics.py::test_tau_051_midshell_density_excess_belongs_to_the_method (1.02 on the same
        # |k| at 32^3) and test_tau_051_midshell_excess_gpu_equals_oracle_32 below.
        syst = 0.06 if tau < 0.55 else 0.01
        tol = 4.0 / np.sqrt(n_eff * mult * cnt[sel] / 2.0) + syst
        print(name, tau, "ER(|k|=4..64): min %.4f max %.4f" % (er.min(), er.max()), "worst/tol %.2f" % (np.abs(er - 1) / tol).max(),
              "| 24<=|k|<=64: mean %.4f min %.4f max %.4f" % (er[20:].mean(), er[20:].min(), er[20:].max()))
        if not (np.abs(er - 1.0) < tol).all() or np.abs(er[20:] - 1.0).max() > syst + 0.01:
            bad.append(name)
    assert not bad, bad


def test_tau_051_midshell_excess_gpu_equals_oracle_32():
    """The few-per-cent density excess on the mid shells at tau = 0.51 (bracketed at 6 % in the 256^3 test above) is
    the method's: on a 32^3 box the CUDA path and the oracle, started from the same thermal populations with the same
    seed, give the same shell spectra to 1e-9 (and the same populations to 1e-11 after 1200 steps), and both show the
    excess on shells 3..8 (tests/test_oracle_physics.py pins the oracle's value over a longer run)."""
    torch = torch_()
    n, kT, tau = 32, 1.0 / 3000.0, 0.51
    w = oracle.tables()[1]
    f0 = synthetic.gaussian_population_field(n, n, n, 1234, w, np.sqrt(3.0 * kT * w))
    sim = binding.Rflbm(n, n, n, tau, kT, 1.0, 21)
    ref = oracle.Ref(n, n, n, tau, kT, 1.0, 21, threads=oracle.max_threads())
    sim.set_populations(torch.from_numpy(f0), 0); ref.set_populations(f0, 0)
    sim.step(200); ref.step(200)
    acc_g, acc_r, ns = 0.0, 0.0, 0
    while sim.step_count <= 1200:
        tot_g, cnt = shell_spectrum(sim.moments()[0].cpu().numpy())
        tot_r, _ = shell_spectrum(ref.moments()[0])
        acc_g, acc_r, ns = acc_g + tot_g / (3 * kT), acc_r + tot_r / (3 * kT), ns + 1
        sim.step(50); ref.step(50)
    assert np.abs(sim.get_populations().cpu().numpy() - ref.get_populations()).max() < 1e-11
    assert np.abs(acc_g[1:] / acc_r[1:] - 1.0).max() < 1e-9
    mid_g = acc_g[3:9].sum() / (ns * cnt[3:9].sum())
    mid_r = acc_r[3:9].sum() / (ns * cnt[3:9].sum())
    print(f"32^3 tau=0.51 ER_rho shells 3..8: CUDA {mid_g:.5f}, oracle {mid_r:.5f}")
    assert mid_g > 1.005 and mid_r > 1.005
