"""P8-P12: the oracle against closed forms of the physics it must reproduce (small boxes, CPU only)."""
import numpy as np
import pytest

import oracle
from analysis import fit_decay_rate, shell_spectrum, tg_amplitude
from paper_2507_08820_b200 import synthetic
from paper_tables import exact_basis, table_II

NT = min(8, oracle.max_threads())


@pytest.mark.parametrize("tau,tol", [(0.51, 0.01), (0.8, 0.005), (1.5, 0.03)])
def test_taylor_green_decay_rate_kT0(tau, tol):
    """P11: amplitude ~ exp(-2 nu k^2 t), nu = (tau - 1/2)/3.  32x32 vortex, uniform in z."""
    n = 32
    r = oracle.Ref(n, n, 2, tau, 0.0, threads=NT)
    rho, u = synthetic.taylor_green_fields(n, n, 2, u0=0.01)
    r.init(rho, u)
    ts, amps = [], []
    r.step(100)
    for _ in range(21):
        ts.append(r.step_count)
        amps.append(tg_amplitude(r.moments()[1], n, n))
        r.step(20)
    k2 = 2 * (2 * np.pi / n) ** 2
    nu = (tau - 0.5) / 3.0
    assert abs(fit_decay_rate(ts, amps) / (nu * k2) - 1.0) < tol


@pytest.fixture(scope="module")
def thermal_run():
    """16^3, kT=1e-4: populations sampled every 10 steps for t in [100, 600] at two tau."""
    out = {}
    for tau in (0.6, 1.0):
        r = oracle.Ref(16, 16, 16, tau, 1e-4, 1.0, 7, threads=NT)
        r.init()
        r.step(100)
        snaps = []
        for _ in range(50):
            snaps.append(r.get_populations())
            r.step(10)
        out[tau] = np.stack(snaps)
    return out


@pytest.mark.parametrize("tau", [0.6, 1.0])
def test_equipartition_all_27_modes(thermal_run, tau):
    """P8 (R11): stationary var(m_k) = rho0 kT b_k / cs2 for every k, hence <u_a^2> = kT/rho0."""
    c = oracle.tables()[0]
    E = np.array([[float(v) for v in row] for row in exact_basis(c)])   # the paper's printed basis
    b = np.array([float(r[4]) for r in table_II()])
    f = thermal_run[tau]                                  # [T,27,z,y,x]
    m = np.einsum("ki,tizyx->ktzyx", E, f)
    kT, rho0 = 1e-4, 1.0
    var = np.array([((m[k] - m[k].mean()) ** 2).mean() for k in range(27)])
    ratio = var / (rho0 * kT * b * 3.0)
    # 204 800 samples per mode (time-correlated for the slow hydrodynamic ones): 3 %
    assert np.abs(ratio - 1.0).max() < 0.03, ratio
    rho = m[0]
    u = m[1:4] / rho
    assert np.abs((u ** 2).mean(axis=(1, 2, 3, 4)) * rho0 / kT - 1.0).max() < 0.03
    # populations: var(f_i) = 3 kT rho0 w_i (completeness), pairwise uncorrelated
    w = oracle.tables()[1]
    vf = np.array([f[:, i].var() for i in range(27)])
    assert np.abs(vf / (3 * kT * rho0 * w) - 1.0).max() < 0.03


@pytest.mark.parametrize("tau", [0.6, 1.0])
def test_flat_structure_factor(thermal_run, tau):
    """P10 (R11): S_rho(k) = <|rho_k|^2>/(N 3 rho0 kT) and S_j(k) = <|j_k|^2>/(N rho0 kT) are 1 for all k != 0."""
    c = oracle.tables()[0].astype(float)
    f = thermal_run[tau]
    kT, rho0 = 1e-4, 1.0
    acc = {}
    for snap in f:
        rho = snap.sum(axis=0)
        j = np.einsum("izyx,ia->azyx", snap, c)
        for name, fld, norm in [("rho", rho, 3 * rho0 * kT)] + [(f"j{a}", j[a], rho0 * kT) for a in range(3)]:
            tot, cnt = shell_spectrum(fld)
            acc.setdefault(name, []).append(tot / norm)
            acc["cnt"] = cnt
    cnt = acc["cnt"]
    for name in ("rho", "j0", "j1", "j2"):
        s = np.mean(acc[name], axis=0)
        shells = np.arange(len(s))
        sk = s[1:] / cnt[1:]
        # all k != 0 together: 4095 modes x 50 snapshots
        assert abs(s[1:].sum() / cnt[1:].sum() - 1.0) < 0.02, (name, s[1:].sum() / cnt[1:].sum())
        # shell by shell, every shell from |k| index 2 up holding >= 30 wavevectors (the lowest shell is slow,
        # nu k^2 t_run ~ 1; the Nyquist corner shells hold 1-12 real modes): within 6 %
        # (shell 2: ~10 independent samples of ~30 vectors at tau=0.6 -> 15 %)
        gate = (shells[1:] >= 3) & (cnt[1:] >= 30)
        assert gate.sum() >= 9
        assert np.abs(sk[gate] - 1.0).max() < 0.06, (name, sk)
        assert abs(sk[1] - 1.0) < 0.15, (name, sk)


def test_poiseuille_steady_profile_with_slip():
    """P12 (R12, R13): halfway bounce-back walls + Guo force, kT=0.  Steady profile
    u_x(z) = g/(2 nu) [ (z-1/2)(nz-3/2-z) + 4 Lambda/3 - 1/4 ], Lambda = (tau-1/2)/2
    (two-relaxation-time wall-slip result with the odd/ghost rate equal to 1)."""
    nz, tau, g = 18, 0.9, 1e-6
    r = oracle.Ref(1, 1, nz, tau, 0.0)
    r.set_walls_z(True)
    r.set_force(g, 0.0, 0.0)
    r.init()
    r.step(12000)                                          # H^2/nu = 1920 steps
    rho, u = r.moments()
    z = np.arange(1, nz - 1)
    nu = (tau - 0.5) / 3.0
    lam = (tau - 0.5) / 2.0
    want = g / (2 * nu) * ((z - 0.5) * (nz - 1.5 - z) + 4 * lam / 3 - 0.25)
    got = u[0, 1:-1, 0, 0]
    assert np.abs(got / want - 1.0).max() < 1e-6
    assert np.abs(u[1:]).max() < 1e-14 and np.abs(rho[1:-1] - 1.0).max() < 1e-10


def test_poiseuille_startup_series():
    """P12: transient = steady - sum_{n odd} 4 g H^2/(nu pi^3 n^3) sin(n pi (z-1/2)/H) exp(-n^2 pi^2 nu t/H^2)."""
    nz, tau, g = 34, 0.9, 1e-6
    H = nz - 2
    nu = (tau - 0.5) / 3.0
    r = oracle.Ref(1, 1, nz, tau, 0.0)
    r.set_walls_z(True)
    r.set_force(g, 0.0, 0.0)
    r.init()
    z = np.arange(1, nz - 1)
    for t in (500, 2000):
        r.step(t - r.step_count)
        got = r.moments()[1][0, 1:-1, 0, 0]
        steady = g / (2 * nu) * (z - 0.5) * (nz - 1.5 - z)
        ser = sum(4 * g * H ** 2 / (nu * np.pi ** 3 * n ** 3) * np.sin(n * np.pi * (z - 0.5) / H)
                  * np.exp(-n ** 2 * np.pi ** 2 * nu * t / H ** 2) for n in range(1, 200, 2))
        want = steady - ser
        assert np.abs(got - want).max() < 2e-3 * (g * H ** 2 / (8 * nu))


@pytest.mark.parametrize("tau", [0.51, 50.0])
def test_stable_and_equilibrated_at_extreme_tau(tau):
    """P9: trend of Table III — Reg-FLBM is stable at tau=0.51 and tau=50 with site-level ER close to 1."""
    r = oracle.Ref(12, 12, 12, tau, 1e-4, 1.0, 31, threads=NT)
    r.init()
    r.step(150)
    vs = []
    for _ in range(40):
        rho, u = r.moments()
        assert np.isfinite(rho).all()
        vs.append([(rho - 1).var() / 3e-4] + [(rho * u[a]).var() / 1e-4 for a in range(3)])
        r.step(10)
    vs = np.mean(vs, axis=0)
    assert np.abs(vs - 1.0).max() < 0.04, vs


def test_tau_051_midshell_density_excess_belongs_to_the_method():
    """at tau = 0.51 the GPU run at 256^3 keeps the density shells 24 <= |k| <= 64 a few per cent
    ABOVE their equipartition value (tests/test_gpu_configs.py::test_fig1_fig2_fluctuation_spectra_256 brackets it at
    6 %).  The ORACLE shows the same excess on the corresponding shells of a 32^3 box (|k| L/2pi = 3..8, the same
    |k| in lattice units), from the same kind of thermal start: it is a property of the scheme next to the stability
    limit - the direction Table III prints for tau = 0.51 (1.005 / 1.013 / 1.004 / 1.012 lattice-wide)
    - and not of the CUDA kernel.  Statistical error of the shell mean: ~0.6 % (1.3e3 independent modes, ~20
    decorrelated snapshots), so the 1.008 .. 1.05 window is a > 2 sigma statement on both sides; measured 1.020.
    The whole lattice stays within 1 % of equipartition (measured 1.004), as Table III says."""
    n, kT, tau = 32, 1.0 / 3000.0, 0.51
    w = oracle.tables()[1]
    r = oracle.Ref(n, n, n, tau, kT, 1.0, 21, threads=oracle.max_threads())
    r.set_populations(synthetic.gaussian_population_field(n, n, n, 1234, w, np.sqrt(3.0 * kT * w)), 0)
    r.step(200)
    acc, ns, cnt = 0.0, 0, None
    while r.step_count <= 2200:
        rho, _ = r.moments()
        tot, cnt = shell_spectrum(rho)
        acc = acc + tot / (3.0 * kT)
        ns += 1
        r.step(50)
    mid = acc[3:9].sum() / (ns * cnt[3:9].sum())
    whole = acc[1:].sum() / (ns * cnt[1:].sum())
    print(f"oracle 32^3 tau=0.51: ER_rho shells 3..8 = {mid:.4f}, all shells = {whole:.4f}")
    assert 1.008 < mid < 1.05, mid
    assert abs(whole - 1.0) < 0.01, whole
