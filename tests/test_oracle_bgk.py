"""Pins of the oracle's BGK-FLBM (Eq.11; reading R19), the paper's comparison model.

The oracle evaluates Eq.11 in population space as printed; the pins look at the result in MODE space with the
paper's printed basis (tests/golden/table_II.txt), so a wrong rate, a missing mode or a wrong noise amplitude in
either representation shows up."""
import numpy as np
import pytest

import oracle
from analysis import fit_decay_rate, tg_amplitude
from paper_2507_08820_b200 import synthetic
from paper_tables import exact_basis, table_II

NT = min(8, oracle.max_threads())


def _paper_basis():
    c = oracle.tables()[0]
    E = np.array([[float(v) for v in row] for row in exact_basis(c)])
    b = np.array([float(r[4]) for r in table_II()])
    return c, E, b


@pytest.mark.parametrize("tau", [0.51, 0.8, 1.0, 50.0])
def test_bgk_every_nonconserved_mode_relaxes_at_omega_kT0(tau):
    """Eq.6 + Eq.4: m*_k = m_k for k=0..3, m*_k = m_k^eq + (1-omega)(m_k - m_k^eq) for ALL k=4..26 (one rate), with
    m_k^eq = rho u^p u^q u^r (Eq.20).  Contrast with Reg-FLBM, whose ghost modes are reset to equilibrium."""
    c, E, b = _paper_basis()
    pqr = oracle.tables()[3]
    for g in synthetic.random_populations(21, 6, spread=0.2):
        fs = oracle.collide_site_bgk(g, tau, kT=0.0)
        m_in, m_out = E @ g, E @ fs
        rho = g.sum()
        u = (g @ c) / rho
        eq = np.array([rho * u[0] ** p * u[1] ** q * u[2] ** r for p, q, r in pqr])
        want = eq + (1.0 - 1.0 / tau) * (m_in - eq)
        want[:4] = m_in[:4]
        assert np.abs(m_out - want).max() < 2e-15
        reg = E @ oracle.collide_site(g, tau, kT=0.0)
        assert np.abs(reg[:10] - m_out[:10]).max() < 2e-15            # same hydrodynamic modes ...
        if tau != 1.0:
            assert np.abs(reg[10:] - m_out[10:]).max() > 1e-6          # ... different ghosts


def test_bgk_tau1_is_equilibrium_and_equilibrium_is_fixed_point():
    def phi(cc, uu):
        return 2.0 / 3.0 - uu * uu if cc == 0 else 1.0 / 6.0 + 0.5 * cc * uu + 0.5 * uu * uu
    c = oracle.tables()[0]
    g = synthetic.random_populations(22, 1, spread=0.2)[0]
    rho, u = g.sum(), (g @ c) / g.sum()
    closed = np.array([rho * phi(ci[0], u[0]) * phi(ci[1], u[1]) * phi(ci[2], u[2]) for ci in c])
    assert np.abs(oracle.collide_site_bgk(g, 1.0) - closed).max() < 1e-15
    for tau in (0.51, 3.0):
        assert np.abs(oracle.collide_site_bgk(closed, tau) - closed).max() < 1e-15


def test_bgk_noise_has_single_rate_fdt_amplitude_and_conserves():
    """Eq.9 with the one omega for every k=4..26; mass and momentum untouched (:95)."""
    c, E, b = _paper_basis()
    tau, kT, seed = 0.9, 2e-4, 77
    r = oracle.Ref(4, 3, 2, tau, kT, 1.0, seed)
    _, normals = r.debug_rng(5)
    g = synthetic.random_populations(23, 1, spread=0.1)[0]
    site = 11
    noisy = oracle.collide_site_bgk(g, tau, kT=kT, seed=seed, site=site, t=5)
    d = E @ (noisy - oracle.collide_site_bgk(g, tau, kT=0.0))
    om = 1.0 / tau
    sigma = np.sqrt(kT * om * (2.0 - om) * b * 3.0)
    want = np.zeros(27)
    want[4:] = np.sqrt(g.sum()) * sigma[4:] * normals.reshape(23, -1)[:, site]
    assert np.abs(d - want).max() < 1e-16 + 1e-13 * np.abs(want).max()
    assert abs(noisy.sum() - g.sum()) < 1e-15 and np.abs(noisy @ c - g @ c).max() < 1e-15


def test_bgk_taylor_green_decay_and_model_switch():
    """nu = (tau - 1/2)/3 also for BGK; set_model validation; force is refused in this model."""
    n, tau = 32, 0.8
    r = oracle.Ref(n, n, 2, tau, 0.0, threads=NT)
    r.set_model(oracle.MODEL_BGK)
    with pytest.raises(oracle.RefError):
        r.set_force(1e-6, 0.0, 0.0)
    with pytest.raises(oracle.RefError):
        r.set_model(7)
    rho, u = synthetic.taylor_green_fields(n, n, 2, u0=0.01)
    r.init(rho, u)
    ts, amps = [], []
    r.step(100)
    for _ in range(21):
        ts.append(r.step_count)
        amps.append(tg_amplitude(r.moments()[1], n, n))
        r.step(20)
    assert abs(fit_decay_rate(ts, amps) / ((tau - 0.5) / 3.0 * 2 * (2 * np.pi / n) ** 2) - 1.0) < 0.005


def test_bgk_equipartition_all_modes():
    """R11 for BGK-FLBM: stationary var(m_k) = rho0 kT b_k / cs2 for every k (12^3, tau=0.8)."""
    c, E, b = _paper_basis()
    kT = 1e-4
    r = oracle.Ref(12, 12, 12, 0.8, kT, 1.0, 5, threads=NT)
    r.set_model(oracle.MODEL_BGK)
    r.init()
    r.step(100)
    acc = np.zeros(27)
    ns = 40
    for _ in range(ns):
        m = np.einsum("ki,izyx->kzyx", E, r.get_populations())
        acc += np.array([((m[k] - m[k].mean()) ** 2).mean() for k in range(27)])
        r.step(10)
    ratio = acc / ns / (kT * b * 3.0)
    assert np.abs(ratio - 1.0).max() < 0.04, ratio
