"""P4/P5/P7: single-site collision of the oracle against what Eq.24-26 fix."""
import numpy as np
import pytest

import oracle
from paper_2507_08820_b200 import synthetic
from paper_tables import exact_basis, table_II


def _paper_basis():
    c = oracle.tables()[0]
    E = np.array([[float(v) for v in row] for row in exact_basis(c)])
    b = np.array([float(r[4]) for r in table_II()])
    return c, E, b


@pytest.mark.parametrize("tau", [0.51, 0.8, 1.0, 50.0])
def test_post_collision_moment_structure_kT0(tau):
    """P7: k=0..3 unchanged, k=4..9 = rho u u + (1-omega_h) a1, k=10..26 = rho u^p u^q u^r."""
    c, E, b = _paper_basis()
    pqr = oracle.tables()[3]
    for g in synthetic.random_populations(11, 6, spread=0.2):
        fs = oracle.collide_site(g, tau, kT=0.0)
        m_in, m_out = E @ g, E @ fs
        rho = g.sum()
        u = (g @ c) / rho
        assert np.abs(m_out[:4] - m_in[:4]).max() < 1e-15
        eq = np.array([rho * u[0] ** p * u[1] ** q * u[2] ** r for p, q, r in pqr])
        want = eq.copy()
        want[4:10] += (1.0 - 1.0 / tau) * (m_in[4:10] - eq[4:10])
        assert np.abs(m_out - want).max() < 1e-15


def test_mass_momentum_conserved_per_site_with_noise():
    c, E, b = _paper_basis()
    for n, g in enumerate(synthetic.random_populations(12, 20, spread=0.2)):
        fs = oracle.collide_site(g, 0.7, kT=1e-3, seed=99, site=n, t=3)
        assert abs(fs.sum() - g.sum()) < 1e-15
        assert np.abs(fs @ c - g @ c).max() < 1e-15
        assert np.abs(fs - oracle.collide_site(g, 0.7, kT=0.0)).max() > 1e-4   # the noise is really there


def test_noise_enters_modes_with_fdt_amplitude_single_site():
    """Eq.8-9: post-collision mode k minus its deterministic value = sqrt(rho) sigma_k r_k with the r_k of
    debug_rng, sigma_k^2 = kT omega_k (2-omega_k) b_k / cs2, omega_k = omega_h (k<=9) or 1 (ghosts)."""
    c, E, b = _paper_basis()
    tau, kT, seed = 0.9, 2e-4, 77
    r = oracle.Ref(4, 3, 2, tau, kT, 1.0, seed)
    _, normals = r.debug_rng(5)
    g = synthetic.random_populations(13, 1, spread=0.1)[0]
    site = 17
    d = E @ (oracle.collide_site(g, tau, kT=kT, seed=seed, site=site, t=5) - oracle.collide_site(g, tau, kT=0.0))
    om = np.array([0.0] * 4 + [1.0 / tau] * 6 + [1.0] * 17)
    sigma = np.sqrt(kT * om * (2.0 - om) * b * 3.0)
    want = np.zeros(27)
    want[4:] = np.sqrt(g.sum()) * sigma[4:] * normals.reshape(23, -1)[:, site]
    assert np.abs(d - want).max() < 1e-16 + 1e-13 * np.abs(want).max()
    assert np.abs(d[:4]).max() < 1e-15


def test_equilibrium_is_fixed_point_and_tau1_projects_to_equilibrium():
    """P5."""
    for u in ([0.0, 0.0, 0.0], [0.1, -0.05, 0.02], [-0.03, 0.08, -0.1]):
        f0 = oracle.equilibrium(1.3, u)
        for tau in (0.51, 1.0, 7.0):
            assert np.abs(oracle.collide_site(f0, tau) - f0).max() < 1e-15
    g = synthetic.random_populations(14, 1, spread=0.2)[0]
    c = oracle.tables()[0]
    rho, u = g.sum(), (g @ c) / g.sum()
    assert np.abs(oracle.collide_site(g, 1.0) - oracle.equilibrium(rho, u)).max() < 1e-15


def test_force_adds_momentum_F_per_site():
    """R13: post-collision momentum = j + F with F = rho g; reduces to the unforced update at g=0."""
    c, E, b = _paper_basis()
    g = synthetic.random_populations(15, 1, spread=0.1)[0]
    acc = np.array([1e-3, -2e-3, 5e-4])
    fs = oracle.collide_site(g, 0.9, gacc=acc)
    assert abs(fs.sum() - g.sum()) < 1e-15
    assert np.abs(fs @ c - (g @ c + g.sum() * acc)).max() < 1e-15
    # stress: rho u u + (1-w)(Pi - rho u u) + (1-w/2)(uF+Fu), u = (j+F/2)/rho  (Guo forcing, textbook form)
    w = 1.0 / 0.9
    rho = g.sum()
    F = rho * acc
    u = (g @ c + 0.5 * F) / rho
    m_in, m_out = E @ g, E @ fs
    idx = [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]
    for n, (a, bb) in enumerate(idx):
        eq = rho * u[a] * u[bb]
        want = eq + (1 - w) * (m_in[4 + n] - eq) + (1 - w / 2) * (u[a] * F[bb] + u[bb] * F[a])
        assert abs(m_out[4 + n] - want) < 1e-15
    assert np.array_equal(oracle.collide_site(g, 0.9, gacc=(0, 0, 0)), oracle.collide_site(g, 0.9))
