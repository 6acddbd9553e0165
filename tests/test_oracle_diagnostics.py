"""Pin of rflbm_ref_diagnostics outputs 4..9 (mean u, var u over FLUID sites; oracle/rflbm_ref.c) against what the
paper fixes: rho and j are rows 0..3 of the PAPER's printed Hermite basis applied to the state (Eq.2-4,
PAPER.md:56-62, Table II :172-202), u = (j + F/2)/rho (Eq.3 with the half-force shift of R13), and the moments of u
are the plain definitions mean(u), mean(u^2) - mean(u)^2 over the fluid layers only (R12: solid layers z = 0 and
z = nz-1 carry no fluid).  Chosen so that a wrong divisor (all sites instead of fluid sites), a missing - mean^2,
a missing g/2 or a transposed component fails."""
import numpy as np
import pytest

import oracle
from paper_2507_08820_b200 import synthetic
from paper_tables import exact_basis


def _printed_rows_0_to_3():
    c = oracle.tables()[0]
    return np.array([[float(v) for v in row] for row in exact_basis(c)[:4]])


@pytest.mark.parametrize("walls", [False, True])
def test_diagnostics_mean_and_variance_against_printed_basis(walls):
    """non-zero, component-dependent mean flow + body force + (optionally) walls; after init and after 7 noisy steps"""
    nx, ny, nz = 6, 5, 7
    g = np.array([3e-4, -1e-4, 2e-4])
    rho, u = synthetic.smooth_random_fields(nx, ny, nz, 17)
    u[0] += 0.04; u[1] -= 0.02; u[2] += 0.01                 # |mean| >> std: dropping "- mean^2" is a 100 % error
    r = oracle.Ref(nx, ny, nz, 0.8, 1e-4, 1.0, 3)
    if walls:
        r.set_walls_z(True)
    r.set_force(*g)
    r.init(rho, u)
    E = _printed_rows_0_to_3()
    for nsteps in (0, 7):
        r.step(nsteps)
        f = r.get_populations()
        d = r.diagnostics()
        m = np.einsum("ki,izyx->kzyx", E, f)                # rho, j_x, j_y, j_z from the printed polynomials
        fluid = slice(1, nz - 1) if walls else slice(0, nz)
        rr = m[0][fluid]
        uu = np.stack([(m[1 + a][fluid] + 0.5 * rr * g[a]) / rr for a in range(3)])
        nf = rr.size
        assert nf == nx * ny * (nz - 2 if walls else nz)
        assert abs(d[0] - rr.sum()) < 1e-12
        for a in range(3):
            assert abs(d[1 + a] - (rr * uu[a]).sum()) < 1e-13
            mean = uu[a].sum() / nf
            var = (uu[a] ** 2).sum() / nf - mean * mean
            assert abs(d[4 + a] - mean) < 1e-16, (a, d[4 + a], mean)
            assert abs(d[7 + a] - var) < 1e-17, (a, d[7 + a], var)
            assert var > 1e-6 and abs(mean) > 5e-3            # the case really exercises both terms
        if walls:                                            # the all-sites divisor would be off by nz/(nz-2)
            wrong = uu[0].sum() / (nx * ny * nz)
            assert abs(d[4] - wrong) > 1e-3


def test_diagnostics_closed_form_uniform_flow_with_force():
    """uniform (rho, u) with an acceleration g: the reported velocity is u_init everywhere at t = 0 (init builds
    f^(0)(rho, u) and the diagnostics add g/2 to j/rho: mean = u + g/2, R13), variance exactly 0 up to round-off;
    after n deterministic steps (kT = 0, periodic) the flow stays uniform and mean = u + g (n + 1/2)."""
    nx, ny, nz = 4, 3, 5
    u0 = (0.03, -0.01, 0.02)
    g = (2e-5, 0.0, -1e-5)
    rho, u = synthetic.uniform_fields(nx, ny, nz, 1.1, u0)
    r = oracle.Ref(nx, ny, nz, 0.9, 0.0, 1.1, 0)
    r.set_force(*g)
    r.init(rho, u)
    for n in (0, 4):
        r.step(n)
        d = r.diagnostics()
        for a in range(3):
            assert abs(d[4 + a] - (u0[a] + g[a] * (n + 0.5))) < 1e-15
            assert abs(d[7 + a]) < 1e-17
        assert abs(d[0] - 1.1 * nx * ny * nz) < 1e-12


def test_diagnostics_variance_is_equipartition_not_second_moment():
    """thermal box with a uniform drift U: var u_a -> kT/rho0 (P8) while <u_a^2> -> kT/rho0 + U^2; the drift is chosen
    so that U^2 = 25 kT/rho0."""
    n, kT, U = 12, 1e-4, 0.05
    rho, u = synthetic.uniform_fields(n, n, n, 1.0, (U, 0.0, 0.0))
    r = oracle.Ref(n, n, n, 1.0, kT, 1.0, 5, threads=min(8, oracle.max_threads()))
    r.init(rho, u)
    r.step(30)
    acc = []
    for _ in range(10):
        r.step(5)
        acc.append(r.diagnostics())
    d = np.mean(acc, axis=0)
    assert abs(d[4] - U) < 1e-4 * U + 1e-5                     # sum rho u is conserved exactly; mean(j/rho) differs at O(U var rho)
    assert np.abs(d[7:10] / kT - 1.0).max() < 0.08, d[7:10] / kT   # 1728 sites x 10 samples: sigma ~ 1 %, Galilean O(U^2) ~ 1 %
