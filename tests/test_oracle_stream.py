"""P13/P14 and conservation: streaming, boundaries and order independence of the oracle."""
import numpy as np
import pytest

import oracle
from paper_2507_08820_b200 import synthetic


def _roll_stream(fstar, c, periodic_z=True):
    """brute-force Eq.7 with numpy: f_i(x + c_i) = f*_i(x)."""
    out = np.empty_like(fstar)
    for i in range(27):
        out[i] = np.roll(fstar[i], shift=(int(c[i][2]), int(c[i][1]), int(c[i][0])), axis=(0, 1, 2))
    return out


@pytest.mark.parametrize("shape", [(2, 2, 2), (3, 1, 1), (5, 7, 9), (4, 4, 1)])
def test_streaming_direction_and_wrap_bruteforce(shape):
    """tau=1, kT=0: f* is the equilibrium of the local (rho,u) (P5), so one step is 'closed-form collide,
    then np.roll' — pins the sign and axis order of the streaming and the periodic wrap (P14)."""
    nx, ny, nz = shape
    c, w = oracle.tables()[:2]
    r = oracle.Ref(nx, ny, nz, 1.0, 0.0)
    f = synthetic.random_population_field(nx, ny, nz, 3, w, spread=0.1)
    r.set_populations(f, 0)
    r.step(1)
    rho = f.sum(axis=0)
    u = np.einsum("izyx,ia->azyx", f, c.astype(float)) / rho

    def phi(cc, uu):
        return 2.0 / 3.0 - uu * uu if cc == 0 else 1.0 / 6.0 + cc * uu / 2 + uu * uu / 2

    fstar = np.stack([rho * phi(int(c[i][0]), u[0]) * phi(int(c[i][1]), u[1]) * phi(int(c[i][2]), u[2])
                      for i in range(27)])
    want = _roll_stream(fstar, c)
    assert np.abs(r.get_populations() - want).max() < 1e-15
    assert r.step_count == 1


def test_single_marked_population_moves_by_c():
    c, w = oracle.tables()[:2]
    nx, ny, nz = 4, 5, 6
    for i in range(27):
        r = oracle.Ref(nx, ny, nz, 1.0, 0.0)
        r.init()
        f0 = r.get_populations()
        # at tau=1,kT=0 a uniform rest state is a fixed point; perturb nothing, just check the index map by
        # comparing against a field whose equilibrium differs per site
        rho, u = synthetic.smooth_random_fields(nx, ny, nz, 4)
        r.init(rho, u)
        f_before = r.get_populations()
        r.step(1)
        f_after = r.get_populations()
        x, y, z = 1, 2, 3
        xd, yd, zd = (x + c[i][0]) % nx, (y + c[i][1]) % ny, (z + c[i][2]) % nz
        site_pops = f_before[:, z, y, x]
        fs = oracle.collide_site(site_pops, 1.0)
        assert f_after[i, zd, yd, xd] == fs[i]


def test_global_conservation_100_steps():
    """P4: mass and momentum on a periodic box, noise on."""
    r = oracle.Ref(8, 6, 10, 0.8, 1e-4, 1.0, 5, threads=2)
    rho, u = synthetic.smooth_random_fields(8, 6, 10, 6)
    r.init(rho, u)
    d0 = r.diagnostics()
    r.step(100)
    d1 = r.diagnostics()
    assert abs(d1[0] - d0[0]) < 1e-13 * d0[0]
    assert np.abs(d1[1:4] - d0[1:4]).max() < 1e-13 * d0[0]


def test_order_independence_threads_and_split_steps():
    """P13: reverse visiting order, threads, and step(50)+step(50) vs step(100) are bit-identical."""
    def run(kind):
        r = oracle.Ref(6, 5, 4, 0.7, 1e-4, 1.0, 9, threads=(3 if kind == "threads" else 1))
        r.init()
        if kind == "rev":
            r.step_reversed(20)
        elif kind == "split":
            r.step(7); r.step(13)
        else:
            r.step(20)
        return r.get_populations()
    base = run("plain")
    for kind in ("rev", "split", "threads"):
        assert np.array_equal(base, run(kind)), kind


def test_checkpoint_resume_bit_exact():
    a = oracle.Ref(5, 4, 3, 0.9, 1e-4, 1.0, 21)
    a.init(); a.step(10)
    b = oracle.Ref(5, 4, 3, 0.9, 1e-4, 1.0, 21)
    b.set_populations(a.get_populations(), a.step_count)
    a.step(10); b.step(10)
    assert np.array_equal(a.get_populations(), b.get_populations())


def test_bounce_back_one_fluid_layer_bruteforce():
    """P14/R12: nz=3 with walls -> one fluid layer z=1.  tau=1,kT=0: populations with c_z != 0 come back
    reversed at the same site; in-plane ones stream periodically."""
    nx, ny, nz = 4, 3, 3
    c, w, opp = oracle.tables()[:3]
    r = oracle.Ref(nx, ny, nz, 1.0, 0.0)
    r.set_walls_z(True)
    f = synthetic.random_population_field(nx, ny, nz, 8, w, spread=0.1)
    r.set_populations(f, 0)
    r.step(1)
    out = r.get_populations()
    assert np.array_equal(out[:, 0], f[:, 0]) and np.array_equal(out[:, 2], f[:, 2])   # solid layers untouched
    for y in range(ny):
        for x in range(nx):
            fs = oracle.collide_site(f[:, 1, y, x], 1.0)
            for i in range(27):
                if c[i][2] != 0:
                    assert out[opp[i], 1, y, x] == fs[i]
                else:
                    assert out[i, 1, (y + c[i][1]) % ny, (x + c[i][0]) % nx] == fs[i]
    rho, u = r.moments()
    assert (rho[0] == 0).all() and (rho[2] == 0).all()
    assert abs(rho[1].sum() - f[:, 1].sum()) < 1e-14                                      # mass stays in the fluid


def test_walls_conserve_mass_and_force_adds_momentum():
    r = oracle.Ref(4, 4, 8, 0.9, 1e-4, 1.0, 3)
    r.set_walls_z(True)
    r.init()
    m0 = r.diagnostics()[0]
    r.step(50)
    assert abs(r.diagnostics()[0] - m0) < 1e-13 * m0
    # periodic box + force: sum rho u = N rho0 g (t + 1/2) exactly (R13; reported u includes F/2)
    p = oracle.Ref(4, 4, 4, 0.9, 0.0, 1.0, 3)
    p.set_force(1e-6, 0.0, -2e-6)
    p.init()
    p.step(10)
    d = p.diagnostics()
    assert abs(d[1] / (64 * 1e-6 * 10.5) - 1) < 1e-11 and abs(d[3] / (-64 * 2e-6 * 10.5) - 1) < 1e-11 and abs(d[2]) < 1e-16


def test_argument_validation():
    import ctypes as C
    lib = oracle.load()
    h = C.c_void_p()
    assert lib.rflbm_ref_create(0, 4, 4, 1.0, 0.0, 1.0, 0, 0, C.byref(h)) == -1
    assert lib.rflbm_ref_create(4, 4, 4, 0.5, 0.0, 1.0, 0, 0, C.byref(h)) == -1
    assert lib.rflbm_ref_create(4, 4, 4, 1.0, -1.0, 1.0, 0, 0, C.byref(h)) == -1
    assert lib.rflbm_ref_create(4, 4, 4, 1.0, 0.0, 0.0, 0, 0, C.byref(h)) == -1
    assert lib.rflbm_ref_create(4, 4, 4, 1.0, 0.0, 1.0, 0, 7, C.byref(h)) == -1
    assert lib.rflbm_ref_create(4, 4, 2, 1.0, 0.0, 1.0, 0, 0, C.byref(h)) == 0
    assert lib.rflbm_ref_set_walls_z(h, 1) == -1          # nz < 3
    assert lib.rflbm_ref_step(h, 1) == -2                  # not initialised
    lib.rflbm_ref_destroy(h)


def test_stress_observable_is_second_hermite_moment():
    """Pi_ab = a_0,ab + a_1,ab (Eq.18-19) = rows k=4..9 of the paper's printed basis applied to the
    state; for an equilibrium state it is rho u_a u_b exactly (Eq.20)."""
    from paper_tables import exact_basis
    c, w = oracle.tables()[:2]
    E = np.array([[float(v) for v in row] for row in exact_basis(c)])
    nx, ny, nz = 5, 4, 6
    f = synthetic.random_population_field(nx, ny, nz, 8, w)
    r = oracle.Ref(nx, ny, nz, 0.8, 1e-4, 1.0, 2)
    r.set_walls_z(True)
    r.set_populations(f, 0)
    pi = r.stress()
    want = np.einsum("ki,izyx->kzyx", E[4:10], f)
    assert np.abs(pi[:, 1:-1] - want[:, 1:-1]).max() < 1e-15
    assert (pi[:, 0] == 0).all() and (pi[:, -1] == 0).all()           # solid layers
    r2 = oracle.Ref(nx, ny, nz, 0.8, 0.0)
    rho, u = synthetic.smooth_random_fields(nx, ny, nz, 3)
    r2.init(rho, u)
    idx = [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]
    eq = np.stack([rho * u[a] * u[b] for a, b in idx])
    assert np.abs(r2.stress() - eq).max() < 1e-15
