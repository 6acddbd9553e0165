"""P1/P6: the oracle's lattice and Hermite tables against what the paper prints (exact rationals)."""
from fractions import Fraction as Fr
from math import factorial

import numpy as np

import oracle
from paper_tables import CS2, exact_basis, table_I, table_II, weight_of


def test_velocity_set_is_d3q27_in_canonical_order():
    c, w, opp, pqr, e, b = oracle.tables()
    assert sorted(map(tuple, c.tolist())) == sorted((x, y, z) for x in (-1, 0, 1) for y in (-1, 0, 1) for z in (-1, 0, 1))
    # canonical order (R1)
    assert c[0].tolist() == [0, 0, 0]
    assert c[1:7].tolist() == [[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]]
    assert c[7:11].tolist() == [[1, 1, 0], [1, -1, 0], [-1, 1, 0], [-1, -1, 0]]
    assert c[11:15].tolist() == [[1, 0, 1], [1, 0, -1], [-1, 0, 1], [-1, 0, -1]]
    assert c[15:19].tolist() == [[0, 1, 1], [0, 1, -1], [0, -1, 1], [0, -1, -1]]
    assert c[19:27].tolist() == [[1, 1, 1], [1, 1, -1], [1, -1, 1], [1, -1, -1],
                                 [-1, 1, 1], [-1, 1, -1], [-1, -1, 1], [-1, -1, -1]]
    # Table I groups: 0 | 1-6 | 7-18 | 19-26 by |c|^2
    c2 = (c ** 2).sum(axis=1)
    assert c2.tolist() == [0] + [1] * 6 + [2] * 12 + [3] * 8
    for i in range(27):
        assert (c[opp[i]] == -c[i]).all()


def test_weights_match_table_I():
    c, w, *_ = oracle.tables()
    t1 = table_I()
    counts = {}
    for i in range(27):
        c2 = int((c[i] ** 2).sum())
        counts[c2] = counts.get(c2, 0) + 1
        assert w[i] == float(t1[c2][1])
    assert counts == {k: v[0] for k, v in t1.items()}
    assert sum(t1[k][0] * t1[k][1] for k in t1) == 1
    # second moment of the weights: sum w c_a c_b = cs2 delta_ab
    for a in range(3):
        for bb in range(3):
            s = sum(weight_of(ci) * int(ci[a]) * int(ci[bb]) for ci in c)
            assert s == (CS2 if a == bb else 0)


def test_basis_matches_table_II_polynomials():
    c, w, opp, pqr, e, b = oracle.tables()
    E = exact_basis(c)
    rows = table_II()
    assert [r[0] for r in rows] == list(range(27))
    for k in range(27):
        for i in range(27):
            assert abs(e[k, i] - float(E[k][i])) <= 2e-16, (k, i)
        # the printed polynomial factorises as H_p(cx) H_q(cy) H_r(cz) with the oracle's exponents (R2)
        n_k = rows[k][2]
        assert pqr[k].sum() == n_k


def test_orthogonality_norms_and_eq22():
    c, w, opp, pqr, e, b = oracle.tables()
    E = exact_basis(c)
    W = [weight_of(ci) for ci in c]
    rows = table_II()
    for k in range(27):
        for l in range(27):
            s = sum(W[i] * E[k][i] * E[l][i] for i in range(27))
            if k == l:
                assert s == rows[k][4], (k, s)                 # printed b_k, Eq.5
                assert abs(b[k] - float(s)) <= 2e-15 * float(s)     # oracle sums Eq.5 in doubles
                n, mu = rows[k][2], rows[k][3]
                assert Fr(factorial(n)) * CS2 ** n / mu == s    # Eq.22
                p, q, r = (int(v) for v in pqr[k])
                assert mu == factorial(n) // (factorial(p) * factorial(q) * factorial(r))
            else:
                assert s == 0, (k, l)
    # completeness: Eq.10 is the exact inverse of Eq.4
    for i in range(27):
        for j in range(27):
            s = sum(W[i] * E[k][i] * E[k][j] / rows[k][4] for k in range(27))
            assert s == (1 if i == j else 0)


def test_roundtrip_eq4_eq10():
    from paper_2507_08820_b200 import synthetic
    c, w, opp, pqr, e, b = oracle.tables()
    f = synthetic.random_populations(1, 5)
    for v in f:
        m = oracle.moments_of(v)
        back = w * ((m / b) @ e)
        assert np.abs(back - v).max() < 2e-15


def test_equilibrium_product_closed_form_exact():
    """P6: Eq.25 with Eq.20 equals rho*phi(cx,ux)phi(cy,uy)phi(cz,uz), phi(0,u)=2/3-u^2,
    phi(+-1,u)=1/6 +- u/2 + u^2/2, and its 27 Hermite moments are rho ux^p uy^q uz^r (rational check
    of the identity, then the oracle's doubles against it)."""
    c, w, opp, pqr, e, b = oracle.tables()
    E = exact_basis(c)
    W = [weight_of(ci) for ci in c]
    rows = table_II()
    rho, u = Fr(9, 8), (Fr(1, 17), Fr(-2, 31), Fr(3, 41))

    def phi(cc, uu):
        return Fr(2, 3) - uu * uu if cc == 0 else Fr(1, 6) + cc * uu / 2 + uu * uu / 2

    M = [rho * u[0] ** int(pqr[k][0]) * u[1] ** int(pqr[k][1]) * u[2] ** int(pqr[k][2]) for k in range(27)]
    for i in range(27):
        f_sum = W[i] * sum(M[k] * E[k][i] / rows[k][4] for k in range(27))
        f_prod = rho * phi(int(c[i][0]), u[0]) * phi(int(c[i][1]), u[1]) * phi(int(c[i][2]), u[2])
        assert f_sum == f_prod
    f0 = oracle.equilibrium(float(rho), [float(x) for x in u])
    for i in range(27):
        f_prod = rho * phi(int(c[i][0]), u[0]) * phi(int(c[i][1]), u[1]) * phi(int(c[i][2]), u[2])
        assert abs(f0[i] - float(f_prod)) < 2e-16
    m = oracle.moments_of(f0)
    for k in range(27):
        assert abs(m[k] - float(M[k])) < 2e-15
