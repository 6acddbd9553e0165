"""Exact (rational) D3Q27 tables read from the golden fixtures typed from the paper.

Test-side helper: parses tests/golden/table_I.txt and table_II.txt (Table I / II) with
fractions.Fraction so that the oracle's double tables can be pinned against what the paper prints.
Holds no oracle or CUDA code.
"""
from __future__ import annotations

import os
from fractions import Fraction as Fr

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
CS2 = Fr(1, 3)


def table_I():
    """{ |c|^2 : (count, weight) } as printed."""
    out = {}
    with open(os.path.join(GOLDEN, "table_I.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            _, count, c2, w = line.split()
            out[int(c2)] = (int(count), Fr(w))
    return out


def table_II():
    """list of (k, polynomial source, n_k, mu_k, b_k) as printed."""
    rows = []
    with open(os.path.join(GOLDEN, "table_II.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            k, poly, n, mu, b = [s.strip() for s in line.split(";")]
            rows.append((int(k), poly, int(n), int(mu), Fr(b)))
    return rows


def eval_poly(poly: str, c):
    env = {"cx": Fr(int(c[0])), "cy": Fr(int(c[1])), "cz": Fr(int(c[2])), "cs2": CS2}
    return Fr(eval(poly, {"__builtins__": {}}, env))


def weight_of(c):
    t1 = table_I()
    return t1[int(c[0]) ** 2 + int(c[1]) ** 2 + int(c[2]) ** 2][1]


def exact_basis(c_list):
    """E[k][i] (Fraction) for the given velocity list, from the printed polynomials."""
    rows = table_II()
    return [[eval_poly(poly, c) for c in c_list] for (_, poly, _, _, _) in rows]
