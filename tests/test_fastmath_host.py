"""CPU check of the CUDA path's own Box-Muller routines (csrc/rflbm_fastmath.cuh compiled for the host through the
test shim tests/fastmath_host_check.cpp) against 80-bit long-double libm over the whole 32-bit input range.

This is host logic of the product, not the oracle: nothing under oracle/ is used here.  The device differs from
this host build only in the reciprocal-square-root seed (MUFU.RSQ64H vs a truncated 1/sqrt), which the third-order
update absorbs; the GPU parity tests compare the device normals with the oracle's libm normals directly."""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "fastmath_host_check.cpp")
INC = os.path.join(ROOT, "paper_2507_08820_b200", "csrc")
LD = np.longdouble
pytestmark = pytest.mark.skipif(np.finfo(LD).nmant < 63, reason="needs 80-bit long double")


@pytest.fixture(scope="module")
def fm(tmp_path_factory):
    so = str(tmp_path_factory.mktemp("fm") / "libfm.so")
    subprocess.run(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC", "-I", INC, "-o", so, SRC], check=True)
    return C.CDLL(so)


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def _inputs(n, seed):
    rng = np.random.default_rng(seed)
    special = [0, 1, 2, 3, 2 ** 32 - 1, 2 ** 32 - 2, 2 ** 31, 2 ** 31 - 1, 2 ** 31 + 1, 2 ** 23 - 1, 2 ** 23, 2 ** 22,
               2 ** 22 - 1, 2 ** 22 + 1]
    special += [2 ** k for k in range(32)] + [2 ** k - 1 for k in range(1, 32)]
    special += [j << 23 for j in range(0, 512, 37)] + [(j << 23) - 1 for j in range(1, 512, 41)]
    x = np.concatenate([rng.integers(0, 2 ** 32, n, dtype=np.uint64), np.array(special, dtype=np.uint64)])
    return np.ascontiguousarray(x, dtype=np.uint32)


def test_tables_match_long_double(fm):
    lg = np.empty(2 * 256)
    sc = np.empty(2 * 512)
    fm.fm_tables(_ptr(lg), _ptr(sc))
    inv, ln = lg[0::2], lg[1::2]
    # -2 ln c_j stored consistently with the stored 1/c_j; bucket 149 is exactly c = 1
    assert np.abs(ln.astype(LD) - 2 * np.log(inv.astype(LD))).max() < 2e-16
    assert inv[149] == 1.0 and ln[149] == 0.0
    j = np.arange(512).astype(LD)
    th = (LD(2) * np.arctan(LD(1)) * 4) * (j * 2 ** 23 + 2 ** 22 + LD(0.5)) / LD(2 ** 32)
    assert np.abs(sc[0::2].astype(LD) - np.sin(th)).max() < 1.2e-16
    assert np.abs(sc[1::2].astype(LD) - np.cos(th)).max() < 1.2e-16


def test_neg2_log_and_sqrt(fm):
    x = _inputs(2_000_000, 1)
    n = len(x)
    W = np.empty(n)
    fm.fm_neg2_log(_ptr(x), _ptr(W), C.c_long(n))
    Wr = -2 * np.log((x.astype(LD) + LD(0.5)) / LD(2 ** 32))
    rel = np.abs((W.astype(LD) - Wr) / Wr).astype(float)
    assert rel.max() < 4 * 2.0 ** -53, rel.max()                 # full RELATIVE accuracy, also as u -> 1
    assert W.min() > 0 and abs(W.max() - 2 * np.log(2.0 ** 33)) < 1e-13
    R = np.empty(n)
    fm.fm_sqrt(_ptr(W), _ptr(R), C.c_long(n))
    rel = np.abs((R.astype(LD) - np.sqrt(W.astype(LD))) / np.sqrt(W.astype(LD))).astype(float)
    assert rel.max() < 2.5 * 2.0 ** -53, rel.max()


def test_sincos_and_normal_pair(fm):
    xa, xb = _inputs(2_000_000, 2), _inputs(2_000_000, 3)
    n = len(xa)
    s, c = np.empty(n), np.empty(n)
    fm.fm_sincos(_ptr(xb), _ptr(s), _ptr(c), C.c_long(n))
    th = (LD(2) * np.arctan(LD(1)) * 4) * (xb.astype(LD) + LD(0.5)) / LD(2 ** 32)
    assert np.abs(s.astype(LD) - np.sin(th)).max() < 4 * 2.0 ** -53
    assert np.abs(c.astype(LD) - np.cos(th)).max() < 4 * 2.0 ** -53
    z0, z1 = np.empty(n), np.empty(n)
    fm.fm_normal_pair(_ptr(xa), _ptr(xb), _ptr(z0), _ptr(z1), C.c_long(n))
    R = np.sqrt(-2 * np.log((xa.astype(LD) + LD(0.5)) / LD(2 ** 32)))
    err = np.maximum(np.abs(z0.astype(LD) - R * np.cos(th)), np.abs(z1.astype(LD) - R * np.sin(th))).astype(float)
    assert (err / R.astype(float)).max() < 8 * 2.0 ** -53        # a few ulp of the radius
    assert err.max() < 5e-15                                      # absolute: |z| <= 6.77
