"""P2/P3: Philox4x32-10 known answers and the uniform->normal map (R8)."""
import math
import os

import numpy as np

import oracle


def test_philox_known_answers(golden_dir):
    n = 0
    with open(os.path.join(golden_dir, "philox_kat.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            v = [int(t, 16) for t in line.replace("->", " ").split()]
            assert len(v) == 10
            out = oracle.philox(v[0:4], v[4:6])
            assert out.tolist() == v[6:10]
            n += 1
    assert n == 3


def test_philox_python_bigint_restatement():
    """Independent restatement with Python integers (brute force) on random counters/keys."""
    rng = np.random.default_rng(5)
    M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
    for _ in range(50):
        ctr = [int(x) for x in rng.integers(0, 2 ** 32, 4)]
        key = [int(x) for x in rng.integers(0, 2 ** 32, 2)]
        c, k = list(ctr), list(key)
        for r in range(10):
            p0, p1 = M0 * c[0], M1 * c[2]
            c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
            k = [(k[0] + W0) & 0xFFFFFFFF, (k[1] + W1) & 0xFFFFFFFF]
        assert oracle.philox(ctr, key).tolist() == c


def test_box_muller_closed_form_points():
    z = oracle.normal_pair(0, 0)
    assert abs(z[0] - math.sqrt(66 * math.log(2))) < 1e-8       # u_b = 2^-33: cos ~ 1 - 1e-19
    assert abs(z[1] - math.sqrt(66 * math.log(2)) * math.sin(2 * math.pi * 2.0 ** -33)) < 1e-20
    # u_a = 1/2 exactly is not representable ((x+0.5)/2^32), use x = 2^31: u_a = 1/2 + 2^-33
    ua = (2 ** 31 + 0.5) / 2 ** 32
    R = math.sqrt(-2 * math.log(ua))
    # u_b = 1/4 + 2^-33 -> angle pi/2 + eps: (cos, sin) ~ (-eps, 1)
    z = oracle.normal_pair(2 ** 31, 2 ** 30)
    assert abs(z[1] - R) < 1e-15 and abs(z[0] + R * 2 * math.pi * 2.0 ** -33) < 5e-16   # angle 2*pi*u_b is rounded to double
    # u_b = 1/2 + 2^-33 -> (-1, -eps)
    z = oracle.normal_pair(2 ** 31, 2 ** 31)
    assert abs(z[0] + R) < 1e-15
    # fp32 mode uses the top 24 bits
    z32 = oracle.normal_pair(0xFFFFFFFF, 0, oracle.F32)
    ua = (2 ** 24 - 0.5) / 2 ** 24
    assert abs(z32[0] - math.sqrt(-2 * math.log(ua))) < 1e-12
    # bound on the tail: |r| <= sqrt(66 ln 2)
    assert abs(oracle.normal_pair(0, 2 ** 31)[0]) <= 6.7638


def test_normals_statistics_and_mode_map():
    r = oracle.Ref(32, 32, 16, 1.0, 1e-4, 1.0, 123)
    words, normals = r.debug_rng(7)
    # mode map: call q, pair h -> k = 4+4q+2h (first), k+1 (second); word layout words[4q+m]
    for (s, q, h) in [(0, 0, 0), (5, 3, 1), (16383, 5, 0), (777, 5, 1)]:
        wa = int(words.reshape(24, -1)[4 * q + 2 * h, s])
        wb = int(words.reshape(24, -1)[4 * q + 2 * h + 1, s])
        z = oracle.normal_pair(wa, wb)
        k = 4 + 4 * q + 2 * h
        assert normals.reshape(23, -1)[k - 4, s] == z[0]
        if k + 1 < 27:
            assert normals.reshape(23, -1)[k + 1 - 4, s] == z[1]
    # counter layout (site, t>>32, t&0xffffffff, q), key = (seed lo, seed hi)
    w = oracle.philox([5, 0, 7, 3], [123, 0])
    assert words.reshape(24, -1)[12:16, 5].tolist() == w.tolist()
    x = normals.ravel()
    n = x.size                                             # 376 832 draws
    assert abs(x.mean()) < 4.0 / math.sqrt(n)
    assert abs(x.var() - 1.0) < 4.0 * math.sqrt(2.0 / n)
    kurt = ((x - x.mean()) ** 4).mean() / x.var() ** 2
    assert abs(kurt - 3.0) < 4.0 * math.sqrt(24.0 / n)
    # different modes / sites / steps are uncorrelated
    nm = normals.reshape(23, -1)
    cm = np.corrcoef(nm)
    assert np.abs(cm - np.eye(23)).max() < 5.0 / math.sqrt(nm.shape[1])
    w2, n2 = r.debug_rng(8)
    assert abs(np.corrcoef(normals.ravel(), n2.ravel())[0, 1]) < 5.0 / math.sqrt(n)
    # uniform words: mean of the top bit
    assert abs((words >> 31).mean() - 0.5) < 4 * 0.5 / math.sqrt(words.size)
