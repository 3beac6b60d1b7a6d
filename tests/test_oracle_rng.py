"""Pin P1: the oracle's Philox4x32-10, U23 and Box-Muller.

Pinned against (a) the published known-answer vectors of the generator (tests/golden),
(b) a big-integer restatement of the algorithm's description written here, (c) the
exact moments / distribution a Box-Muller pair must have.
"""
import math
import os

import numpy as np
from scipy import stats

import oracle

M0, M1 = 0xD2511F53, 0xCD9E8D57
W0, W1 = 0x9E3779B9, 0xBB67AE85


def philox_bigint(ctr, key, rounds=10):
    """Salmon et al. SC'11: an S-P network; per round two 32x32->64 products, the high
    halves are XORed with the other two words and the round key, key bumped by Weyl
    constants.  Python integers, no 32-bit tricks."""
    c = list(ctr); k = list(key)
    for _ in range(rounds):
        p0 = M0 * c[0]; p1 = M1 * c[2]
        c = [((p1 >> 32) ^ c[1] ^ k[0]) & 0xFFFFFFFF, p1 & 0xFFFFFFFF,
             ((p0 >> 32) ^ c[3] ^ k[1]) & 0xFFFFFFFF, p0 & 0xFFFFFFFF]
        k = [(k[0] + W0) & 0xFFFFFFFF, (k[1] + W1) & 0xFFFFFFFF]
    return c


def test_known_answer_vectors(golden_dir):
    n = 0
    for line in open(os.path.join(golden_dir, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        assert oracle.philox(w[0:4], w[4:6]) == w[6:10]
        assert philox_bigint(w[0:4], w[4:6]) == w[6:10]
        n += 1
    assert n == 2


def test_against_bigint_restatement_random_inputs():
    rng = np.random.default_rng(0)
    for _ in range(300):
        ctr = [int(x) for x in rng.integers(0, 2 ** 32, 4)]
        key = [int(x) for x in rng.integers(0, 2 ** 32, 2)]
        assert oracle.philox(ctr, key) == philox_bigint(ctr, key)


def test_stream_counter_layout():
    # counter = (step lo, domain<<28 | step bits 32..59, chain, item), key = (seed lo, seed hi)
    seed, dom, step, chain, item = 0x1234567890ABCDEF, 3, (5 << 32) | 77, 123456, 9
    want = philox_bigint([77, (3 << 28) | 5, 123456, 9], [0x90ABCDEF, 0x12345678])
    assert oracle.stream(seed, dom, step, chain, item) == want
    # every coordinate matters
    base = oracle.stream(1, 0, 0, 0, 0)
    assert len({tuple(base), tuple(oracle.stream(2, 0, 0, 0, 0)), tuple(oracle.stream(1, 1, 0, 0, 0)),
                tuple(oracle.stream(1, 0, 1, 0, 0)), tuple(oracle.stream(1, 0, 0, 1, 0)),
                tuple(oracle.stream(1, 0, 0, 0, 1)), tuple(oracle.stream(1 << 32, 0, 0, 0, 0)),
                tuple(oracle.stream(1, 0, 1 << 32, 0, 0))}) == 8


def test_u23_is_exact_midpoint_grid():
    assert oracle.u23(0) == 0.5 * 2.0 ** -23
    assert oracle.u23(0xFFFFFFFF) == 1.0 - 0.5 * 2.0 ** -23
    assert oracle.u23(0x80000000) == 0.5 + 0.5 * 2.0 ** -23
    for w in (0, 511, 512, 0x12345678, 0xFFFFFFFF):
        u = oracle.u23(w)
        assert u == float(np.float32(u))            # representable in fp32, so GPU and oracle see the same u


def test_threshold23_equivalence_brute_force():
    # "u < p" <=> code < T(p), checked over every code near the threshold for many p
    rng = np.random.default_rng(1)
    ps = list(rng.random(200)) + [0.0, 1.0, 0.1, 0.025, 0.5, 2.0 ** -24, 1 - 2.0 ** -24, 3 * 2.0 ** -23]
    for p in ps:
        T = oracle.threshold23(p)
        lo = max(0, T - 3); hi = min(2 ** 23, T + 3)
        for k in range(lo, hi):
            u = (k + 0.5) * 2.0 ** -23
            assert (u < p) == (k < T), (p, k, T)
        # number of accepted codes out of 2^23 is T exactly
        assert 0 <= T <= 2 ** 23
        assert abs(T / 2 ** 23 - p) <= 2.0 ** -23


def test_box_muller_closed_form_and_polar_identity():
    # r^2 = -2 ln u_a and angle 2 pi (u_b - 1/2), "Box-Muller transform"; reading R24:
    # u_a, u_b = midpoints of the 16-bit codes in the low / high half of one Philox word
    for w in [0, 0xFFFFFFFF, 0x80000000, 0x12345678, 0x9ABCDEF0, 0x0000FFFF, 0xFFFF0000]:
        z0, z1 = oracle.box_muller(w)
        ua = ((w & 0xFFFF) + 0.5) / 65536.0
        ub = ((w >> 16) + 0.5) / 65536.0
        assert math.isclose(z0 * z0 + z1 * z1, -2.0 * math.log(ua), rel_tol=1e-13)
        assert math.isclose(math.atan2(z1, z0), 2 * math.pi * (ub - 0.5), rel_tol=1e-12, abs_tol=1e-15)
    z0, z1 = oracle.box_muller(0)
    assert abs(math.hypot(z0, z1)) < 4.86          # |normal| <= sqrt(2 ln 2^17) = 4.855


def test_box_muller_16bit_grid_moments_by_enumeration():
    """Reading R24 spends 16 bits per Box-Muller input.  The resulting normal is a discrete
    law on 2^16 radii x 2^16 angles; its moments follow EXACTLY from enumerating the radii
    (the angle average of cos^2 over the equally spaced half-offset grid is exactly 1/2, of
    cos^4 exactly 3/8): E z^2 = E r^2 / 2, E z^4 = 3 E r^4 / 8.  They must agree with the
    standard normal's to far better than the O(dt) = 1e-2 bias of the Euler scheme."""
    k = np.arange(65536, dtype=np.float64)
    r2 = -2.0 * np.log((k + 0.5) / 65536.0)
    th = 2 * np.pi * ((k + 0.5) / 65536.0 - 0.5)
    assert abs(np.mean(np.cos(th) ** 2) - 0.5) < 1e-15 and abs(np.mean(np.cos(th) ** 4) - 0.375) < 1e-15
    assert abs(np.mean(np.cos(th))) < 1e-15 and abs(np.mean(np.cos(th) * np.sin(th))) < 1e-15
    var = 0.5 * r2.mean(); m4 = 0.375 * (r2 ** 2).mean()
    assert abs(var - 1.0) < 1e-5, var
    assert abs(m4 - 3.0) < 5e-4, m4
    # the oracle's own box_muller lands on that grid: radius from the low half, angle from the high half
    for ka, kb in [(0, 0), (65535, 0), (123, 45678), (40000, 65535)]:
        z0, z1 = oracle.box_muller(ka | (kb << 16))
        assert math.isclose(z0 * z0 + z1 * z1, r2[ka], rel_tol=1e-13)
        assert math.isclose(math.atan2(z1, z0), th[kb], rel_tol=1e-12, abs_tol=1e-15)


def test_stream_normals_are_standard_normal():
    n = 40000
    z = np.array([oracle.stream_normal(7, oracle.DOM_NOISE, 3, 11, m) for m in range(n)])
    assert abs(z.mean()) < 4 / math.sqrt(n)
    assert abs(z.var() - 1) < 4 * math.sqrt(2 / n)
    assert abs((z ** 4).mean() - 3) < 4 * math.sqrt(96 / n)
    assert stats.kstest(z, "norm").pvalue > 1e-3
    # the eight normals of one call are uncorrelated with each other
    q = z.reshape(-1, 8)
    c = np.corrcoef(q.T)
    assert np.abs(c - np.eye(8)).max() < 5 / math.sqrt(n / 8)
    # normal m comes from call m>>3: word e -> z_{2e}, z_{2e+1}
    w = oracle.stream(7, oracle.DOM_NOISE, 3, 11, 5)
    want = [x for e in range(4) for x in oracle.box_muller(w[e])]
    assert [z[40 + i] for i in range(8)] == want

