"""A/B pin of DESIGN.md reading R24: the bead noise w_i of eqs (46), (47) is drawn by
Box-Muller from 16-bit codes in the RNG contract shared with the GPU.  P:L307 fixes no generator and no
resolution, so the reading is admissible -- but only if the DYNAMICS do not see it.  The oracle keeps the
full-resolution law it was first written with (noise_bits = 23: 23-bit uniforms, |z| <= 5.77) and these tests
run both laws side by side: equilibrium bond length, <Z>, G(t) over five correlator levels and the start-up
viscosity growth at shear rate 0.1 must agree within their combined standard errors.  Both arms are the
oracle; no value comes from the CUDA path.
"""
import math
import os

import numpy as np
from scipy import stats

import oracle

NT = min(8, os.cpu_count() or 1)
N, M = 16, 4096


def test_box_muller_23bit_law_is_a_standard_normal():
    """The full-resolution transform itself: 2e5 normals from consecutive Philox words pass a
    Kolmogorov-Smirnov test against N(0,1) and have the moments of a normal; special inputs give the
    closed forms r = sqrt(-2 ln u), theta = 0 -> (r, 0)."""
    z = []
    for q in range(50000):
        w = oracle.stream(7, oracle.DOM_NOISE, 3, 11, q)
        z.extend(oracle.box_muller23(w[0], w[1])); z.extend(oracle.box_muller23(w[2], w[3]))
    z = np.array(z)
    assert stats.kstest(z, "norm").pvalue > 1e-3
    n = z.size
    assert abs(z.mean()) < 4.5 / math.sqrt(n)
    assert abs((z ** 2).mean() - 1.0) < 4.5 * math.sqrt(2.0 / n)
    assert abs((z ** 4).mean() - 3.0) < 4.5 * math.sqrt(96.0 / n)
    # theta = 2 pi (u_b - 1/2) with u_b = (k + 1/2) 2^-23: code 2^22 gives theta = pi 2^-23 ~ 0;
    # u_a code 0 gives the largest radius sqrt(-2 ln 2^-24) = sqrt(48 ln 2) = 5.768
    z0, z1 = oracle.box_muller23(0 << 9, (1 << 22) << 9)
    assert math.isclose(z0, math.sqrt(48 * math.log(2.0)), rel_tol=1e-12) and abs(z1) < 1e-5
    # the 16-bit law's largest radius is sqrt(34 ln 2) = 4.855 (reading R24)
    z0, z1 = oracle.box_muller((1 << 15) << 16)
    assert math.isclose(z0, math.sqrt(34 * math.log(2.0)), rel_tol=1e-8) and abs(z1) < 3e-4      # cos(pi 2^-16) = 1 - 1.2e-9


def _equilibrium_observables(bits, seed):
    """bond^2, <Z> (each with its standard error over chains, from 15 snapshots 400 steps apart) and G(t)."""
    e = oracle.Ensemble(N, M, seed=seed, noise_bits=bits)
    e.run(600, n_threads=NT)
    corr = oracle.Correlator(M, levels=5, bins=16, groups=32)
    b2, zz = [], []
    for _ in range(15):
        e.run(400, sample_every=10, corr=corr, n_threads=NT)
        b2.append((np.diff(e.R, axis=1) ** 2).sum(2).mean(1))      # per chain, mean over its bonds
        zz.append(e.Z.astype(np.float64))
    b2 = np.array(b2); zz = np.array(zz)
    # snapshots 4 tau0 apart: bonds decorrelate (Rouse time 4.3 tau0 for the slowest mode only), Z does so
    # more slowly: take the standard error from the chain-to-chain scatter of the TIME-AVERAGED value
    t, G, se = corr.result(N, 0.1)
    return (b2.mean(), b2.mean(0).std() / math.sqrt(M)), (zz.mean(), zz.mean(0).std() / math.sqrt(M)), (t, G, se)


def test_equilibrium_bond_length_slipspring_number_and_gt_do_not_depend_on_the_noise_resolution():
    (b16, sb16), (z16, sz16), (t, G16, se16) = _equilibrium_observables(16, seed=101)
    (b23, sb23), (z23, sz23), (_, G23, se23) = _equilibrium_observables(23, seed=102)
    assert abs(b16 - b23) < 3.0 * math.hypot(sb16, sb23), (b16, b23, sb16, sb23)
    assert abs(z16 - z23) < 3.0 * math.hypot(sz16, sz23), (z16, z23, sz16, sz23)
    # both sit where the paper puts them: <Z> = N/N0 (eq 10) and the Euler map's bond^2 = 1.03 (O(dt) above 1)
    assert abs(z16 - N / 4.0) < 0.1 and abs(b16 - 1.03) < 0.01
    assert len(t) == 16 + 4 * 8                                   # five levels: lags up to 24 tau0
    zs = (G16 - G23) / np.hypot(se16, se23)
    assert np.abs(zs).max() < 4.5, (np.abs(zs).max(), t[np.abs(zs).argmax()])
    assert (np.abs(zs) < 3.0).mean() >= 0.95
    assert G16[0] > 20 * np.hypot(se16[0], se23[0])                # the comparison resolves G(0) to a few per cent


def _startup(bits, seed, rate=0.1, marks=(50, 100, 200, 400, 800)):
    e = oracle.Ensemble(N, M, seed=seed, noise_bits=bits)
    e.run(600, n_threads=NT)
    out = []
    done = 0
    for m in marks:
        e.run(m - done, shear_rate=rate, n_threads=NT); done = m
        sxy = np.array([e.chain_stress(k)[0][3] for k in range(M)])
        out.append((sxy.mean() / (N * rate), sxy.std() / math.sqrt(M) / (N * rate)))      # eta+ (eq 61, R13) and its SE
    return np.array(out)


def test_startup_viscosity_growth_does_not_depend_on_the_noise_resolution():
    a = _startup(16, seed=103); b = _startup(23, seed=104)
    zs = (a[:, 0] - b[:, 0]) / np.hypot(a[:, 1], b[:, 1])
    assert np.abs(zs).max() < 3.5, zs
    assert a[-1, 0] > a[0, 0] > 0 and a[-1, 0] > 8 * a[-1, 1]     # the growth curve itself is resolved
