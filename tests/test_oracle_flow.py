"""Pins of the oracle under a general velocity gradient tensor kappa (eqs 18, 21).
Expected values are closed forms of the Euler map of eqs (44), (45) (stationary covariance of a linear map by its
discrete Lyapunov equation, solved by scipy; powers of the matrix 1 + dt kappa by numpy) or invariants; none comes
from the oracle or from the CUDA path.
"""
import math
import os

import numpy as np
import scipy.linalg

import oracle

NT = min(8, os.cpu_count() or 1)

# a traceless, non-symmetric tensor with every kind of entry: a transposed operand, a wrong index or a dropped
# term of the affine step changes the stationary stress below by many standard errors
KAPPA = np.array([[0.30, 0.80, 0.00],
                  [-0.20, -0.10, 0.50],
                  [0.10, 0.00, -0.20]])


def test_simple_shear_is_the_xy_entry_of_the_tensor():
    """eq (60): kappa_xy = gamma_dot, all other entries zero."""
    a = oracle.Ensemble(8, 32, seed=5); b = oracle.Ensemble(8, 32, seed=5)
    k = np.zeros((3, 3)); k[0, 1] = 0.3
    sa = a.run(60, shear_rate=0.3, stress_every=1)
    sb = b.run_kappa(60, k, stress_every=1)
    assert np.array_equal(a.S, b.S) and np.array_equal(a.Z, b.Z)
    assert np.allclose(a.R, b.R, rtol=0, atol=1e-12) and np.allclose(a.A, b.A, rtol=0, atol=1e-12)
    assert np.allclose(sa, sb, rtol=0, atol=1e-10)


def test_anchors_follow_the_powers_of_the_affine_map():
    """eq (45): A_j(t + dt) = (1 + dt kappa) A_j(t) and nothing else moves an anchor ("the anchoring point
    of a slip-spring moves only by the external flow").  With zeta_s huge no slip-spring hops, is created or is
    destroyed, so after n steps every anchor is (1 + dt kappa)^n A_j(0)."""
    e = oracle.Ensemble(8, 16, zeta_s=1e12, seed=9)
    A0, S0 = e.A.copy(), e.S.copy()
    n = 37
    e.run_kappa(n, KAPPA)
    assert np.array_equal(e.S, S0)
    F = np.linalg.matrix_power(np.eye(3) + e.p.dt * KAPPA, n)
    assert np.allclose(e.A, A0 @ F.T, rtol=0, atol=1e-12)


def _rouse_stationary_stress(N, dt, kappa):
    """Free Rouse chain, Z = 0, under steady kappa: per normal mode p (lambda_p = 4 sin^2(p pi / 2N), App. B of
    SURVEY.md) the Euler map of eq (44) is X' = [(1 - 3 lambda_p dt) 1 + dt kappa] X + sqrt(2 dt) w, whose stationary
    covariance solves C = M C M^T + 2 dt 1; sum over bonds of <b_a b_b> = sum_p lambda_p C_p, so by eq (16)
    <sigma_ab> = 3 sum_p lambda_p C_p,ab - N delta_ab (the p = 0 mode carries no bond)."""
    sig = -float(N) * np.eye(3)
    for p in range(1, N):
        lam = 4.0 * math.sin(p * math.pi / (2 * N)) ** 2
        Mp = (1.0 - 3.0 * lam * dt) * np.eye(3) + dt * kappa
        Cp = scipy.linalg.solve_discrete_lyapunov(Mp, 2.0 * dt * np.eye(3))
        sig += 3.0 * lam * Cp
    return sig


def test_rouse_chain_under_general_kappa_reaches_the_lyapunov_stress():
    N, M, dt = 8, 2048, 0.01
    want = _rouse_stationary_stress(N, dt, KAPPA)
    # sanity of the closed form itself: without flow it is the equilibrium value of App. B
    kp = 12 * np.sin(np.arange(1, N) * math.pi / (2 * N)) ** 2
    assert np.allclose(_rouse_stationary_stress(N, dt, np.zeros((3, 3))),
                       (np.sum(1.0 / (1.0 - kp * dt / 2)) - N) * np.eye(3), atol=1e-12)
    e = oracle.Ensemble(N, M, n_0=0.0, dt=dt, seed=77)
    e.run_kappa(800, KAPPA, n_threads=NT)                        # > 7 Rouse times (1.09 tau0)
    # independent blocks: chains x well separated times; standard error over chains of the time average
    acc = np.zeros((M, 6)); n_s = 0
    for _ in range(40):
        e.run_kappa(50, KAPPA, n_threads=NT)
        acc += np.array([e.chain_stress(k)[0] for k in range(M)]); n_s += 1
    per_chain = acc / n_s
    mean, se = per_chain.mean(0), per_chain.std(0, ddof=1) / math.sqrt(M)
    comp = [(0, 0), (1, 1), (2, 2), (0, 1), (1, 2), (2, 0)]
    for t, (a, b) in enumerate(comp):
        assert abs(mean[t] - want[a, b]) < 4.0 * se[t] + 1e-3, (t, mean[t], want[a, b], se[t])
    # the pin has teeth: the transposed tensor gives a different normal-stress difference
    wrong = _rouse_stationary_stress(N, dt, KAPPA.T)
    assert abs((wrong[0, 0] - wrong[1, 1]) - (want[0, 0] - want[1, 1])) > 20 * math.hypot(se[0], se[1])


def test_groups_of_chains_each_follow_their_own_tensor():
    """One tensor per block of chains: a run with two groups equals two separate runs of the halves
    (Philox is keyed by the global chain index)."""
    k2 = np.stack([KAPPA, -0.5 * KAPPA.T])
    both = oracle.Ensemble(8, 24, seed=3)
    both.run_kappa(40, k2, chains_per_group=12)
    for g in range(2):
        half = oracle.Ensemble(8, 12, seed=3, chain_offset=12 * g)
        half.run_kappa(40, k2[g])
        sl = slice(12 * g, 12 * g + 12)
        assert np.array_equal(both.S[sl], half.S) and np.array_equal(both.R[sl], half.R)
        assert np.array_equal(both.A[sl], half.A)
