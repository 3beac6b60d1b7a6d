"""Pins P2, P5 (deterministic part), P7, P8 and the stress definitions of the oracle
(DESIGN.md section 5).  Cheap, exact or near-exact checks; statistical pins of the
dynamics live in test_oracle_dynamics.py.  P:Lnnn = PAPER.md line nnn.
"""
import ctypes as C
import math

import numpy as np

import oracle


def _one_chain(N, R, A=None, S=None, n_s=0.5, n_0=4.0, dt=0.01, zeta_s=0.1, seed=1):
    e = oracle.Ensemble(N, 1, n_s=n_s, n_0=n_0, zeta_s=zeta_s, dt=dt, seed=seed, init=False)
    e.R[0] = R
    if A is not None:
        Z = len(S)
        e.A[0, :Z] = A; e.S[0, :Z] = S; e.Z[0] = Z
    return e


# ----------------------------------------------------------------------------- hop, P2
def test_hop_glauber_detailed_balance_identity():
    """P:L164-L172 eqs (23),(24): W(s->s+1)/W(s+1->s) = exp(-[U(s+1)-U(s)]/kT) with
    U(s) = (3/2N_s)|R_s - A|^2 (eq 1).  1 - tanh x = 2/(1+e^{2x})."""
    rng = np.random.default_rng(3)
    for n_s in (0.5, 1.3):
        R = 0.3 * rng.normal(size=(5, 3)); A = rng.normal(size=3) * 0.2 + R[2]
        U = 1.5 / n_s * ((R - A) ** 2).sum(1)
        for s in range(1, 5):                       # pair (s, s+1), 1-based
            e = _one_chain(5, R, [A], [s], n_s=n_s)
            pp, _ = e.hop_probabilities(0, 0)
            e2 = _one_chain(5, R, [A], [s + 1], n_s=n_s)
            _, pm = e2.hop_probabilities(0, 0)
            assert math.isclose(pp / pm, math.exp(-(U[s] - U[s - 1])), rel_tol=1e-7)
            # the rate itself: (dt/zeta_s) * 2/(1+exp(dU))
            assert math.isclose(pp, 0.1 * 2 / (1 + math.exp(U[s] - U[s - 1])), rel_tol=1e-7)


def test_hop_stationary_vector_is_boltzmann_on_three_beads():
    """Brute force on N = 3 with frozen beads: the 3x3 transition matrix built from the
    oracle's probabilities has stationary vector ~ exp(-U_i) (eq 1)."""
    rng = np.random.default_rng(4)
    R = 0.5 * rng.normal(size=(3, 3)); A = rng.normal(size=3) * 0.3 + R[1]
    P = np.zeros((3, 3))
    for s in (1, 2, 3):
        pp, pm = _one_chain(3, R, [A], [s]).hop_probabilities(0, 0)
        if s == 3:
            assert pp == 0.0                        # eq (48): 0 for S_j = N
        if s == 1:
            assert pm == 0.0                        # eq (49): 0 for S_j = 1
        if s < 3:
            P[s - 1, s] = pp
        if s > 1:
            P[s - 1, s - 2] = pm
        P[s - 1, s - 1] = 1 - pp - pm
    w, v = np.linalg.eig(P.T)
    pi = np.real(v[:, np.argmax(np.real(w))]); pi /= pi.sum()
    boltz = np.exp(-1.5 / 0.5 * ((R - A) ** 2).sum(1)); boltz /= boltz.sum()
    assert np.allclose(pi, boltz, rtol=1e-8)


def test_hop_cap_one_half():
    """'each transition probability does not exceed 1/2' (binds only for dt/zeta_s > 1/4)."""
    R = np.array([[0.0, 0, 0], [5.0, 0, 0], [0.0, 0, 0]]); A = np.zeros(3)
    pp, pm = _one_chain(3, R, [A], [2], dt=0.08).hop_probabilities(0, 0)     # h = 0.8, tanh -> -1
    assert pp == 0.5 and pm == 0.5
    pp, pm = _one_chain(3, R, [A], [2], dt=0.01).hop_probabilities(0, 0)
    assert math.isclose(pp, 0.2, rel_tol=1e-9)


def test_hop_decision_uses_moved_beads_one_uniform_and_strict_intervals():
    """Readings R4, R6: the hop sees R', A' of substep 1; one uniform per slip-spring,
    [0,p+) -> +1, [p+,p+ + p-) -> -1.  Checked by replaying the decision from the
    stream word and the post-step positions for many chains."""
    L = oracle.lib()
    moved = {+1: 0, -1: 0, 0: 0}
    for chain in range(1200):
        e = oracle.Ensemble(6, 1, seed=11, chain_offset=chain)
        if e.Z[0] == 0:
            continue
        S0 = e.S[0].copy(); Z0 = int(e.Z[0]); A0 = e.A[0].copy()
        # n_0 -> huge would switch springs off; instead keep the ends out of play by only checking interior hops
        z = C.c_int32(Z0); mm = C.c_double(1e9)
        L.oracle_step_chain(C.byref(e.p), chain, 5, 0.3, oracle._dp(e.R[0]), oracle._dp(e.A[0]),
                            oracle._ip(e.S[0]), C.byref(z), C.byref(mm))
        # anchors advected by simple shear, eq (45) with kappa_xy (eq 60)
        for j in range(Z0):
            Aadv = A0[j] + np.array([0.01 * 0.3 * A0[j, 1], 0, 0])
            s = int(S0[j])
            ref = _one_chain(6, e.R[0], [Aadv], [s])
            pp, pm = ref.hop_probabilities(0, 0)
            u = oracle.u23(oracle.stream(11, oracle.DOM_SLOT, 5, chain, j >> 1)[2 * (j & 1)])
            want = s + 1 if u < pp else (s - 1 if u < pp + pm else s)
            moved[want - s] += 1
            # survivors keep their order; a slot that left through an end is destroyed with prob 0.1 only,
            # so find slot j among the survivors by its (unique) advected anchor
            hit = [jj for jj in range(int(z.value)) if np.allclose(e.A[0, jj], Aadv, atol=0, rtol=0)]
            if hit:
                assert int(e.S[0, hit[0]]) == want
            else:
                assert want in (1, 6)               # only end slip-springs can vanish
    assert moved[+1] > 30 and moved[-1] > 30 and moved[0] > 300, moved


# ----------------------------------------------------------------------------- stress
def test_stress_definitions_eq16_eq76():
    rng = np.random.default_rng(5)
    N = 7
    R = rng.normal(size=(N, 3)); S = [1, 4, 4, 7]; A = rng.normal(size=(4, 3))
    e = _one_chain(N, R, A, S, n_s=0.7)
    sig, sv = e.chain_stress(0)
    b = np.diff(R, axis=0)
    full = 3 * np.einsum("ia,ib->ab", b, b) - N * np.eye(3)               # eq (16), P:L122 (kT = b = 1)
    d = R[np.array(S) - 1] - A
    fullv = 3 / 0.7 * np.einsum("ia,ib->ab", d, d) - len(S) * np.eye(3)   # eq (76)
    order = [(0, 0), (1, 1), (2, 2), (0, 1), (1, 2), (2, 0)]
    assert np.allclose(sig, [full[a, b_] for a, b_ in order], rtol=1e-13)
    assert np.allclose(sv, [fullv[a, b_] for a, b_ in order], rtol=1e-13)


def test_stress_translation_and_rotation_properties():
    rng = np.random.default_rng(6)
    R = rng.normal(size=(6, 3)); S = [2, 5]; A = rng.normal(size=(2, 3))
    s0, v0 = _one_chain(6, R, A, S).chain_stress(0)
    s1, v1 = _one_chain(6, R + 7.5, A + 7.5, S).chain_stress(0)
    assert np.allclose(s0, s1, atol=1e-11) and np.allclose(v0, v1, atol=1e-11)
    # swap x and y: xx<->yy, yz<->zx, xy unchanged
    P = np.array([[0, 1, 0], [1, 0, 0], [0, 0, 1.0]])
    s2, v2 = _one_chain(6, R @ P, A @ P, S).chain_stress(0)
    perm = [1, 0, 2, 3, 5, 4]
    assert np.allclose(s2, s0[perm]) and np.allclose(v2, v0[perm])


def test_equal_time_stress_statistics_on_sampled_ensemble():
    """eq (17): <sigma> = -kT 1; P7: <sigma_xy^2> = N-1 and <sigma_xy sigma^v_xy> = 0,
    <sigma^v_aa> = 0 on the equilibrium sample (eqs 6, 13, 15)."""
    N, M = 8, 20000
    e = oracle.Ensemble(N, M, seed=21)
    sig = np.zeros((M, 6)); sv = np.zeros((M, 6))
    for k in range(M):
        sig[k], sv[k] = e.chain_stress(k)
    se = sig.std(0) / math.sqrt(M)
    assert np.all(np.abs(sig[:, :3].mean(0) + 1.0) < 4 * se[:3])
    assert np.all(np.abs(sig[:, 3:].mean(0)) < 4 * se[3:])
    assert np.all(np.abs(sv.mean(0)) < 4 * sv.std(0) / math.sqrt(M))
    x = sig[:, 3] ** 2
    assert abs(x.mean() - (N - 1)) < 4 * x.std() / math.sqrt(M)
    y = sig[:, 3] * sv[:, 3]
    assert abs(y.mean()) < 4 * y.std() / math.sqrt(M)


# ----------------------------------------------------------------------------- init, P4 (static part)
def test_initial_state_distributions():
    """bonds N(0,1/3) per axis (eq 6), Z ~ Poisson(N/N0) (eq 12), S uniform
    (eq 14), R_S - A ~ N(0, N_s/3) per axis (eq 15), R_1 = 0 (reading R15)."""
    from scipy import stats
    N, M = 16, 6000
    e = oracle.Ensemble(N, M, seed=5, n_s=0.5, n_0=4.0)
    assert np.all(e.R[:, 0] == 0)
    b = np.diff(e.R, axis=1).reshape(-1)
    assert abs(b.mean()) < 4 * math.sqrt(1 / 3 / b.size)
    assert abs(b.var() - 1 / 3) < 4 * (1 / 3) * math.sqrt(2 / b.size)
    assert stats.kstest(b * math.sqrt(3), "norm").pvalue > 1e-3
    # Poisson(4): chi-square on 0..10 + tail
    lam = N / 4.0
    obs = np.bincount(np.minimum(e.Z, 11), minlength=12).astype(float)
    pmf = stats.poisson.pmf(np.arange(11), lam); exp = np.append(pmf, 1 - pmf.sum()) * M
    assert stats.chisquare(obs, exp).pvalue > 1e-3
    assert abs(e.Z.mean() - lam) < 4 * math.sqrt(lam / M)                 # eq (10): <Z> = N/N0
    occ = e.S[e.S > 0]
    assert occ.size == e.Z.sum()
    assert np.all((e.S > 0) == (np.arange(e.zmax)[None, :] < e.Z[:, None]))   # first Z slots occupied
    assert stats.chisquare(np.bincount(occ, minlength=N + 1)[1:]).pvalue > 1e-3
    d = np.concatenate([e.R[k, e.S[k, :e.Z[k]] - 1] - e.A[k, :e.Z[k]] for k in range(M)]).reshape(-1)
    assert abs(d.mean()) < 4 * math.sqrt(0.5 / 3 / d.size)
    assert abs(d.var() - 0.5 / 3) < 4 * (0.5 / 3) * math.sqrt(2 / d.size)


def test_initial_z_is_clamped_at_capacity():
    """Reading R7 (P:L366 'Z <= N'): the Poisson draw is clamped at z_max."""
    e = oracle.Ensemble(4, 3000, n_0=1.0, seed=9)        # Poisson(4) with capacity 4
    assert e.Z.max() == 4 and (e.Z == 4).mean() > 0.5
    e = oracle.Ensemble(8, 200, n_0=float("inf"), seed=9)
    assert e.Z.max() == 0                                  # springs off (Rouse limit)


# ----------------------------------------------------------------------------- P5 deterministic part
def test_rouse_limit_difference_of_twins_follows_linear_map():
    """Z = 0: two chains with the same (seed, chain, step) noise but different
    start differ by exactly (I + dt*L)^n dR(0), L = 3 x free-end Laplacian (eq 1, eq 44),
    plus the shear map.  Pins force signs, end beads, Jacobi evaluation (R2, R3)."""
    N, n, dt, gd = 9, 25, 0.01, 0.7
    rng = np.random.default_rng(8)
    Ra = rng.normal(size=(N, 3)); Rb = rng.normal(size=(N, 3))
    ea = _one_chain(N, Ra, n_0=0.0, seed=3); eb = _one_chain(N, Rb, n_0=0.0, seed=3)
    ea.run(n, shear_rate=gd); eb.run(n, shear_rate=gd)
    Lap = np.zeros((N, N))
    for i in range(N - 1):
        Lap[i, i] -= 1; Lap[i, i + 1] += 1; Lap[i + 1, i + 1] -= 1; Lap[i + 1, i] += 1
    Mx = np.eye(N) + dt * 3 * Lap
    K = np.zeros((3, 3)); K[0, 1] = gd                      # kappa_xy, eq (60)
    D = Ra - Rb
    for _ in range(n):
        D = Mx @ D + dt * D @ K.T
    assert np.allclose(ea.R[0] - eb.R[0], D, rtol=0, atol=1e-12)


def test_single_step_matches_hand_computed_update_with_springs():
    """eq (44)/(45) written out for a 3-bead chain with two slip-springs on bead 2:
    R_i' = R_i + dt F_i + dt kappa R_i + sqrt(2dt) w_i, with w from the NOISE stream."""
    N, dt, gd, ns = 3, 0.01, 0.5, 0.5
    R = np.array([[0.0, 0, 0], [1.0, 0.5, -0.2], [1.5, 1.5, 0.3]])
    A = np.array([[0.8, 0.4, 0.0], [1.3, 0.9, -0.5]]); S = [2, 2]
    e = _one_chain(N, R, A, S, seed=77)
    z = C.c_int32(2); mm = C.c_double(1e9)
    oracle.lib().oracle_step_chain(C.byref(e.p), 0, 12, gd, oracle._dp(e.R[0]), oracle._dp(e.A[0]),
                                   oracle._ip(e.S[0]), C.byref(z), C.byref(mm))
    F = np.zeros((3, 3))
    F[0] = 3 * (R[1] - R[0]); F[2] = -3 * (R[2] - R[1])
    F[1] = 3 * (R[2] - R[1]) - 3 * (R[1] - R[0]) - 3 / ns * (R[1] - A[0]) - 3 / ns * (R[1] - A[1])
    w = np.array([oracle.stream_normal(77, oracle.DOM_NOISE, 12, 0, m) for m in range(9)]).reshape(3, 3)
    want = R + dt * F + math.sqrt(2 * dt) * w
    want[:, 0] += dt * gd * R[:, 1]
    assert np.allclose(e.R[0], want, rtol=0, atol=1e-14)


# ----------------------------------------------------------------------------- P8 bookkeeping
def test_split_run_and_chain_subset_invariance():
    a = oracle.Ensemble(8, 64, seed=1); b = oracle.Ensemble(8, 64, seed=1); c = oracle.Ensemble(8, 16, seed=1)
    sa = a.run(60, stress_every=1)
    sb = np.concatenate([b.run(25, stress_every=1), b.run(35, stress_every=1)])
    c.run(60)
    assert np.array_equal(a.R, b.R) and np.array_equal(a.S, b.S) and np.array_equal(a.A, b.A)
    assert np.array_equal(sa, sb)
    assert np.array_equal(a.R[:16], c.R) and np.array_equal(a.S[:16], c.S)
    # chain_offset addresses the same global chains
    d = oracle.Ensemble(8, 16, seed=1, chain_offset=48); d.run(60)
    assert np.array_equal(a.R[48:], d.R) and np.array_equal(a.Z[48:], d.Z)
    # threads do not change anything but the summation order of the ensemble mean
    t = oracle.Ensemble(8, 64, seed=1); st = t.run(60, stress_every=1, n_threads=4)
    assert np.array_equal(a.R, t.R) and np.allclose(sa, st, rtol=0, atol=1e-12)


def test_translation_invariance_of_the_dynamics():
    a = oracle.Ensemble(8, 8, seed=2); b = oracle.Ensemble(8, 8, seed=2)
    b.R += 3.25; b.A[np.arange(8)[None, :] < b.Z[:, None]] += 3.25      # exactly representable shift
    a.run(40); b.run(40)
    assert np.array_equal(a.S, b.S)
    assert np.allclose(np.diff(a.R, axis=1), np.diff(b.R, axis=1), atol=1e-11)


def test_construction_attempt_uniform_is_assembled_as_reading_r22_states():
    """DESIGN.md reading R22: attempt k has the 23-bit code (h << 7) | e with h = half k&1 of
    word (k&7)>>1 of ATTEMPT call k>>3 and e = top 7 bits of word 2 of ANCHOR call k; success at
    bead 1 if code < T(p_c), at bead N if code < T(2 p_c) (eqs 50, 51), the anchor from normals
    0..2 of the same ANCHOR call (eq 52).  An empty chain is stepped once at many step numbers
    and the slip-springs that appear are compared with that statement written against the raw
    stream (the big-integer Philox pins the stream itself)."""
    N, seed = 16, 11
    h = 0.01 / 0.1
    pc = h / (4.0 * N)                                   # K = N - Z = N attempts
    T1, T2 = oracle.threshold23(pc), oracle.threshold23(2.0 * pc)
    made = 0
    for step in range(1500):
        e = oracle.Ensemble(N, 1, seed=seed, chain_offset=7)
        e.S[:] = 0; e.A[:] = 0.0; e.Z[:] = 0
        e.step = step
        e.run(1)
        want = []
        for k in range(N):
            w = oracle.stream(seed, oracle.DOM_ATTEMPT, step, 7, k >> 3)
            wa = oracle.stream(seed, oracle.DOM_ANCHOR, step, 7, k)
            code = (((w[(k & 7) >> 1] >> (16 * (k & 1))) & 0xFFFF) << 7) | (wa[2] >> 25)
            if code < T2:
                z0, z1 = oracle.box_muller(wa[0]); z2, _ = oracle.box_muller(wa[1])
                want.append((1 if code < T1 else N, (z0, z1, z2)))
        assert e.Z[0] == len(want)
        for j, (s, z) in enumerate(want):
            assert e.S[0, j] == s
            assert np.allclose(e.A[0, j], e.R[0, s - 1] + np.sqrt(0.5 / 3.0) * np.array(z), rtol=0, atol=1e-12)
        made += len(want)
    assert 40 < made < 120                               # 2 h / N0 = 0.05 per step expected
