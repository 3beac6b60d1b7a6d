"""GPU parity: the CUDA path (through the C ABI of include/ssm.h) against the fp64 oracle on
the same seeded inputs.  Acceptance (BASELINE.json north_star):
slip-spring indices, counts and accept/reject decisions bit-exact on every chain up to its
first fragile hop decision; bead positions, anchors and stresses within 1e-5 relative."""
import numpy as np
import pytest

import oracle
from parity_util import GUARD, TOL, close, compare_state, from_external, to_external, upload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ssm():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1106_2899_b200 as m
    m.lib()
    return m


def _pair(ssm, N, M, steps, seed=1, n_0=4.0, dt=0.01, stress_every=1, **kw):
    e = oracle.Ensemble(N, M, n_0=n_0, dt=dt, seed=seed)
    g = ssm.Ensemble(N, M, n_0=n_0, dt=dt, seed=seed, stress_every=stress_every,
                     stress_capacity=steps // max(stress_every, 1) + 1, **kw)
    upload(e, g)
    return e, g


def _min_unflagged(M, N, steps):
    """Chains the oracle flags as fragile are excluded from the comparison.  A chain makes
    about (N/4) x 2 hop comparisons per step, each within GUARD of its threshold with
    probability ~ 2 GUARD (u is uniform), so the unflagged fraction after n steps is about
    exp(-N n GUARD); fewer than that minus 4 sigma means the flags hide a bug."""
    f = np.exp(-N * steps * GUARD)
    return M * f - 4.0 * np.sqrt(M * f * (1.0 - f)) - 1.0


def test_set_get_state_roundtrip_is_bit_exact(ssm):
    e = oracle.Ensemble(32, 37, seed=5)            # 37 chains: ragged last warp tile (4 chains per warp)
    e.round_to_fp32()
    R, A, S = to_external(e)
    g = ssm.Ensemble(32, 37, seed=5)
    g.set_state(R, A, S, 123)
    R2, A2, S2, step = g.get_state()
    assert step == 123
    assert np.array_equal(R, R2) and np.array_equal(A, A2) and np.array_equal(S, S2)
    # the staging chunk of host-pointer transfers does not matter: many small chunks, or one for everything
    for chunk in (5, 37, 1000):
        h = ssm.Ensemble(32, 37, seed=5, stage_chains=chunk)
        h.set_state(R, A, S, 7)
        R3, A3, S3, step = h.get_state()
        assert step == 7 and np.array_equal(R, R3) and np.array_equal(A, A3) and np.array_equal(S, S3)


def test_state_import_export_every_shape_and_chunk(ssm):
    """a10: the import / export kernel moves 32 chains (G whole tiles) per CTA through an image of the tiles; chunks
    that start and end inside a tile, ragged bead numbers (N < 8G) and every G must give the same bytes back, and the
    import must count Z (read back as the mean of Z over all chains, exact in int64)."""
    for N, M in ((8, 203), (16, 77), (20, 131), (32, 300), (80, 45), (128, 70)):
        e = oracle.Ensemble(N, M, seed=11)
        e.round_to_fp32()
        R, A, S = to_external(e)
        for chunk in (0, 7, 33, 64, M):
            g = ssm.Ensemble(N, M, seed=99, stage_chains=chunk)       # another seed: every byte must come from the import
            g.set_state(R, A, S, 5)
            R2, A2, S2, step = g.get_state()
            assert step == 5 and np.array_equal(R, R2) and np.array_equal(A, A2) and np.array_equal(S, S2), (N, M, chunk)
            assert abs(g.group_stress()[0, 12] * M - float((S != 0).sum())) < 1e-6, (N, M, chunk)
        # device pointers: one launch for the whole ensemble
        import torch
        g = ssm.Ensemble(N, M, seed=98)
        dR, dA, dS = [torch.from_numpy(x).cuda() for x in (R, A, S)]
        g.set_state(dR, dA, dS, 6)
        R2, A2, S2, step = g.get_state()
        assert np.array_equal(R, R2) and np.array_equal(A, A2) and np.array_equal(S, S2), (N, M, "device")


def test_device_init_matches_oracle_init(ssm):
    """a0: Z and S bit-exact (integer-domain sampling), R and A to fp32 rounding."""
    for N, M in ((8, 300), (32, 130), (128, 20)):
        e = oracle.Ensemble(N, M, seed=9)
        g = ssm.Ensemble(N, M, seed=9)
        Rg, Ag, Sg, Zg = from_external(*g.get_state()[:3])
        assert np.array_equal(Sg, e.S) and np.array_equal(Zg, e.Z)
        # R_i is a running fp32 sum of i bonds, each a special-function-unit normal (absolute error
        # <= 2^-21.4 in log2, sin, cos): the error grows like sqrt(i)
        tol = 3e-6 if N <= 32 else 8e-6
        ok, w = close(Rg, e.R, tol)
        assert ok, "N=%d: R off by %.3g" % (N, w)
        ok, w = close(Ag, e.A, tol)
        assert ok, "N=%d: A off by %.3g" % (N, w)


def test_rouse_limit_positions_and_ensemble_stress_1000_steps(ssm):
    """Slip-springs off: no discrete decisions, so all chains and the ensemble
    stress of every step must match.  M = 1030 leaves a ragged tile.  (The ensemble stress is a
    mean over M chains of sums of 3 b_a b_b over N-1 bonds; the bonds carry the fp32 rounding of
    the absolute coordinates, ~2e-6 after 1000 steps, so the mean is good to about
    6 |b| 2e-6 sqrt(N-1)/sqrt(M): 1e-5 needs M of several hundred at N = 32.)"""
    N, M, steps = 32, 1030, 1000
    e, g = _pair(ssm, N, M, steps, seed=3, n_0=0.0)
    want = e.run(steps, stress_every=1)
    g.step(steps)
    n, worst = compare_state(e, g)
    assert n == M
    got = g.stress()
    ok, w = close(got, want)
    assert ok, "ensemble stress off by %.3g" % w
    assert np.all(got[:, 6:] == 0.0)


def test_c1_tiny_equilibrium_ensemble(ssm):
    """BASELINE.json config 1: 256 chains, N = 8, 2000 steps, dumps at 1, 10, 100, 1000, 2000."""
    N, M = 8, 256
    e, g = _pair(ssm, N, M, 2000, seed=1)
    done, wants = 0, []
    for upto in (1, 10, 100, 1000, 2000):
        wants.append(e.run(upto - done, stress_every=1, guard=GUARD))
        g.step(upto - done)
        done = upto
        n, worst = compare_state(e, g)
        # expected cut-short chains ~ hop decisions x 2 x 2 GUARD ~ 20 per 1000 steps; more is a bug
        assert n >= M - (3 + upto // 20), (upto, n)
    want = np.concatenate(wants)
    got = g.stress()
    first = e.first_fragile[e.first_fragile >= 0]
    clean = int(first.min()) if first.size else 2000        # steps before any chain could have forked
    assert clean >= 5
    ok, w = close(got[:clean], want[:clean])
    assert ok, "ensemble stress off by %.3g over the first %d steps" % (w, clean)
    # after forks the ensemble means differ by O(forked chains / M) only
    assert np.abs(got - want).max() < 0.5


@pytest.mark.parametrize("N,M,steps", [(16, 200, 300), (32, 100, 1000), (64, 33, 200), (128, 19, 200)])
def test_slipspring_chains_all_sizes(ssm, N, M, steps):
    e, g = _pair(ssm, N, M, steps, seed=7)
    e.run(steps, guard=GUARD)
    g.step(steps)
    n, worst = compare_state(e, g)
    assert n >= _min_unflagged(M, N, steps)
    # per-chain stresses of the final state on the chains that cannot have forked
    cs = g.chain_stress()
    ok = (e.first_fragile < 0)
    want = np.array([np.concatenate(e.chain_stress(k)) for k in np.nonzero(ok)[0]])
    # one chain, no averaging: 6 |b| delta_b sqrt(N-1) with delta_b ~ 3e-6
    good, w = close(cs.T[ok], want, 2e-5 * np.sqrt(N / 8.0))
    assert good, w


def test_shear_flow(ssm):
    """eq 44/45 with kappa_xy = gamma_dot (eq 60): beads and anchors are advected."""
    N, M, steps = 32, 64, 400
    e, g = _pair(ssm, N, M, steps, seed=11)
    want = e.run(steps, shear_rate=0.1, stress_every=1, guard=GUARD)
    g.step(steps, shear_rate=0.1)
    n, worst = compare_state(e, g)
    assert n >= _min_unflagged(M, N, steps)
    first = e.first_fragile[e.first_fragile >= 0]
    clean = int(first.min()) if first.size else steps
    ok, w = close(g.stress()[:clean], want[:clean])
    assert ok, w


def test_split_runs_fusion_depth_and_ensemble_size_do_not_change_results(ssm):
    """P8: step(a); step(b) == step(a+b); results do not depend on the fusion depth nor on M
    (Philox is keyed by the global chain index and step)."""
    N = 32
    ref = ssm.Ensemble(N, 256, seed=21, stress_every=1, stress_capacity=100)
    ref.step(90)
    R0, A0, S0, _ = ref.get_state()
    a = ssm.Ensemble(N, 256, seed=21, stress_every=1, stress_capacity=100)
    for n in (1, 7, 32, 33, 17):
        a.step(n)
    b = ssm.Ensemble(N, 256, seed=21, stress_every=1, stress_capacity=100)
    b.set_fusion(5)
    b.step(90)
    for x in (a, b):
        R, A, S, step = x.get_state()
        assert step == 90
        assert np.array_equal(R, R0) and np.array_equal(A, A0) and np.array_equal(S, S0)
        assert np.array_equal(x.stress_sums(), ref.stress_sums())
    small = ssm.Ensemble(N, 64, seed=21)
    small.step(90)
    R, A, S, _ = small.get_state()
    assert np.array_equal(R, R0[:, :, :64]) and np.array_equal(S, S0[:, :64]) and np.array_equal(A, A0[:, :, :64])
    # a shard with chain_offset reproduces its part of the full run (multi-GPU partition)
    shard = ssm.Ensemble(N, 64, seed=21, chain_offset=128)
    shard.step(90)
    R, A, S, _ = shard.get_state()
    assert np.array_equal(R, R0[:, :, 128:192]) and np.array_equal(S, S0[:, 128:192])


@pytest.mark.parametrize("M,offset,comps", [(512, 0, 1), (500, 7, 1), (512, 0, 3), (500, 7, 3)])
def test_correlator_matches_oracle_on_identical_trajectories(ssm, M, offset, comps):
    """Rouse limit (no forks): GPU multi-tau sums against the oracle's correlator fed by
    the oracle's own stresses of the same trajectories.  (500, 7): a ragged last warp and a
    shard that does not start on a multiple of 32, so that a warp's chains fall into two
    groups (the per-lane path of the correlator kernel).  comps = 3: the isotropic average, xy, yz and
    zx histories feeding the same sums."""
    N, steps = 8, 2000
    e = oracle.Ensemble(N, M, n_0=0.0, seed=13, chain_offset=offset)
    g = ssm.Ensemble(N, M, n_0=0.0, seed=13, chain_offset=offset, sample_every=10, corr_levels=6, corr_bins=16,
                     corr_groups=32, corr_components=comps)
    upload(e, g)
    corr = oracle.Correlator(M, levels=6, bins=16, groups=32, components=comps)
    e.run(steps, sample_every=10, corr=corr)
    g.step(steps)
    t0, G0, se0 = corr.result(N, 0.1)
    t1, G1, se1 = g.gt()
    assert np.allclose(t0, t1)
    assert np.allclose(G1, G0, rtol=0, atol=2e-4 * np.abs(G0).max())
    assert np.allclose(se1, se0, rtol=0.02, atol=1e-6)


def test_device_view_of_the_stress_sums_is_what_the_exchange_reduces(ssm):
    """the only multi-GPU exchange is an in-place int64 all-reduce of the
    fixed-point sums inside the workspace; the device view must alias exactly what ssm_stress_sums
    and ssm_stress report (one rank: the reduction is the identity)."""
    import torch
    from paper_1106_2899_b200 import shard
    g = ssm.Ensemble(16, 300, seed=31, stress_every=1, stress_capacity=40)
    g.step(40)
    dev = g.stress_sums_device(5, 20)
    assert dev.is_cuda and dev.dtype == torch.int64 and tuple(dev.shape) == (20, 12)
    shard.allreduce_sums(dev)
    torch.cuda.synchronize()
    host = g.stress_sums()[5:25]
    assert np.array_equal(dev.cpu().numpy(), host)
    assert np.allclose(shard.stress_means(host, 300), g.stress(5, 20), rtol=0, atol=1e-12)


def test_issue_rate_probe(ssm):
    """ssm_issue_rates: plain ALU and FP32 instructions issue about once per
    cycle per scheduler, IMAD at half rate, and the 32 x 32 -> 64-bit multiply of Philox slower still."""
    g = ssm.Ensemble(8, 64, seed=1)
    r = g.issue_rates()
    assert 0.9 < r["ffma"] < 1.6 and 0.9 < r["alu"] < 1.6
    assert 1.7 < r["imad"] < 2.6
    assert 3.0 < r["imad_wide"] < 6.0
    R, A, S, step = g.get_state()          # the probe used the staging area only
    g2 = ssm.Ensemble(8, 64, seed=1)
    assert np.array_equal(R, g2.get_state()[0]) and np.array_equal(S, g2.get_state()[2])
