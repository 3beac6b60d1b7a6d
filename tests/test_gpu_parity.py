"""GPU parity: the CUDA path (through the C ABI of include/ssm.h) against the fp64 oracle on
the same seeded inputs.  Acceptance (BASELINE.json north_star):
slip-spring indices, counts and accept/reject decisions bit-exact on every chain up to its
first fragile hop decision; bead positions, anchors and stresses within 1e-5 relative."""
import numpy as np
import pytest

import oracle
from parity_util import GUARD, TOL, close, compare_chain_stress_sums, compare_state, from_external, to_external, upload

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
    for N, M in ((3, 50), (8, 203), (16, 77), (20, 131), (32, 300), (64, 40), (80, 45), (100, 33), (128, 70)):
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
        # the stress at this step, summed over the chains that cannot have forked, within 1e-5
        ns, _ = compare_chain_stress_sums(e, g)
        assert ns == n
    want = np.concatenate(wants)
    got = g.stress()
    first = e.first_fragile[e.first_fragile >= 0]
    clean = int(first.min()) if first.size else 2000        # steps before any chain could have forked
    assert clean >= 5
    ok, w = close(got[:clean], want[:clean])
    assert ok, "ensemble stress off by %.3g over the first %d steps" % (w, clean)
    # after forks the ensemble means differ by O(forked chains / M) only
    assert np.abs(got - want).max() < 0.5


@pytest.mark.parametrize("N,M", [(16, 1003), (32, 1001), (64, 1001), (128, 1031)])
def test_slipspring_chains_all_sizes(ssm, N, M):
    """Every kernel size (G = 2, 4, 8, 16; ragged last tiles) over north_star's full window of 1000 steps, with
    dumps at 1, 10, 100, 1000: S, Z bit-exact and R, A within 1e-5 on every chain up to its first fragile step,
    and the stress summed over those chains within 1e-5 at every dump.  (A thousand chains, as in the Rouse-limit
    test: the stress is an ensemble quantity, eq 54 -- one chain's 3 sum b_a b_b carries the fp32 rounding of
    its N - 1 bonds, ~1e-4 at N = 128, and it is the mean over the ensemble that north_star
    bounds; at N = 128 a quarter of the chains are still unforked at step 1000.)"""
    steps = 1000
    e, g = _pair(ssm, N, M, steps, seed=7)
    done = 0
    for upto in (1, 10, 100, 1000):
        e.run(upto - done, guard=GUARD, n_threads=8)
        g.step(upto - done)
        done = upto
        n, worst = compare_state(e, g)
        assert n >= _min_unflagged(M, N, upto), (upto, n)
        ns, _ = compare_chain_stress_sums(e, g)
        assert ns == n
    # per-chain stresses of the final state on the chains that cannot have forked
    cs = g.chain_stress()
    ok = (e.first_fragile < 0)
    want = np.array([np.concatenate(e.chain_stress(k)) for k in np.nonzero(ok)[0]])
    # one chain, no averaging: 6 |b| delta_b sqrt(N-1) with delta_b ~ 3e-6
    good, w = close(cs.T[ok], want, 2e-5 * np.sqrt(N / 8.0))
    print("per-chain stress N=%d worst/TOL=%.2f" % (N, w / TOL))
    assert good, w


def test_noise_amplitude_is_calibrated(ssm):
    """the thermal noise of eqs 44, 46 is drawn through the special-function unit from 2^16 x 2^16
    codes, so its variance on this GPU is a finite sum; ssm_init forms it and picks the fp32 Box-Muller constant whose
    variance is nearest the exact sigma^2 mean(-2 ln u_a) / 2.  Left alone, the constant gives a variance low by
    about 2.8e-7 -- the systematic error that made the diagonal stress 3 sum b_a^2 - N miss 1e-5 for N >= 64."""
    for dt in (0.01, 0.005):
        g = ssm.Ensemble(16, 64, dt=dt)
        c = g.noise_calibration()
        print("dt=%g: variance error plain %.3g, calibrated %.3g, %d ulps; cos2 %.3g sin2 %.3g"
              % (dt, c["variance_error_plain"], c["variance_error_used"], c["ulps_moved"], c["cos2_bias"], c["sin2_bias"]))
        assert abs(c["variance_error_used"]) <= 3.5e-8                 # half an ulp of the constant (mantissa 1.77)
        assert abs(c["variance_error_used"]) <= abs(c["variance_error_plain"])
        assert abs(c["bm_used"] / (-2.0 * np.log(2.0) * 2.0 * dt) - 1.0) < 2e-6 and abs(c["ulps_moved"]) < 16
        assert abs(c["cos2_bias"] - c["sin2_bias"]) < 2e-8             # one constant serves both members of a pair
        g.close()


def test_shear_flow(ssm):
    """eq 44/45 with kappa_xy = gamma_dot (eq 60): beads and anchors are advected."""
    N, M, steps = 32, 64, 400
    e, g = _pair(ssm, N, M, steps, seed=11)
    want = e.run(steps, shear_rate=0.1, stress_every=1, guard=GUARD)
    g.step(steps, shear_rate=0.1)
    n, worst = compare_state(e, g)
    assert n >= _min_unflagged(M, N, steps)
    compare_chain_stress_sums(e, g)
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


def test_results_do_not_depend_on_which_warp_runs_a_tile(ssm):
    """a8: warps draw their tiles first come, first served and add fixed-point integers, so neither the number of CTAs
    nor the order in which warps arrive may show in anything: one CTA (8 warps walk 500 tiles), three, and the default
    grid give the same state, stress sums and correlator sums bit for bit; also under shear (compensated anchors)."""
    N, M = 32, 4000
    kw = dict(seed=33, stress_every=1, stress_capacity=200, sample_every=4, corr_levels=3)
    outs = []
    for blocks in (0, 1, 3):
        g = ssm.Ensemble(N, M, **kw)
        g.set_grid(blocks)
        g.step(70)
        g.step(30, shear_rate=0.2)
        R, A, S, _ = g.get_state()
        outs.append((R, A, S, g.stress_sums(), g.gt_sums()[0]))
    for o in outs[1:]:
        for x, y in zip(outs[0], o):
            assert np.array_equal(x, y)


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
    assert np.allclose(se1, se0, rtol=0.02, atol=1e-6)
    # the raw sums, group by group and lag by lag, each against a bound of ITS OWN size: a product f g carries the
    # fp32 error of the two stresses (relative 1e-5 of sqrt(<f^2><g^2>) at worst, TOL) and the 2^-16 fixed point
    # of its sum; the errors of a bin's n products are independent in sign, so the bin's sum is good to
    # TOL |sum| + 4 sqrt(n) (TOL <f g>_0 + 2^-17), <f g>_0 = the lag-0 mean product
    so, sgo, co = corr.sums()
    sg, cg = g.gt_sums()
    assert np.array_equal(cg, co)                          # the host-side schedule counts the same products
    used = co > 0
    fg0 = so[:, 0, 0].sum() / co[:, 0, 0].sum()
    bound = TOL * np.abs(so) + 4.0 * np.sqrt(co) * (TOL * fg0 + 2.0 ** -17)
    assert np.all(np.abs(sg - so)[used] <= bound[used]), float((np.abs(sg - so)[used] / bound[used]).max())
    # and G(t) itself lag by lag: the same bound summed over the groups
    n_lag = co.sum(0)[co.sum(0) > 0]
    assert np.all(np.abs(G1 - G0) <= TOL * np.abs(G0) + 4.0 * (TOL * fg0 + 2.0 ** -17) / (np.sqrt(n_lag) * N))


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
    """ssm_issue_rates8: FP32 issues once per cycle per scheduler, the ALU pipe (LOP3) and
    IMAD every second cycle, the special-function unit every eighth, and the 32 x 32 -> 64-bit multiply of Philox
    holds the issue port for about three cycles beyond its own -- FFMAs beside it do not hide."""
    g = ssm.Ensemble(8, 64, seed=1)
    r = g.issue_rates()
    assert 0.9 < r["ffma"] < 1.6
    assert 1.7 < r["alu"] < 2.6 and 1.7 < r["imad"] < 2.6
    assert 7.0 < r["mufu"] < 9.5 and 7.0 < r["i2f_f2i"] < 9.5
    assert 2.5 < r["imad_wide"] < 5.0
    assert r["wide_lop3_4ffma"] - r["wide_lop3"] > 3.0            # four FFMA cost four more cycles: no overlap
    assert 7.0 < r["philox_round"] < 10.5
    R, A, S, step = g.get_state()          # the probe used the staging area only
    g2 = ssm.Ensemble(8, 64, seed=1)
    assert np.array_equal(R, g2.get_state()[0]) and np.array_equal(S, g2.get_state()[2])


def test_pipelined_upload_and_step_equals_set_state_then_step(ssm):
    """ssm_step_from_host uploads the ensemble in chunks on a copy stream and steps a chunk's tiles as soon as it has
    landed: state and stress sums must be those of ssm_set_state + ssm_step bit for bit, for ragged ensembles, ragged
    bead numbers, any staging size, with and without shear, and appended to earlier samples."""
    import torch
    for N, M, stage in ((32, 1000, 128), (32, 1000, 512), (20, 333, 64), (128, 77, 64), (8, 5000, 2048)):
        e = oracle.Ensemble(N, M, seed=21)
        e.round_to_fp32()
        R, A, S = to_external(e)
        pin = [torch.from_numpy(x).pin_memory().numpy() for x in (R, A, S)]
        for rate in (0.0, 0.05):
            a = ssm.Ensemble(N, M, seed=21, stress_every=1, stress_capacity=200, stage_chains=stage)
            a.step(7, rate)                                     # earlier samples stay where they are
            a.set_state(R, A, S, 40)
            a.step(75, rate)
            b = ssm.Ensemble(N, M, seed=21, stress_every=1, stress_capacity=200, stage_chains=stage)
            b.step(7, rate)
            b.step_from_host(*pin, 40, 75, rate)
            for x, y in zip(a.get_state(), b.get_state()):
                assert np.array_equal(x, y), (N, M, stage, rate)
            assert np.array_equal(a.stress_sums(), b.stress_sums()) and a.stress_count() == 82
    g = ssm.Ensemble(16, 100, seed=1, sample_every=10)
    with pytest.raises(ssm.SsmError) as err:
        g.step_from_host(*[np.ascontiguousarray(x) for x in g.get_state()[:3]], 0, 10)
    assert err.value.code == ssm.SSM_ESTATE                     # the correlator must be off


def test_two_contexts_stepping_concurrently_give_the_same_samples(ssm):
    """Two contexts on two streams, driven by two host threads, same seed and input: their kernels share the SMs, so a
    CTA finds in shared memory whatever the other context's CTA left there.  Everything the step kernel reads must have
    been written by it first (round 2 found the chains' last-candidate words read through atomicMax uninitialised this
    way); the samples and states of the two must be identical, and equal to a context run alone."""
    import threading
    import torch
    N, M, steps = 32, 200000, 64
    ref = ssm.Ensemble(N, M, seed=9, stress_every=1, stress_capacity=steps)
    ref.step(steps)
    want = ref.stress_sums(); Rw = ref.get_state()
    del ref
    for _ in range(2):
        ctx = [ssm.Ensemble(N, M, seed=9, stress_every=1, stress_capacity=steps, stream=torch.cuda.Stream()) for _ in range(2)]
        def work(g):
            for _ in range(steps // 16):
                g.step(16)
            g.synchronize()
        th = [threading.Thread(target=work, args=(g,)) for g in ctx]
        for t in th:
            t.start()
        for t in th:
            t.join()
        for g in ctx:
            assert np.array_equal(g.stress_sums(), want)
            for x, y in zip(g.get_state(), Rw):
                assert np.array_equal(x, y)


def test_set_state_rejects_malformed_slip_spring_indices(ssm):
    """The checkpoint-restore path validates S on the device: occupied slots must be the leading ones and
    hold bead indices 1..N.  A bad chain keeps its valid leading slots only, the call fails with SSM_EINVAL, and the
    ensemble can still be stepped (no out-of-range scatter)."""
    N, M = 20, 70                                          # ragged: 20 beads in 32 places
    e = oracle.Ensemble(N, M, seed=3)
    e.round_to_fp32()
    R, A, S = to_external(e)
    g = ssm.Ensemble(N, M, seed=3)
    g.set_state(R, A, S, 0)                                # well-formed: accepted
    for what in ("gap", "range"):
        S2 = S.copy()
        k = int(np.argmax(e.Z >= 2))
        if what == "gap":
            S2[e.Z[k] + 1, k] = 3                          # an occupied slot after an empty one
        else:
            S2[1, k] = N + 1                               # a bead index beyond the chain
        with pytest.raises(ssm.SsmError) as err:
            g.set_state(R, A, S2, 0)
        assert err.value.code == ssm.SSM_EINVAL
        Rb, Ab, Sb, _ = g.get_state()
        want = S.copy()
        if what == "range":
            want[1:, k] = 0                                # the valid leading slot survives
        assert np.array_equal(Sb, want)
        g.step(40)                                         # still safe to step
        assert g.get_state()[2].max() <= N
        g.set_state(R, A, S, 0)                            # and a good state is accepted again


def test_two_contexts_on_two_devices_in_one_process(ssm):
    """The dynamic shared-memory attribute of the step kernel is per device: a second context on cuda:1 (first use
    of FLOW 0 / 1 and of the non-ragged kernels there) must launch, and every call must run on its own device."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    out = []
    for dev in ("cuda:0", "cuda:1"):
        g = ssm.Ensemble(32, 300, seed=5, stress_every=1, stress_capacity=64, sample_every=10, corr_levels=3, device=dev)
        g.step(20)
        g.step(20, shear_rate=0.1)
        out.append((g.get_state(), g.stress_sums(), g.gt_sums()[0], g.chain_stress()))
    for a, b in zip(out[0][0][:3], out[1][0][:3]):
        assert np.array_equal(a, b)
    assert np.array_equal(out[0][1], out[1][1]) and np.array_equal(out[0][2], out[1][2]) and np.array_equal(out[0][3], out[1][3])


def _nccl_rank(rank, world, port, q):
    import os
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    import paper_1106_2899_b200 as m
    from paper_1106_2899_b200 import shard
    M, N, steps = 1000, 16, 48
    k0, k1 = shard.strong_range(M, rank, world)
    st = torch.cuda.Stream()                                # the context's own stream, NOT the one NCCL syncs with
    g = m.Ensemble(N, k1 - k0, seed=41, chain_offset=k0, stress_every=1, stress_capacity=steps, device="cuda:%d" % rank, stream=st)
    g.step(steps)
    sums = g.stress_sums_device(0, steps)
    shard.allreduce_sums(sums, ctx=g)                       # orders the two streams with events (ssm_stream_wait_ctx)
    out = g.stress_sums()                                   # on the ctx's stream, after the exchange
    dist.destroy_process_group()
    q.put((rank, out))


def test_nccl_allreduce_of_two_shards_equals_the_single_gpu_sums(ssm):
    """two NCCL ranks, each a contiguous shard of the global chain index on its own GPU and its own
    stream; the in-place all-reduce of ssm_stress_sums_device gives, on both ranks, exactly the int64 sums of the
    single-GPU run of the whole ensemble."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_nccl_rank, args=(r, 2, 29541, q)) for r in range(2)]
    for p in ps:
        p.start()
    got = dict(q.get(timeout=300) for _ in ps)
    for p in ps:
        p.join(60)
    ref = ssm.Ensemble(16, 1000, seed=41, stress_every=1, stress_capacity=48)
    ref.step(48)
    want = ref.stress_sums()
    assert np.array_equal(got[0], want) and np.array_equal(got[1], want)
