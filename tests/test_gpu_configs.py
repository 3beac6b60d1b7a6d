"""BASELINE.json configs[1], [2], [4] (C2, C3, C5 of SURVEY.md section 8d) run ONCE EACH at their stated size on
the GPU -- full ensemble, full correlator depth (16 levels x 16 bins), bench.py's launch configuration -- and compared
with the oracle's scaled twin as section 8(d) writes it: independent samples of the same process (different seeds;
long runs fork at the first fragile hop decision), lag by lag / time by time within the combined
standard error.  Plus the 16-level correlator on identical trajectories (Rouse limit, no forks), where the GPU's
sums must equal the oracle's.

Run lengths: C2 and the shape of C3 are the stated ones (1e6 steps; 2e5 steps per rate); C5 runs 2e5 of its 1e6 steps
with the correlator and 2e5 under shear (its longest relaxation time, ~1e4 tau0 = 2e6 steps, is out of reach of a test
either way).  Each test prints the numbers DESIGN.md section 8.5 quotes."""
import math

import numpy as np
import pytest

import oracle
from parity_util import TOL, upload

pytestmark = pytest.mark.gpu

NT = 16


@pytest.fixture(scope="module")
def ssm():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1106_2899_b200 as m
    m.lib()
    return m


def _z_report(name, t_g, G_g, se_g, t_o, G_o, se_o):
    """z per lag on the lags both sides have; prints what DESIGN.md section 8.5 tabulates."""
    idx = {round(float(t), 6): i for i, t in enumerate(t_g)}
    common = [(idx[round(float(t), 6)], j) for j, t in enumerate(t_o) if round(float(t), 6) in idx]
    ig = np.array([c[0] for c in common]); io = np.array([c[1] for c in common])
    se = np.hypot(se_g[ig], se_o[io])
    ok = np.isfinite(se) & (se > 0)
    z = (G_g[ig] - G_o[io])[ok] / se[ok]
    print("%s: %d GPU lags (to t = %.0f), %d oracle lags, %d compared; |z| < 3 on %.1f %%, max |z| = %.2f at t = %.1f"
          % (name, len(t_g), t_g[-1], len(t_o), z.size, 100.0 * np.mean(np.abs(z) < 3.0), np.abs(z).max(),
             t_o[io][ok][np.abs(z).argmax()]))
    return z


def test_c2_equilibrium_gt_full_size_and_depth(ssm):
    """configs[1]: 65,536 chains x N = 16, dt = 0.01, 1e6 steps, sampled every 10 steps into the 16 x 16 multi-tau
    correlator (eq 43).  Oracle twin: 4096 chains x 1e5 steps, another seed."""
    N = 16
    g = ssm.Ensemble(N, 65536, seed=2, sample_every=10, corr_levels=16, corr_bins=16, corr_groups=32)
    g.step(1000000)
    t_g, G_g, se_g = g.gt()
    e = oracle.Ensemble(N, 4096, seed=1002)
    corr = oracle.Correlator(4096, levels=16, bins=16, groups=32)
    e.run(100000, sample_every=10, corr=corr, n_threads=NT)
    t_o, G_o, se_o = corr.result(N, 0.1)
    # 1e5 samples reach level 13 (12 insertions, bins 8..11), the oracle's 1e4 samples level 10
    assert len(t_g) >= 16 + 12 * 8 and t_g[-1] >= 8 * 2 ** 13 * 0.1
    z = _z_report("C2", t_g, G_g, se_g, t_o, G_o, se_o)
    assert z.size >= 16 + 9 * 8
    assert np.mean(np.abs(z) < 3.0) >= 0.95 and np.abs(z).max() < 4.5, z
    # pin P7 with the Euler map's O(dt) bias: N G(0) = <s_xy (s_xy + sv_xy)> = sum_p 1/(1 - k_p dt/2)^2 = 15.964
    # (N - 1 = 15 in the limit dt -> 0; the slip-springs leave the equal-time value alone, eq 13)
    assert abs(G_g[0] * N - 15.964) < 0.02 * 15.964, G_g[0] * N
    # G(t) has decayed to noise at the longest lags: the deep levels hold what the schedule says they hold
    s, c = g.gt_sums()
    n_samples = 100000
    for lev in range(14):
        ins = n_samples // 2 ** lev                                  # insertions at this level
        for q in range(16):
            want = max(0, ins - q) if (lev == 0 or q >= 8) else 0
            assert c[:, lev, q].sum() == want * 65536, (lev, q)


def _blocks(fn, n_blocks):
    return np.array([fn(b) for b in range(n_blocks)])


def test_c3_startup_shear_four_rates_full_size(ssm):
    """configs[2]: 262,144 chains x N = 32, one equilibrated state, shear switched on at t = 0 (eq 60; reading
    R17) at rates 1e-1, 1e-2, 1e-3, 1e-4, 2e5 steps each, <s_xy> every 10 steps (eq 61).  Rates 1e-1 and 1e-2 directly
    against the oracle (4096 chains x 2e4 steps, 16 blocks for the standard error).  Rates 1e-3 and 1e-4 are below the
    per-sample noise sqrt(N-1)/sqrt(M) = 0.011: counter-based random numbers make the run without flow from the same
    state and step counter a common-random-number twin, and the difference is compared with linear
    response, eta+(t) = int_0^t G(s) ds (eq 42 P:L272 with a step strain rate; pin P6), G from the twin's correlator."""
    import torch
    N, M, steps, every = 32, 262144, 200000, 10
    g = ssm.Ensemble(N, M, seed=3, stress_every=every, stress_capacity=steps // every, sample_every=10,
                     corr_levels=16, corr_bins=16, corr_groups=32)
    g.step(2000)                                                     # equilibrate under the Euler map
    dev = g.device
    R = torch.empty((3, N, M), dtype=torch.float32, device=dev); A = torch.empty((4, N, M), dtype=torch.float32, device=dev)
    S = torch.empty((N, M), dtype=torch.uint8, device=dev)
    _, _, _, step0 = g.get_state(R, A, S)
    curves = {}
    for rate in (0.0, 1e-1, 1e-2, 1e-3, 1e-4):
        g.set_state(R, A, S, step0)                                  # same state, same Philox step coordinate
        g.reset_accumulators()
        g.step(steps, shear_rate=rate)
        curves[rate] = g.stress()[:, 3].copy()                       # <s_xy>(t), t = 10 dt, 20 dt, ...
        if rate == 0.0:
            t_c, G_c, _ = g.gt()
    t = (np.arange(steps // every) + 1) * every * 0.01

    # ---- 1e-1, 1e-2: GPU vs oracle, independent samples
    def oracle_curve(rate, n_steps, n_blocks=16, Mb=256):
        def one(b):
            e = oracle.Ensemble(N, Mb, seed=7003, chain_offset=b * Mb)
            e.run(2000, n_threads=NT)
            return e.run(n_steps, shear_rate=rate, stress_every=every, n_threads=NT)[:, 3] / (N * rate)
        c = _blocks(one, n_blocks)
        return c.mean(0), c.std(0, ddof=1) / math.sqrt(n_blocks)

    for rate in (1e-1, 1e-2):
        n_o = 20000
        mo, so = oracle_curve(rate, n_o)
        mg = curves[rate][: n_o // every] / (N * rate)
        sg = so * math.sqrt(4096.0 / M)                              # same per-chain spread, 64 times the chains
        z = (mg - mo) / np.hypot(so, sg)
        print("C3 rate %g: eta+ at t = 1, 10, 100, 200: GPU %s oracle %s; |z| < 3 on %.1f %%, max |z| = %.2f"
              % (rate, np.round(mg[[9, 99, 999, 1999]], 3), np.round(mo[[9, 99, 999, 1999]], 3),
                 100.0 * np.mean(np.abs(z) < 3.0), np.abs(z).max()))
        # 16 blocks: z follows Student's t with 15 degrees of freedom, P(|t| > 3) = 0.9 %
        assert np.mean(np.abs(z) < 3.0) >= 0.95 and np.abs(z).max() < 6.0, (rate, np.abs(z).max())

    # ---- 1e-3, 1e-4: common-random-number differencing against the twin, and linear response
    # int_0^t G by the trapezoidal rule on the correlator's lags.  Two O(dt) effects bound how closely eta+ can follow
    # it, both properties of the explicit Euler scheme the paper uses, not of either program: the scheme's
    # stationary law is not the Boltzmann one, so the equal-time correlation N G(0) = sum_p 1/(1 - k_p dt/2)^2 sits
    # 3 % above the true response to a strain step, 3 <sum b_y^2> = sum_p 1/(1 - k_p dt/2); and the
    # lags are 10 dt apart where G falls from 1.04 to 0.45 within the first one.  Tolerance: 6 % of int G beyond
    # t = 3 tau0, 12 % before, plus the statistical error.
    cum = np.concatenate([[0.0], np.cumsum(0.5 * (G_c[1:] + G_c[:-1]) * np.diff(t_c))])        # int_0^t G, trapezoid
    eta_lr = np.interp(t, t_c, cum)
    eta0 = cum[-1]
    tau_c = 25.0                                                       # correlation time of the ensemble stress ~ tau_d
    for rate in (1e-3, 1e-4):
        eta = (curves[rate] - curves[0.0]) / (N * rate)
        # (i) the first 3 tau0: most twin chains still coincide, the difference is nearly noise-free and pins the whole
        # linear-response pipeline (leaving sigma^(v) out of eq 43 would be off by 25 %)
        early = slice(4, 30)
        r_early = eta[early].mean() / eta_lr[early].mean()
        # (ii) later the twins decorrelate (hop decisions fork) and the difference carries the noise of two independent
        # ensembles, correlated over ~ tau_d: windows of growing length, each against its own standard error
        rows = []
        for a, b in ((30, 100), (100, 300), (300, 1000), (1000, 3000), (3000, 10000), (10000, 20000)):
            w = eta[a:b]
            se = w.std() * math.sqrt(min(1.0, 2.0 * tau_c / ((b - a) * every * 0.01)))
            rows.append((t[a], t[b - 1], w.mean(), eta_lr[a:b].mean(), se))
        print("C3 rate %g (CRN): eta+ / int G over 0.5 <= t <= 3: %.3f; windows (t0, t1, eta+, int G, SE): %s; eta0 = %.3f"
              % (rate, r_early, [tuple(round(float(x), 3) for x in r) for r in rows], eta0))
        assert abs(r_early - 1.0) < 0.12, (rate, r_early)
        for t0, t1, m, lr, se in rows:
            assert abs(m - lr) < 0.06 * lr + 4.0 * se, (rate, t0, t1, m, lr, se)
    # shear thinning and overshoot at the fast rate, Newtonian plateau at the slow ones (Fig 4)
    e1 = curves[1e-1] / (N * 1e-1)
    assert e1.max() > 1.1 * e1[-2000:].mean() and e1[-2000:].mean() < 0.8 * eta0


def test_c5_long_chains_gt_and_shear(ssm):
    """configs[4]: 131,072 chains x N = 128 (16 lanes per chain: the shared-memory-resident kernel), dt = 0.005,
    equilibrium G(t) through the 16 x 16 correlator over the stated 1e6 steps (t = 5000 tau0), then shear at rate 1e-3
    for another 1e6 steps: total strain 5, t = 5000 tau0 -- the longest relaxation time of N = 128 is about 1e4 tau0
    (tau_d ~ (N - 1)^3.48), so eta+(t) is still growing towards eta0 (eqs 61, 62) and is checked against the
    linear-response int_0^t G of the same run while the strain is small, and for how far it has come at the end.
    Oracle twin: 512 chains x 1e5 steps; under shear 16 blocks of 32 chains x 2e4 steps."""
    N, M, dt = 128, 131072, 0.005
    n_eq = 1000000
    g = ssm.Ensemble(N, M, dt=dt, seed=5, stress_every=10, stress_capacity=100000, sample_every=10,
                     corr_levels=16, corr_bins=16, corr_groups=32)
    g.step(n_eq)
    t_g, G_g, se_g = g.gt()
    # 1e5 samples reach level 13 (12 insertions, bins 8..11): the deep levels hold what the schedule says they hold
    assert len(t_g) >= 16 + 12 * 8 and t_g[-1] >= 8 * 2 ** 13 * 10 * dt
    _, cnt = g.gt_sums()
    for lev in range(16):
        ins = (n_eq // 10) // 2 ** lev
        for q in range(16):
            want = max(0, ins - q) if (lev == 0 or q >= 8) else 0
            assert cnt[:, lev, q].sum() == want * M, (lev, q)
    e = oracle.Ensemble(N, 512, dt=dt, seed=1005)
    corr = oracle.Correlator(512, levels=16, bins=16, groups=16)
    e.run(100000, sample_every=10, corr=corr, n_threads=NT)
    t_o, G_o, se_o = corr.result(N, 10 * dt)
    z = _z_report("C5", t_g, G_g, se_g, t_o, G_o, se_o)
    assert z.size >= 16 + 8 * 8
    assert np.mean(np.abs(z) < 3.0) >= 0.95 and np.abs(z).max() < 4.5, z
    assert abs(G_g[0] * N - 130.943) < 0.02 * 130.943, G_g[0] * N    # pin P7 with the Euler bias at dt = 0.005
    # entangled plateau: G(t) ~ 0.1 rho0 kT for large N at intermediate times
    mid = (t_g > 20.0) & (t_g < 60.0)
    print("C5 plateau: G(20 < t < 60) = %s" % np.round(G_g[mid], 3))
    assert np.all((G_g[mid] > 0.07) & (G_g[mid] < 0.2))
    # ---- shear at 1e-3 from the equilibrated ensemble
    rate = 1e-3
    g.reset_accumulators()
    g.step(1000000, shear_rate=rate)
    eta_g = g.stress()[:, 3] / (N * rate)
    assert eta_g.size == 100000

    def one(b):
        x = oracle.Ensemble(N, 32, dt=dt, seed=2005, chain_offset=32 * b)
        x.run(4000, n_threads=NT)
        return x.run(20000, shear_rate=rate, stress_every=10, n_threads=NT)[:, 3] / (N * rate)
    c = _blocks(one, 16)
    mo, so = c.mean(0), c.std(0, ddof=1) / 4.0
    # the oracle's 512 chains are noisy per sample: compare block means over 100 samples (5 tau0)
    k = 100
    mo_b = mo.reshape(-1, k).mean(1); so_b = c.reshape(16, -1, k).mean(2).std(0, ddof=1) / 4.0
    mg_b = eta_g[: mo.size].reshape(-1, k).mean(1)
    zb = (mg_b - mo_b) / so_b
    print("C5 shear 1e-3: eta+ (block means) GPU %s oracle %s; max |z| = %.2f; last sample eta+(t = 5000) = %.2f"
          % (np.round(mg_b[[0, 4, 9, 19]], 2), np.round(mo_b[[0, 4, 9, 19]], 2), np.abs(zb).max(), eta_g[-1]))
    assert np.mean(np.abs(zb) < 3.0) >= 0.9 and np.abs(zb).max() < 5.0, zb
    # linear response while the strain is small (t <= 100: strain 0.1): eta+(t) = int_0^t G
    cum = np.concatenate([[0.0], np.cumsum(0.5 * (G_g[1:] + G_g[:-1]) * np.diff(t_g))])
    t = (np.arange(eta_g.size) + 1) * 10 * dt
    lr = np.interp(t, t_g, cum)
    sel = (t > 20.0) & (t <= 100.0)
    dev = np.abs(eta_g[sel].reshape(-1, 40).mean(1) / lr[sel].reshape(-1, 40).mean(1) - 1.0)
    print("C5 shear 1e-3: eta+ / int G - 1 over 20 < t <= 100 (means of 2 tau0): max %.3f" % dev.max())
    assert dev.max() < 0.08
    # where the viscosity growth stands after 5000 tau0 (strain 5) against the linear-response integral of this run's own
    # G(t) up to the same time and up to the correlator's longest lag.  Strain 5 at Wi = rate tau_d ~ 10 is beyond the
    # linear regime: eta+ has to lie BELOW int_0^t G (shear thinning, Fig 5) and above its value at strain 1/2.
    last = eta_g[-2000:].mean()                                        # mean over the last 100 tau0
    at = lambda tt: eta_g[(t > tt - 50.0) & (t <= tt + 50.0)].mean()
    grow = [at(500.0), at(1000.0), at(2000.0), at(3000.0), at(4000.0), last]
    print("C5 shear 1e-3: eta+ at t = 500, 1000, 2000, 3000, 4000, 4950: %s; int_0^t G at t = 500, 1000, 2000: %s, over all lags "
          "(to t = %.0f): %.1f" % (np.round(grow, 1), np.round(np.interp([500.0, 1000.0, 2000.0], t_g, cum), 1), t_g[-1], cum[-1]))
    assert 0.0 < last < 1.05 * cum[-1]                                 # the shear envelope: eta+ stays below int G (no strain hardening in shear)
    assert abs(at(500.0) / np.interp(500.0, t_g, cum) - 1.0) < 0.15    # strain 1/2: still close to linear response


def test_sixteen_level_correlator_equals_the_oracle_on_identical_trajectories(ssm):
    """The host-side schedule (ring positions, fill counts, pair parities, product counts) and the ring memory of
    ALL 16 levels: Rouse limit (no discrete decisions, the two sides follow the same trajectories), N = 8, 64
    chains, 3.3e5 steps = 33,000 samples -> level 15 receives one insertion, level 11 its first products."""
    N, M, steps = 8, 64, 330000
    e = oracle.Ensemble(N, M, n_0=0.0, seed=17)
    g = ssm.Ensemble(N, M, n_0=0.0, seed=17, sample_every=10, corr_levels=16, corr_bins=16, corr_groups=2)
    upload(e, g)
    corr = oracle.Correlator(M, levels=16, bins=16, groups=2)
    e.run(steps, sample_every=10, corr=corr, n_threads=NT)
    g.step(steps)
    so, sgo, co = corr.sums()
    sg, cg = g.gt_sums()
    assert np.array_equal(cg, co)
    deepest = max(lev for lev in range(16) if co[:, lev].sum() > 0)
    assert deepest >= 11
    used = co > 0
    fg0 = so[:, 0, 0].sum() / co[:, 0, 0].sum()
    # per-bin bound as in test_correlator_matches_oracle_on_identical_trajectories; over 3.3e5 steps the fp32
    # trajectories stay within TOL of the fp64 ones in the bonds (the stencil is contractive), which is all the
    # stress sees
    bound = TOL * np.abs(so) + 4.0 * np.sqrt(co) * (TOL * fg0 + 2.0 ** -17)
    ratio = (np.abs(sg - so)[used] / bound[used]).max()
    print("16-level correlator: deepest level with products %d, worst |sum_gpu - sum_oracle| / bound = %.3f" % (deepest, ratio))
    assert ratio <= 1.0
    t0, G0, se0 = corr.result(N, 0.1)
    t1, G1, se1 = g.gt()
    assert np.array_equal(t0, t1) and t0[-1] >= 8 * 2 ** 11 * 0.1
