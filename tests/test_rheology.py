"""Host post-processing of G(t) (section 4.1, eqs 55-59, 64):
the oracle's definitions against closed forms, then libssm's ssm_moduli / ssm_eta0 / ssm_tau_d
against the oracle on the lag grid the multi-tau correlator produces.  No GPU is involved."""
import numpy as np
import pytest

import paper_1106_2899_b200 as ssm
from oracle import rheology as ref


def multitau_lags(levels=16, bins=16, base=0.1):
    """The 136 distinct lags of DESIGN.md section 7: level 0 bins 0..15, level l > 0 bins 8..15."""
    t = [k * base for k in range(bins)]
    for lev in range(1, levels):
        t += [k * 2.0 ** lev * base for k in range(bins // 2, bins)]
    return np.array(t)


def test_oracle_against_maxwell_closed_forms():
    tau, g = 3.0, 0.7
    t = np.linspace(0.0, 90.0, 90001)                  # fine grid: trapezoid error ~ (dt w)^2 / 12
    G = g * np.exp(-t / tau)
    w = np.array([0.01, 0.1, 1.0 / 3.0, 1.0, 3.0])
    g1, g2 = ref.moduli(t, G, w)
    x = w * tau
    assert np.allclose(g1, g * x * x / (1 + x * x), rtol=2e-5, atol=1e-9)
    assert np.allclose(g2, g * x / (1 + x * x), rtol=2e-5, atol=1e-9)
    assert abs(ref.eta0(t, G) - g * tau) < 1e-6
    assert abs(ref.tau_d(t, G, 10.0, 60.0) - tau) < 1e-9
    # |eta*|(w) = g tau / sqrt(1 + w^2 tau^2): tends to eta0 = g tau as w -> 0 (what the Cox-Merz rule, eq 63, needs)
    assert np.allclose(ref.dynamic_viscosity(g1, g2, w), g * tau / np.sqrt(1 + x * x), rtol=2e-5)
    assert abs(ref.dynamic_viscosity(g1, g2, w)[0] - ref.eta0(t, G)) < 1e-3 * g * tau


def test_oracle_against_the_rouse_spectrum():
    """Rouse chain (Z = 0): G(t) N = sum_p exp(-2 k_p t), k_p = 12 sin^2(p pi / 2N):
    eta0 N = sum 1/(2 k_p), tau_d = 1/(2 k_1), G'(w) N = sum w^2 tau_p^2/(1 + w^2 tau_p^2)."""
    N = 16
    kp = 12.0 * np.sin(np.arange(1, N) * np.pi / (2 * N)) ** 2
    tp = 1.0 / (2.0 * kp)
    t = np.linspace(0.0, 200.0, 200001)
    G = np.exp(-t[:, None] / tp[None, :]).sum(1) / N
    assert abs(ref.eta0(t, G) * N - tp.sum()) < 1e-4          # trapezoid error dt^2/12 sum_p 1/tau_p = 1.5e-5
    assert abs(ref.tau_d(t, G, 60.0, 150.0) - tp[0]) < 1e-3 * tp[0]
    w = np.array([0.02, 0.2, 2.0])
    g1, g2 = ref.moduli(t, G, w)
    x = w[:, None] * tp[None, :]
    assert np.allclose(g1 * N, (x * x / (1 + x * x)).sum(1), rtol=1e-4)
    assert np.allclose(g2 * N, (x / (1 + x * x)).sum(1), rtol=1e-4)


def test_library_equals_oracle_on_the_multitau_grid():
    rng = np.random.default_rng(5)
    t = multitau_lags()
    assert len(t) == 136
    G = 0.6 * np.exp(-t / 0.8) + 0.1 * np.exp(-t / 150.0) + 1e-3 * rng.standard_normal(len(t))
    w = np.logspace(-4, 1, 41)
    a1, a2 = ssm.moduli(t, G, w)
    b1, b2 = ref.moduli(t, G, w)
    assert np.allclose(a1, b1, rtol=1e-12, atol=1e-14) and np.allclose(a2, b2, rtol=1e-12, atol=1e-14)
    assert abs(ssm.eta0(t, G) - ref.eta0(t, G)) < 1e-12
    assert np.allclose(ssm.eta_star(t, G, w), ref.dynamic_viscosity(b1, b2, w), rtol=1e-12)
    with pytest.raises(ssm.SsmError):
        ssm.eta_star(t, G, [0.0])
    assert abs(ssm.tau_d(t, G, 100.0, 600.0) - ref.tau_d(t, G, 100.0, 600.0)) < 1e-9 * 150.0
    # ragged input: two lags; a window whose points are all non-positive
    assert abs(ssm.eta0([0.0, 2.0], [1.0, 0.5]) - 1.5) < 1e-15
    with pytest.raises(ssm.SsmError) as e:
        ssm.tau_d(t, -np.abs(G), 1.0, 100.0)
    assert e.value.code == ssm.SSM_ERANGE


def test_library_rejects_bad_tables():
    t = multitau_lags(4)
    G = np.exp(-t)
    for bad_t in (t[::-1], np.r_[t[:5], t[4], t[5:]], -t):
        with pytest.raises(ssm.SsmError) as e:
            ssm.eta0(bad_t, np.ones(len(bad_t)))
        assert e.value.code == ssm.SSM_EINVAL
    with pytest.raises(ssm.SsmError):
        ssm.moduli(t, G, [-1.0])
    with pytest.raises(ssm.SsmError):
        ssm.eta0([0.0], [1.0])
    with pytest.raises(ssm.SsmError):
        ssm.tau_d(t, G, 5.0, 1.0)


def test_stress_from_sums_is_the_mean_with_the_diagonal_constant():
    """ssm_stress_from_sums: value = sum / (2^18 M), sigma_aa one more -1 (eq 16: -N, the sums hold N - 1)."""
    sums = np.arange(24, dtype=np.int64).reshape(2, 12) * (1 << 18) * 5
    out = ssm.stress_from_sums(sums, 5)
    want = np.arange(24, dtype=np.float64).reshape(2, 12)
    want[:, :3] -= 1.0
    assert np.array_equal(out, want)
    from paper_1106_2899_b200 import shard
    assert np.array_equal(shard.stress_means(sums, 5), want)
    with pytest.raises(ssm.SsmError):
        ssm.stress_from_sums(sums, 0)
