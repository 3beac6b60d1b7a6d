// ssm_rheo.cu -- host post-processing of the relaxation modulus (section 4.1).
//
// The paper turns the tabulated G(t) of eq (43) into the storage and loss moduli (eqs 55, 56, "numerically
// calculated by using the trapezoidal rule"), the zero-shear viscosity (eq 59), the longest
// relaxation time (eq 58) and the dynamic viscosity (eq 64).  These are O(lags x frequencies)
// host loops over the 136 lags ssm_gt() returns: no kernel is involved, and nothing here touches the device.
#include <cmath>
#include <cstdint>

#include "../../include/ssm.h"

namespace {
bool increasing(int32_t n, const double *t)
{
    for (int32_t i = 0; i < n; ++i) {
        if (!std::isfinite(t[i]) || t[i] < 0.0) return false;
        if (i > 0 && !(t[i] > t[i - 1])) return false;
    }
    return true;
}
}  // namespace

// eqs (55), (56): G'(w) = w int_0^inf G(t) sin(wt) dt, G''(w) = w int_0^inf G(t) cos(wt) dt, trapezoidal rule
// over the tabulated lags, truncated at the last lag
extern "C" int ssm_moduli(int32_t n_lags, const double *h_t, const double *h_G, int32_t n_omega, const double *h_omega,
                          double *h_storage, double *h_loss)
{
    if (n_lags < 2 || n_omega < 0 || !h_t || !h_G || (n_omega > 0 && (!h_omega || !h_storage || !h_loss))) return SSM_EINVAL;
    if (!increasing(n_lags, h_t)) return SSM_EINVAL;
    for (int32_t q = 0; q < n_omega; ++q) {
        const double w = h_omega[q];
        if (!std::isfinite(w) || w < 0.0) return SSM_EINVAL;
        double s = 0.0, c = 0.0;
        for (int32_t i = 0; i + 1 < n_lags; ++i) {
            const double dt = h_t[i + 1] - h_t[i];
            s += 0.5 * dt * (h_G[i] * std::sin(w * h_t[i]) + h_G[i + 1] * std::sin(w * h_t[i + 1]));
            c += 0.5 * dt * (h_G[i] * std::cos(w * h_t[i]) + h_G[i + 1] * std::cos(w * h_t[i + 1]));
        }
        h_storage[q] = w * s;
        h_loss[q] = w * c;
    }
    return SSM_OK;
}

// eq (64): dynamic viscosity eta*(w) = sqrt(G'^2 + G''^2) / w for the Cox-Merz comparison of eq (63), eta(rate) ~
// eta*(w = rate).  (P:L424 prints the square root without the 1/w; eq (63) needs it: for w -> 0, G'' -> eta_0 w, so
// only sqrt(G'^2 + G''^2) / w tends to eta_0 = eta(rate -> 0).  DESIGN.md reading R25.)
extern "C" int ssm_eta_star(int32_t n_lags, const double *h_t, const double *h_G, int32_t n_omega, const double *h_omega,
                            double *h_eta_star)
{
    if (n_omega < 0 || (n_omega > 0 && (!h_omega || !h_eta_star))) return SSM_EINVAL;
    for (int32_t q = 0; q < n_omega; ++q)
        if (!(h_omega[q] > 0.0) || !std::isfinite(h_omega[q])) return SSM_EINVAL;
    for (int32_t q = 0; q < n_omega; ++q) {
        double g1 = 0.0, g2 = 0.0;
        const int rc = ssm_moduli(n_lags, h_t, h_G, 1, h_omega + q, &g1, &g2);
        if (rc != SSM_OK) return rc;
        h_eta_star[q] = std::sqrt(g1 * g1 + g2 * g2) / h_omega[q];
    }
    return SSM_OK;
}

// Ensemble means (eq 54) of sigma (eq 16) and sigma^(v) (eq 76) from the raw fixed-point sums of ssm_stress_sums /
// ssm_stress_sums_device -- summed over every rank of a sharded ensemble -- and the TOTAL number of chains behind
// them: value = sum / (2^18 M); sigma_aa = 3 sum b_a^2 - N, of which the sums hold N - 1 of the N (one per bond), so
// the three diagonal components of sigma take one more -1 per chain (ssm_stress does the same for one context).
extern "C" int ssm_stress_from_sums(const int64_t *h_sums, int64_t n_samples, int64_t n_chains_total, double *h_out)
{
    if (n_samples < 0 || n_chains_total < 1 || (n_samples > 0 && (!h_sums || !h_out))) return SSM_EINVAL;
    const double scale = 1.0 / (262144.0 * (double)n_chains_total);
    for (int64_t i = 0; i < n_samples; ++i)
        for (int t = 0; t < 12; ++t) h_out[i * 12 + t] = (double)h_sums[i * 12 + t] * scale - (t < 3 ? 1.0 : 0.0);
    return SSM_OK;
}

// eq (59): eta_0 = int_0^inf G(t) dt, trapezoidal rule, truncated at the last lag
extern "C" int ssm_eta0(int32_t n_lags, const double *h_t, const double *h_G, double *h_eta0)
{
    if (n_lags < 2 || !h_t || !h_G || !h_eta0 || !increasing(n_lags, h_t)) return SSM_EINVAL;
    double s = 0.0;
    for (int32_t i = 0; i + 1 < n_lags; ++i) s += 0.5 * (h_t[i + 1] - h_t[i]) * (h_G[i] + h_G[i + 1]);
    *h_eta0 = s;
    return SSM_OK;
}

// eq (58): 1/tau_d = -lim ln G(t) / t.  On a finite noisy table the limit is read as the slope of the
// least-squares line through ln G(t) over the window t_lo <= t <= t_hi (points with G <= 0 are skipped).
extern "C" int ssm_tau_d(int32_t n_lags, const double *h_t, const double *h_G, double t_lo, double t_hi, double *h_tau_d)
{
    if (n_lags < 2 || !h_t || !h_G || !h_tau_d || !(t_hi > t_lo) || !increasing(n_lags, h_t)) return SSM_EINVAL;
    double n = 0.0, sx = 0.0, sy = 0.0, sxx = 0.0, sxy = 0.0;
    for (int32_t i = 0; i < n_lags; ++i) {
        if (h_t[i] < t_lo || h_t[i] > t_hi || !(h_G[i] > 0.0)) continue;
        const double x = h_t[i], y = std::log(h_G[i]);
        n += 1.0; sx += x; sy += y; sxx += x * x; sxy += x * y;
    }
    const double den = n * sxx - sx * sx;
    if (n < 2.0 || !(den > 0.0)) return SSM_ERANGE;
    const double slope = (n * sxy - sx * sy) / den;
    if (!(slope < 0.0)) return SSM_ERANGE;
    *h_tau_d = -1.0 / slope;
    return SSM_OK;
}
