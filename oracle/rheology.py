"""ORACLE (test infrastructure, not the product): the post-processing of G(t) of PAPER.md
section 4.1 written out as the definitions, in numpy fp64.  Shares no code with libssm.

  storage / loss moduli  eqs (55), (56) P:L386-L390, "trapezoidal rule" P:L392
  zero-shear viscosity   eq (59)
  longest relaxation     eq (58): 1/tau_d = -lim ln G(t)/t, read on a finite table as the
                         least-squares slope of ln G over a window
  dynamic viscosity      eq (64), with the 1/w eq (63) needs (reading R25)

Pinned in tests/test_rheology.py by closed forms: a Maxwell mode G = g exp(-t/tau) has
G' = g w^2 tau^2/(1 + w^2 tau^2), G'' = g w tau/(1 + w^2 tau^2), eta0 = g tau, tau_d = tau;
the Rouse spectrum sums such modes."""
import numpy as np


def trapezoid(y, t):
    y = np.asarray(y, dtype=np.float64); t = np.asarray(t, dtype=np.float64)
    return float(np.sum(0.5 * (y[1:] + y[:-1]) * np.diff(t)))


def moduli(t, G, omega):
    t = np.asarray(t, dtype=np.float64); G = np.asarray(G, dtype=np.float64)
    g1 = np.array([w * trapezoid(G * np.sin(w * t), t) for w in omega])
    g2 = np.array([w * trapezoid(G * np.cos(w * t), t) for w in omega])
    return g1, g2


def eta0(t, G):
    return trapezoid(G, t)


def tau_d(t, G, t_lo, t_hi):
    t = np.asarray(t, dtype=np.float64); G = np.asarray(G, dtype=np.float64)
    m = (t >= t_lo) & (t <= t_hi) & (G > 0.0)
    slope = np.polyfit(t[m], np.log(G[m]), 1)[0]
    return -1.0 / slope


def dynamic_viscosity(g1, g2, omega):
    """eq (64) as the Cox-Merz rule of eq (63) needs it: |eta*|(w) = sqrt(G'^2 + G''^2) / w (the printed formula
    lacks the 1/w; reading R25)."""
    return np.sqrt(np.asarray(g1) ** 2 + np.asarray(g2) ** 2) / np.asarray(omega, dtype=np.float64)
