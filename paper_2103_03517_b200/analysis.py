"""Host-side analysis of what the library exports: susceptibilities (Eq. 6), Bloch-law fit (Eq. 3),
domain-wall tanh fit and exchange stiffness (Eq. 5), anisotropy from the constrained torque, power-law
exponents K ~ m^k.  NumPy / SciPy on a handful of numbers per temperature point: none of this is on the hot path
and none of it touches the device.  "P:NN" = line of the paper's text.
"""
from __future__ import annotations

import numpy as np
from scipy.optimize import curve_fit


def susceptibilities(obs, T: float):
    """Relative susceptibilities of Eq. (6) in reduced units (mu_S = k_B = 1) from the accumulators of
    mc_observables: chi_alpha = (N / T) (<m_alpha^2> - <m_alpha>^2), alpha = l, x, y, z (C-18)."""
    n = float(obs.n_samples)
    if n < 2:
        raise ValueError("need at least two samples")
    mean = np.array(list(obs.sum_m)) / n
    mean2 = np.array(list(obs.sum_m2)) / n
    return float(obs.n_sites) / T * (mean2 - mean * mean)


def fit_bloch(T, m, tc0: float = 1.44, beta0: float = 0.34):
    """m(T) = (1 - T/T_C)^beta (Eq. 3) fitted over the points below T_C.  Returns (T_C, beta, covariance)."""
    T = np.asarray(T, float); m = np.asarray(m, float)
    f = lambda t, tc, beta: np.clip(1.0 - t / tc, 0.0, None) ** beta
    p, cov = curve_fit(f, T, m, p0=(tc0, beta0), bounds=([T[m > 0.05].max() * 1.0001, 0.05], [10 * tc0, 2.0]))
    return float(p[0]), float(p[1]), cov


def fit_domain_wall(mz, periodic_image: bool = False):
    """Fit m_z(x) = m tanh(-pi (x - x0) / Delta) (Fig. 2) to a slice profile (mc_profile_x()[:, 2]).
    Returns (m, x0, Delta) with Delta the wall width of Eq. (5) in lattice units (Delta = pi delta)."""
    mz = np.asarray(mz, float); x = np.arange(len(mz), dtype=float)
    sign = 1.0 if mz[: max(1, len(mz) // 8)].mean() >= 0 else -1.0         # the fit form has +m on the left
    y = sign * mz
    x0 = float(np.interp(0.0, -y, x)) if (np.diff(y) < 0).all() else float(np.argmin(np.abs(y)))
    m0 = max(1e-3, float(np.abs(y).max()))
    f = lambda xx, m, c, d: m * np.tanh(-np.pi * (xx - c) / d)
    p, _ = curve_fit(f, x, y, p0=(m0, x0, max(2.0, len(mz) / 6.0)), maxfev=20000)
    return float(abs(p[0])), float(p[1]), float(abs(p[2]))


def exchange_stiffness(K: float, Delta: float) -> float:
    """A(T) = K(T) Delta(T)^2 / pi^2 from Eq. (5), P:63 (energy per lattice spacing in reduced units)."""
    return K * Delta * Delta / (np.pi * np.pi)


def anisotropy_from_torque(theta, torque_y):
    """Uniaxial K(T) from the constrained torque (the route of Ref. [15]): tau_y(theta) = -K sin(2 theta) per site
    for M held at polar angle theta in the x-z plane; least squares over the theta points (BASELINE.json configs[3])."""
    s = np.sin(2.0 * np.asarray(theta, float)); t = np.asarray(torque_y, float)
    return float(-(s * t).sum() / (s * s).sum())


def power_law_exponent(m, K, m_min: float = 0.0):
    """k of K(T)/K(0) ~ m^k (2.95 uniaxial, 9.90 cubic; Table I for the exchange stiffness) by a log-log fit."""
    m = np.asarray(m, float); K = np.asarray(K, float)
    sel = (m > m_min) & (K > 0) & (m < 1.0)
    k, lnK0 = np.polyfit(np.log(m[sel]), np.log(K[sel]), 1)
    return float(k), float(np.exp(lnK0))
