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


def anisotropy_scaling_easy_axis(E_aniso_per_site: float, Ku: float = 0.0, Kc: float = 0.0) -> float:
    """Eq. (4): the anisotropy scaling k(T) = K(T)/K(0) from a STANDARD (unconstrained) run whose magnetisation
    stays along an easy axis, through the average easy-axis anisotropy energy alone:
        k_u = 1 - 3 K_easy / (2 K_0,hard),   k_c = 1 - 5 K_easy / (3 K_0,hard).
    The paper measures the anisotropy energy from its minimum: K_easy = <E_aniso> - E_aniso(easy axis, T = 0) and
    K_0,hard = E_aniso(hard axis, T = 0) - E_aniso(easy axis, T = 0).  With this library's Eq. (2) conventions
    (uniaxial -Ku (S.e)^2: easy -Ku, hard 0; cubic +Kc (Sx^2 Sy^2 + Sy^2 Sz^2 + Sz^2 Sx^2): easy 0, hard <111> Kc/3)
    that is K_easy = Ku + <E_aniso>, K_0,hard = Ku and K_easy = <E_aniso>, K_0,hard = Kc/3.  Both are the thermal averages
    of the l = 2 / l = 4 harmonics, (3 <cos^2> - 1)/2 and 1 - 5 <Sx^2 Sy^2 + ...> (Callen-Callen).
    `E_aniso_per_site` is mc_obs.E_aniso averaged over sampling sweeps; exactly one of Ku, Kc must be non-zero."""
    if (Ku != 0.0) == (Kc != 0.0):
        raise ValueError("exactly one of Ku, Kc")
    if Ku != 0.0:
        return 1.0 - 3.0 * (Ku + E_aniso_per_site) / (2.0 * Ku)
    return 1.0 - 5.0 * E_aniso_per_site / (3.0 * (Kc / 3.0))


def chi_perp_uniaxial(m: float, K_T: float) -> float:
    """Eq. (7): transverse susceptibility of a uniaxial magnet below T_C, chi_perp = M_S(0) m^2 / (2 K_u(T)).
    In the reduced units of `susceptibilities` (mu_S = k_B = 1, energies per spin, C-18) M_S(0) -> 1 per site and
    K_u(T) -> K(T) = K k_u(T) per site, so chi_perp = m^2 / (2 K(T)); compare with the mean of the two hard-axis chi_alpha."""
    if not K_T > 0.0:
        raise ValueError("Eq. (7) holds for T < T_C where K(T) > 0")
    return m * m / (2.0 * K_T)


def multi_bloch(T, w, tc, beta):
    """Right-hand side of Eq. (8): sum_i w_i (1 - T/T_C,i)^beta_i, a term vanishing above its own T_C,i."""
    T = np.asarray(T, float)[:, None]
    w = np.asarray(w, float)[None, :]; tc = np.asarray(tc, float)[None, :]; beta = np.asarray(beta, float)[None, :]
    return (w * np.clip(1.0 - T / tc, 0.0, None) ** beta).sum(axis=1)


def fit_multi_bloch(T, m, n_terms: int, tc_range=None, beta0: float = 0.34, seed: int = 0):
    """Fit Eq. (8) with N_B = n_terms Bloch terms to a film's m(T): weights w_i >= 0 with sum 1, one
    (T_C,i, beta_i) per term.  Returns (w, T_C, beta, Tbar_C, rms) with Tbar_C = sum_i w_i T_C,i (second line of Eq. 8).
    Variable projection: for given (T_C,i, beta_i) the weights solve a non-negative least-squares problem with the
    sum-to-one condition as a heavily weighted extra row; the outer least squares moves (T_C,i, beta_i) inside tc_range
    (default: from the lowest T with m < 0.98 to 1.5 x the highest T) and [0.1, 1].  The paper increases N_B until
    Tbar_C converges (N_B > 10 for its films)."""
    from scipy.optimize import least_squares, nnls
    T = np.asarray(T, float); m = np.asarray(m, float)
    if tc_range is None:
        lo = float(T[m < 0.98].min()) if (m < 0.98).any() else float(T.min())
        tc_range = (max(lo, 1e-6), 1.5 * float(T.max()))
    n = int(n_terms)
    lam = 1e3

    def weights(tc, beta):
        A = np.clip(1.0 - T[:, None] / tc[None, :], 0.0, None) ** beta[None, :]
        w, _ = nnls(np.vstack([A, lam * np.ones((1, n))]), np.concatenate([m, [lam]]))
        s = w.sum()
        return w / s if s > 0 else np.full(n, 1.0 / n)

    def resid(p):
        tc, beta = p[:n], p[n:]
        return multi_bloch(T, weights(tc, beta), tc, beta) - m

    lb = np.concatenate([np.full(n, tc_range[0]), np.full(n, 0.1)])
    ub = np.concatenate([np.full(n, tc_range[1]), np.full(n, 1.0)])
    span = tc_range[1] - tc_range[0]
    # starting T_C,i: spread over the temperatures where m(T) falls (a term switches off at its own T_C,i)
    falling = T[m > 1e-3]
    t_hi = float(falling.max()) if falling.size else tc_range[1]
    tc0 = np.clip(np.linspace(tc_range[0] + 0.5 * (t_hi - tc_range[0]), min(tc_range[1], t_hi * 1.1), n + 2)[1:-1], lb[:n], ub[:n])
    p0 = np.concatenate([tc0, np.full(n, beta0)])
    best = None
    rng = np.random.default_rng(seed)
    for trial in range(6):
        start = p0 if trial == 0 else np.clip(p0 + np.concatenate([rng.normal(0, 0.08 * span, n), rng.normal(0, 0.05, n)]), lb, ub)
        r = least_squares(resid, start, bounds=(lb, ub), x_scale=np.concatenate([np.full(n, 0.1 * span), np.full(n, 0.1)]))
        if best is None or r.cost < best.cost:
            best = r
    tc, beta = best.x[:n], best.x[n:]
    w = weights(tc, beta)
    order = np.argsort(tc)
    w, tc, beta = w[order], tc[order], beta[order]
    return w, tc, beta, float((w * tc).sum()), float(np.sqrt(np.mean(best.fun ** 2)))
