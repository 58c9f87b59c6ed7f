"""Host analysis helpers on synthetic numbers with known answers, and on the oracle's wall."""
import types

import numpy as np

import oracle
from paper_2103_03517_b200 import analysis


def test_susceptibility_of_a_known_sample():
    rng = np.random.default_rng(0)
    N, T, n = 4096, 1.3, 500
    m = 0.5 + 0.01 * rng.standard_normal((n, 4))
    obs = types.SimpleNamespace(n_samples=n, n_sites=N, sum_m=m.sum(axis=0), sum_m2=(m * m).sum(axis=0))
    assert np.allclose(analysis.susceptibilities(obs, T), N / T * m.var(axis=0), rtol=1e-10)


def test_bloch_fit_recovers_the_papers_exponent():
    T = np.linspace(0.1, 1.4, 14)
    m = (1 - T / 1.4451) ** 0.340                           # k_B T_C / J = 1.4451, beta = 0.340
    tc, beta, _ = analysis.fit_bloch(T, m + 1e-4 * np.random.default_rng(1).standard_normal(len(T)))
    assert abs(tc - 1.4451) < 5e-3 and abs(beta - 0.340) < 5e-3


def test_wall_fit_and_stiffness_on_a_synthetic_profile():
    x = np.arange(80)
    mz = 0.83 * np.tanh(-np.pi * (x - 37.3) / 21.0) + 2e-3 * np.random.default_rng(2).standard_normal(80)
    m, x0, D = analysis.fit_domain_wall(mz)
    assert abs(m - 0.83) < 5e-3 and abs(x0 - 37.3) < 0.1 and abs(D - 21.0) < 0.2
    m2, _, D2 = analysis.fit_domain_wall(-mz)               # wall of the other handedness
    assert abs(m2 - m) < 1e-6 and abs(D2 - D) < 1e-6
    assert abs(analysis.exchange_stiffness(0.02, np.pi * 5.0) - 0.5) < 1e-12      # A = K delta^2 with delta = sqrt(A/K)


def test_wall_fit_on_the_oracles_relaxed_wall():
    """T -> 0: Delta = pi sqrt(J / 2K) and A = K Delta^2 / pi^2 = J / 2 (the continuum stiffness of the sc chain)."""
    L, J, K = 64, 1.0, 0.02
    o = oracle.Oracle(L, 2, 2, periodic=(2, 1, 1), J=J, Ku=K, cone0=0.3, adaptive=False, seed=3)
    x = np.arange(L); th = 2 * np.arctan(np.exp((x - 31.3) / 6.0))
    o.set_spins(np.tile(np.stack([np.sin(th), np.zeros(L), np.cos(th)], axis=1), (4, 1)))
    o.set_sampling(False)
    for cone, n in ((0.1, 3000), (0.02, 8000), (0.005, 8000), (0.002, 6000)):
        o.set_cone(cone); o.sweep(1e-7, n)
    m, x0, D = analysis.fit_domain_wall(o.profile_x()[:, 2])
    assert abs(m - 1) < 5e-3 and abs(D / (np.pi * np.sqrt(J / (2 * K))) - 1) < 0.02
    assert abs(analysis.exchange_stiffness(K, D) / (J / 2) - 1) < 0.04


def test_torque_route_and_power_law():
    theta = np.deg2rad(np.arange(0, 91, 9))                 # BASELINE.json configs[3]: 0..90 deg in 10 steps
    K = 0.0371
    tau = -K * np.sin(2 * theta) + 1e-5 * np.random.default_rng(3).standard_normal(len(theta))
    assert abs(analysis.anisotropy_from_torque(theta, tau) - K) < 2e-5
    m = np.linspace(0.3, 0.98, 12)
    k, K0 = analysis.power_law_exponent(m, 0.05 * m ** 2.95)                        # P:52 uniaxial exponent
    assert abs(k - 2.95) < 1e-9 and abs(K0 - 0.05) < 1e-9


def test_eq4_easy_axis_scaling_special_values():
    """Eq. (4): k = 1 on the easy axis at T = 0, k = 0 for an isotropic spin distribution (<S_z^2> = 1/3,
    <Sx^2 Sy^2 + Sy^2 Sz^2 + Sz^2 Sx^2> = 1/5), and the l = 2 / l = 4 harmonic averages in between."""
    Ku, Kc = 0.05, 0.01
    assert abs(analysis.anisotropy_scaling_easy_axis(-Ku, Ku=Ku) - 1.0) < 1e-14
    assert abs(analysis.anisotropy_scaling_easy_axis(-Ku / 3.0, Ku=Ku)) < 1e-14
    assert abs(analysis.anisotropy_scaling_easy_axis(0.0, Kc=Kc) - 1.0) < 1e-14
    assert abs(analysis.anisotropy_scaling_easy_axis(Kc / 5.0, Kc=Kc)) < 1e-14
    rng = np.random.default_rng(5)                           # a cone of spins about z: compare with the harmonics directly
    c = 1 - 0.3 * rng.random(200000); ph = 2 * np.pi * rng.random(200000); s = np.sqrt(1 - c * c)
    S = np.stack([s * np.cos(ph), s * np.sin(ph), c], axis=1)
    Eu = (-Ku * S[:, 2] ** 2).mean()
    Ec = (Kc * (S[:, 0] ** 2 * S[:, 1] ** 2 + S[:, 1] ** 2 * S[:, 2] ** 2 + S[:, 2] ** 2 * S[:, 0] ** 2)).mean()
    assert abs(analysis.anisotropy_scaling_easy_axis(Eu, Ku=Ku) - (1.5 * (c * c).mean() - 0.5)) < 1e-12
    x2, y2, z2 = (S ** 2).T
    assert abs(analysis.anisotropy_scaling_easy_axis(Ec, Kc=Kc) - (1 - 5 * (x2 * y2 + y2 * z2 + z2 * x2).mean())) < 1e-12


def test_eq4_agrees_with_the_constrained_torque_route_on_the_oracle():
    """P:59 "obtaining identical results to the constrained Monte Carlo algorithm": 16^3, K_u = 0.05, T = 0.3 (pin P-18's point).
    Eq. (4) from an unconstrained run and K(T)/K from the constrained torque at theta = 45 deg agree within 2 %."""
    Ku, T = 0.05, 0.3
    o = oracle.Oracle(16, 16, 16, Ku=Ku, cone0=0.5, adaptive=True, seed=11)
    o.sweep(T, 300)
    Ea = []
    for _ in range(120):
        o.sweep(T, 5); Ea.append(o.observables().E_aniso)
    k4 = analysis.anisotropy_scaling_easy_axis(float(np.mean(Ea)), Ku=Ku)
    c = oracle.Oracle(16, 16, 16, Ku=Ku, cone0=0.5, adaptive=True, seed=12)
    th = np.pi / 4
    c.constrained_sweep(T, th, 0.0, 300); c.reset_accumulators(); c.constrained_sweep(T, th, 0.0, 600)
    ob = c.observables()
    ktq = analysis.anisotropy_from_torque([th], [ob.sum_torque[1] / ob.n_samples]) / Ku
    assert abs(k4 - ktq) < 0.02 * ktq and 0.75 < k4 < 0.83                                   # SURVEY P-18 scratch value 0.7915


def test_eq7_transverse_susceptibility_on_the_oracle():
    """Eq. (7): the hard-axis susceptibility of Eq. (6) equals m^2 / (2 K(T)) below T_C (reduced units, C-18).
    Strong anisotropy keeps the transverse fluctuations small against the box (N chi_perp T << N^2): 12^3, K_u = 0.5, T = 0.6."""
    Ku, T, L = 0.5, 0.6, 12
    o = oracle.Oracle(L, L, L, Ku=Ku, cone0=0.5, adaptive=True, seed=21)
    o.sweep(T, 400); o.reset_accumulators()
    Ea = []
    for _ in range(300):
        o.sweep(T, 10); Ea.append(o.observables().E_aniso)
    ob = o.observables()
    chi = analysis.susceptibilities(ob, T)
    chi_perp = 0.5 * (chi[1] + chi[2])                                                        # easy axis z: hard axes x, y
    m = ob.sum_m[0] / ob.n_samples
    K_T = Ku * analysis.anisotropy_scaling_easy_axis(float(np.mean(Ea)), Ku=Ku)
    pred = analysis.chi_perp_uniaxial(m, K_T)
    assert abs(chi_perp / pred - 1) < 0.15


def test_eq8_multi_bloch_fit_recovers_the_mean_curie_temperature():
    """Eq. (8): a film's m(T) synthesised from five grains' Bloch laws; the fit's weighted mean T_C converges."""
    T = np.linspace(0.05, 1.5, 30)
    w = np.array([0.1, 0.2, 0.3, 0.25, 0.15]); tc = np.array([0.9, 1.05, 1.2, 1.3, 1.4]); beta = np.full(5, 0.34)
    m = analysis.multi_bloch(T, w, tc, beta)
    assert abs(m[0] - (w * (1 - T[0] / tc) ** 0.34).sum()) < 1e-14 and m[-1] == 0.0
    tbar = float((w * tc).sum())
    w1, tc1, b1, t1, rms1 = analysis.fit_multi_bloch(T, m, 1)
    w5, tc5, b5, t5, rms5 = analysis.fit_multi_bloch(T, m, 5)
    assert abs(w5.sum() - 1) < 1e-12 and (np.diff(tc5) >= 0).all()
    assert rms5 < rms1 and rms5 < 5e-3
    assert abs(t5 - tbar) < 0.04 and abs(t5 - tbar) <= abs(t1 - tbar) + 1e-9
