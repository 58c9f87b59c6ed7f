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
