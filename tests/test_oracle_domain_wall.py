"""Pins for the domain-wall workload: anti-periodic boundary along x and the slice profile.

An anti-periodic wrap makes the spin on the other side enter Eq. (2) as -S_j.  Closed forms that fix the sign, the place
where it is applied and the profile:
  * the uniformly twisted state S_x = (sin(pi x/L), 0, cos(pi x/L)) is stationary in an anti-periodic box (every local
    field is parallel to its spin) with exchange energy -J (cos(pi/L) + 2) per site on an L x 2 x 2 lattice; in a
    PERIODIC box the same state has the wrap bond frustrated and is not stationary;
  * the uniform state is the ground state of the periodic box and costs +2J per wrap bond in the anti-periodic one;
  * at low temperature a wall relaxes to the tanh profile of Eq. (5) with width pi sqrt(A/K) = pi sqrt(J/(2K)) lattice units.
"""
import numpy as np
import pytest

import oracle


def _twist(L, ny=2, nz=2):
    x = np.arange(L)
    row = np.stack([np.sin(np.pi * x / L), np.zeros(L), np.cos(np.pi * x / L)], axis=1)
    return np.tile(row, (ny * nz, 1))                    # lexicographic: x fastest


@pytest.mark.parametrize("L", [4, 10, 24])
def test_twisted_state_energy_and_stationarity_under_the_antiperiodic_wrap(L):
    J = 0.8
    o = oracle.Oracle(L, 2, 2, periodic=(2, 1, 1), J=J)
    S = _twist(L); o.set_spins(S)
    ob = o.observables()
    assert abs(ob.E_exch - (-J * (np.cos(np.pi / L) + 2.0))) < 1e-13
    assert abs(o.total_energy() / o.N - ob.E_exch) < 1e-13
    # stationarity: rotating any single spin by +-eps about y changes the energy only at second order, equally both ways
    eps = 1e-4
    for site in (0, L // 2, L - 1, L + 1):
        t = np.arctan2(S[site, 0], S[site, 2])
        e0 = o.site_energy(site, S[site])
        up = o.site_energy(site, [np.sin(t + eps), 0, np.cos(t + eps)]) - e0
        dn = o.site_energy(site, [np.sin(t - eps), 0, np.cos(t - eps)]) - e0
        assert up > 0 and dn > 0 and abs(up - dn) < 1e-10 and abs(up - 0.5 * eps**2 * J * (2 * np.cos(np.pi / L) + 4)) < 1e-10
    # the same state in a periodic box: the wrap bond is frustrated, first-order energy change at the wrap
    p = oracle.Oracle(L, 2, 2, periodic=(1, 1, 1), J=J); p.set_spins(S)
    assert abs(p.observables().E_exch - (-J * (((L - 1) * np.cos(np.pi / L) - np.cos(np.pi / L)) / L + 2.0))) < 1e-14
    t = 0.0
    up = p.site_energy(0, [np.sin(eps), 0, np.cos(eps)]) - p.site_energy(0, S[0])
    dn = p.site_energy(0, [np.sin(-eps), 0, np.cos(-eps)]) - p.site_energy(0, S[0])
    assert abs(up + dn) < 1e-7 and abs(up - dn) > 1e-5      # linear term present: not stationary


def test_uniform_state_costs_two_j_per_wrap_bond():
    L, ny, nz, J = 8, 4, 6, 1.3
    up = np.tile([0.0, 0.0, 1.0], (L * ny * nz, 1))
    a = oracle.Oracle(L, ny, nz, periodic=(2, 1, 1), J=J); a.set_spins(up)
    p = oracle.Oracle(L, ny, nz, periodic=(1, 1, 1), J=J); p.set_spins(up)
    assert abs(p.total_energy() - (-3.0 * J * L * ny * nz)) < 1e-10
    assert abs((a.total_energy() - p.total_energy()) - 2.0 * J * ny * nz) < 1e-10     # ny nz wrap bonds, each +J instead of -J


def test_profile_is_the_slice_average():
    o = oracle.Oracle(6, 4, 2, periodic=(2, 1, 1))
    rng = np.random.default_rng(0)
    S = rng.standard_normal((o.N, 3)); S /= np.linalg.norm(S, axis=1, keepdims=True)
    o.set_spins(S)
    want = S.reshape(2, 4, 6, 3).mean(axis=(0, 1))
    assert np.allclose(o.profile_x(), want, atol=1e-15)


def test_wall_relaxes_to_the_tanh_profile_of_eq5():
    """T -> 0 limit of Eq. (5): m_z(x) = tanh((x - x0)/delta), delta = sqrt(J/(2K)) lattice units (continuum wall of the
    sc lattice with A = J/2a, K per site; Delta = pi delta).  delta = 5 sites: discreteness corrections are below 1 %."""
    L, J, K = 64, 1.0, 0.02
    delta = np.sqrt(J / (2 * K))
    o = oracle.Oracle(L, 2, 2, periodic=(2, 1, 1), J=J, Ku=K, cone0=0.3, adaptive=False, seed=3)
    x = np.arange(L)
    th = 2 * np.arctan(np.exp((x - 31.3) / 8.0))            # start from a wall of the wrong width (8 sites) and position
    row = np.stack([np.sin(th), np.zeros(L), np.cos(th)], axis=1)
    o.set_spins(np.tile(row, (4, 1)))
    o.set_sampling(False)
    for cone, n in ((0.2, 2000), (0.05, 6000), (0.02, 8000), (0.005, 8000), (0.002, 6000)):
        o.set_cone(cone); o.sweep(1e-7, n)                  # zero-temperature descent with a shrinking cone
    mz = o.profile_x()[:, 2]
    x0 = np.interp(0.0, -mz, x)                             # zero crossing (mz decreases)
    assert np.abs(mz - np.tanh(-(x - x0) / delta)).max() < 0.02
    # wall energy per unit cross-section 4 sqrt(A K) = 2 sqrt(2 J K) (Eq. 5 with C = 1 site), relative to the uniform state
    e_wall = (o.total_energy() - (-(3 * J + K) * o.N)) / 4.0
    assert abs(e_wall / (2 * np.sqrt(2 * J * K)) - 1) < 0.01
