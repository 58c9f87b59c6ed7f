"""Pins for the oracle's fcc mode ("4 simple cubic sub-lattices for fcc"; reading C-31): FOUR colours.  No GPU.

Fixed from outside the oracle: the geometry of the fcc lattice (built from coordinates), the classical ground state and
equipartition, linear spin-wave theory on the actual finite lattice, local dE = full recomputation, and the known Curie
temperature of the classical fcc Heisenberg model, k_B T_C / J = 3.178 (z = 12; high-temperature series and Monte Carlo give
J / k_B T_C = 0.3147).
"""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

import oracle
from stats_util import blocked_mean_se

OFF = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]])


def _positions(nx, ny, nz):
    """Site s = sub*Ncell + i + nx*(j + ny*k): sublattice 0 at the cell corner, 1..3 at the centres of the faces through it."""
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    A = np.stack([i.ravel(), j.ravel(), k.ravel()], axis=1).astype(float)
    return np.concatenate([A + o for o in OFF])


def _bond_matrix(shape, periodic):
    r = _positions(*shape); n = len(r)
    W = np.zeros((n, n))
    shifts = {(a * shape[0] if periodic[0] else 0, b * shape[1] if periodic[1] else 0, c * shape[2] if periodic[2] else 0)
              for a in (-1, 0, 1) for b in (-1, 0, 1) for c in (-1, 0, 1)}
    for t in shifts:
        d = r[None, :, :] + np.array(t, float)[None, None, :] - r[:, None, :]
        W += np.isclose((d ** 2).sum(axis=2), 0.5)
    return W


def _rand_spins(n, seed):
    v = np.random.default_rng(seed).standard_normal((n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


CASES = [((4, 4, 4), (1, 1, 1)), ((3, 5, 2), (1, 1, 1)), ((2, 2, 2), (1, 1, 1)), ((1, 3, 4), (1, 1, 1)),
         ((4, 3, 3), (1, 0, 1)), ((3, 3, 3), (0, 0, 0)), ((5, 1, 2), (0, 1, 0))]


@pytest.mark.parametrize("shape,periodic", CASES)
def test_bonds_are_the_geometric_nearest_neighbours(shape, periodic):
    W = _bond_matrix(shape, periodic); n = len(W); nc = n // 4
    assert np.allclose(W, W.T)
    for a in range(4):                                            # four non-interacting subsets
        assert not W[a * nc:(a + 1) * nc, a * nc:(a + 1) * nc].any()
    if all(periodic):
        assert (W.sum(axis=1) == 12).all()
        for a in range(4):
            for b in range(4):
                if a != b: assert (W[a * nc:(a + 1) * nc, b * nc:(b + 1) * nc].sum(axis=1) == 4).all()
    o = oracle.Oracle(*shape, periodic=periodic, structure="fcc", J=0.7, seed=1)
    S = _rand_spins(n, 3); o.set_spins(S)
    E_geo = -0.7 * 0.5 * np.einsum("st,sa,ta->", W, S, S)
    assert abs(o.total_energy() - E_geo) < 1e-10 * max(1.0, abs(E_geo))
    assert abs(o.observables().E_exch * n - E_geo) < 1e-10 * max(1.0, abs(E_geo))
    h = 0.7 * W @ S
    for s in (0, nc - 1, nc, 2 * nc + 1 if nc > 1 else 2 * nc, 3 * nc, n - 1):
        v = _rand_spins(1, 100 + s)[0]
        assert abs(o.site_energy(s, v) + v @ h[s]) < 1e-12


@pytest.mark.parametrize("shape,periodic", CASES[:5])
def test_local_energy_difference_is_the_full_recomputation(shape, periodic):
    n = 4 * shape[0] * shape[1] * shape[2]
    o = oracle.Oracle(*shape, periodic=periodic, structure="fcc", J=1.0, Ku=0.3, eu=(1, 2, 2), Kc=0.2, B=(0.1, -0.2, 0.3), seed=2)
    S = _rand_spins(n, 5); o.set_spins(S)
    for s in np.random.default_rng(6).integers(0, n, 12):
        new = _rand_spins(1, int(s) + 50)[0]
        dE_local = o.site_energy(int(s), new) - o.site_energy(int(s), S[s])
        E0 = o.total_energy(); S2 = S.copy(); S2[s] = new; o.set_spins(S2)
        assert abs((o.total_energy() - E0) - dE_local) < 1e-12
        o.set_spins(S)


def test_ground_state_and_four_colours():
    o = oracle.Oracle(3, 3, 3, structure="fcc", Ku=0.05, seed=3)
    ob = o.observables()
    assert abs(ob.E_total - (-6.0 - 0.05)) < 1e-12 and abs(ob.m - 1) < 1e-15     # z/2 = 6 bonds per spin
    S = o.get_spins()
    for colour in range(4):                                       # a pass of colour c moves sublattice c only
        n = o.half_sweep(1.5, colour); S2 = o.get_spins()
        moved = (S2 != S).any(axis=1)
        assert n > 0 and moved[colour * 27:(colour + 1) * 27].any() and not np.delete(moved, np.s_[colour * 27:(colour + 1) * 27]).any()
        S = S2
    assert abs(np.linalg.norm(S, axis=1) - 1).max() < 1e-12
    o.sweep(1.5, 3)                                               # a sweep = four passes: acceptance counts every site once
    assert 0.0 < o.observables().last_acceptance <= 1.0
    with pytest.raises(ValueError):
        o.constrained_sweep(1.0, 0.3, 0.0, 1)


_POOL = ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1))


def _trace(shape, T, n_eq, n_s, seed, **kw):
    o = oracle.Oracle(*shape, structure="fcc", seed=seed, **kw)
    o.set_sampling(False); o.sweep(T, n_eq); o.set_sampling(True); o.sweep(T, n_s)
    return o.trace()


def test_low_temperature_spin_waves_and_equipartition():
    shape, K = (4, 4, 4), 0.01
    lam = np.linalg.eigvalsh((12.0 + 2 * K) * np.eye(256) - _bond_matrix(shape, (1, 1, 1)))
    assert abs(lam[0] - 2 * K) < 1e-9
    futs = {T: _POOL.submit(_trace, shape, T, 1500, 8000, 11, Ku=K, cone0=0.3) for T in (0.03, 0.15)}
    for T, tol in ((0.03, 1.5e-4), (0.15, 1.5e-3)):
        tr = futs[T].result()
        m, se = blocked_mean_se(np.linalg.norm(tr[:, 2:5], axis=1))
        assert abs((1 - m) - T * (1 / lam[1:]).sum() / 256) < tol + 3 * se
        E, seE = blocked_mean_se(tr[:, 5])
        assert abs(E - (-6 - K + T)) < 2e-3 + 3 * seE


def _binder(L, T):
    tr = _trace((L, L, L), T, 2000, 20000, 7, cone0=1.2)
    m = np.linalg.norm(tr[:, 2:5], axis=1)
    nb = 20; mb = m[: (len(m) // nb) * nb].reshape(nb, -1)
    m2, m4 = (mb ** 2).mean(axis=1), (mb ** 4).mean(axis=1)
    U = 1 - m4.mean() / (3 * m2.mean() ** 2)
    Uj = np.array([1 - np.delete(m4, i).mean() / (3 * np.delete(m2, i).mean() ** 2) for i in range(nb)])
    return U, np.sqrt((nb - 1) * Uj.var())


def test_curie_temperature_of_the_fcc_heisenberg_model():
    """Binder cumulants of 4^3 and 6^3 cells (256 / 864 spins) order below, cross at, and invert above k_B T_C / J = 3.178."""
    Ts = (2.95, 3.178, 3.42)
    futs = {(L, T): _POOL.submit(_binder, L, T) for L in (4, 6) for T in Ts}
    U = {k: f.result() for k, f in futs.items()}
    err = lambda T: np.hypot(U[(6, T)][1], U[(4, T)][1])
    assert U[(6, Ts[0])][0] - U[(4, Ts[0])][0] > 3 * err(Ts[0])
    assert U[(4, Ts[2])][0] - U[(6, Ts[2])][0] > 3 * err(Ts[2])
    assert abs(U[(6, Ts[1])][0] - U[(4, Ts[1])][0]) < 3 * err(Ts[1]) + 0.008
    assert abs(U[(6, Ts[1])][0] - 0.62) < 0.03
