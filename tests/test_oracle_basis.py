"""Pins for the oracle's basis mode ("4 simple tetragonal sub-lattices for hcp ... up to 8 non-interacting
subsets ... next-nearest neighbours"; reading C-32): hcp and simple cubic with next-nearest neighbours, EIGHT colours.  No GPU.

Fixed from outside the oracle: the geometry (sites from real-space coordinates, bonds = pairs at the bonding distance, periodic
images included), that no bond joins two sites of a sublattice, the classical ground state and equipartition, linear spin-wave
theory on the actual finite lattice, local dE = full recomputation; for the cubic lattice also the oracle's own simple cubic mode
(an independent code path with its own pins): with J2 = 0 the two describe the same Hamiltonian site by site, and their
equilibrium ensembles agree."""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

import oracle
from stats_util import blocked_mean_se

A_HCP, C_HCP = 1.0, np.sqrt(8.0 / 3.0)                          # ideal hcp: c/a = sqrt(8/3), nearest-neighbour distance a
# fractional coordinates of the orthohexagonal cell (a, sqrt3 a, c) of hcp: A layer (0,0,0), (1/2,1/2,0); B layer (1/2,1/6,1/2), (0,2/3,1/2)
HCP_FRAC = np.array([[0, 0, 0], [.5, .5, 0], [.5, 1 / 6, .5], [0, 2 / 3, .5]])


def _cell_and_basis(structure):
    if structure == "hcp":                                       # the cell is the orthohexagonal cell doubled along x
        cell = np.array([2 * A_HCP, np.sqrt(3) * A_HCP, C_HCP])
        single = HCP_FRAC * np.array([A_HCP, np.sqrt(3) * A_HCP, C_HCP])
        return cell, np.concatenate([single, single + np.array([A_HCP, 0, 0])])
    cell = np.array([2.0, 2.0, 2.0])                             # 2 x 2 x 2 block of a simple cubic lattice, sublattice = x + 2y + 4z
    return cell, np.array([[s & 1, (s >> 1) & 1, (s >> 2) & 1] for s in range(8)], float)


def _positions(structure, nx, ny, nz):
    cell, basis = _cell_and_basis(structure)
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    origin = np.stack([i.ravel(), j.ravel(), k.ravel()], axis=1) * cell
    return np.concatenate([origin + b for b in basis]), cell * np.array([nx, ny, nz])


def _bond_matrices(structure, shape):
    """W1[s, t], W2[s, t]: number of bonds of the nearest / next-nearest length between s and t over the periodic images."""
    r, box = _positions(structure, *shape); n = len(r)
    W1, W2 = np.zeros((n, n)), np.zeros((n, n))
    for a in (-1, 0, 1):
        for b in (-1, 0, 1):
            for c in (-1, 0, 1):
                d = r[None, :, :] + (np.array([a, b, c]) * box)[None, None, :] - r[:, None, :]
                d2 = (d ** 2).sum(axis=2)
                W1 += np.isclose(d2, 1.0)
                if structure == "sc_nnn": W2 += np.isclose(d2, 2.0)
    return W1, W2


def _rand_spins(n, seed):
    v = np.random.default_rng(seed).standard_normal((n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


CASES = [("hcp", (3, 2, 2)), ("hcp", (2, 3, 4)), ("hcp", (1, 1, 1)), ("hcp", (4, 1, 2)),
         ("sc_nnn", (3, 2, 2)), ("sc_nnn", (2, 3, 4)), ("sc_nnn", (1, 1, 1)), ("sc_nnn", (4, 1, 2))]


@pytest.mark.parametrize("structure,shape", CASES)
def test_bonds_are_the_geometric_neighbours(structure, shape):
    W1, W2 = _bond_matrices(structure, shape); n = len(W1); nc = n // 8
    assert np.allclose(W1, W1.T) and np.allclose(W2, W2.T)
    for a in range(8):                                            # eight non-interacting subsets
        blk = np.s_[a * nc:(a + 1) * nc]
        assert not W1[blk, blk].any() and not W2[blk, blk].any()
    assert (W1.sum(axis=1) == (12 if structure == "hcp" else 6)).all()
    if structure == "sc_nnn": assert (W2.sum(axis=1) == 12).all()
    J, J2 = 0.7, -0.3
    o = oracle.Oracle(*shape, structure=structure, J=J, J2=J2, seed=1)
    S = _rand_spins(n, 3); o.set_spins(S)
    Wj = J * W1 + J2 * W2
    E_geo = -0.5 * np.einsum("st,sa,ta->", Wj, S, S)
    assert abs(o.total_energy() - E_geo) < 1e-10 * max(1.0, abs(E_geo))
    assert abs(o.observables().E_exch * n - E_geo) < 1e-10 * max(1.0, abs(E_geo))
    h = Wj @ S
    for s in sorted({0, nc - 1, nc, 3 * nc, 5 * nc + nc // 2, n - 1}):
        v = _rand_spins(1, 100 + s)[0]
        assert abs(o.site_energy(s, v) + v @ h[s]) < 1e-12


def test_cubic_basis_mode_is_the_simple_cubic_lattice_site_by_site():
    """The 2 x 2 x 2-block description against the oracle's simple cubic mode (independent index arithmetic): with J2 = 0 the
    energy of a configuration, mapped site by site, is the same; with J2 the difference is the next-nearest-neighbour sum
    computed here from the array."""
    shape = (3, 2, 4); X, Y, Z = 2 * shape[0], 2 * shape[1], 2 * shape[2]
    S = _rand_spins(X * Y * Z, 9).reshape(Z, Y, X, 3)            # lexicographic simple cubic array [z][y][x]
    sc = oracle.Oracle(X, Y, Z, J=0.9, Ku=0.2, eu=(1, 1, 0), seed=1); sc.set_spins(S.reshape(-1, 3))
    mapped = np.concatenate([S[(s >> 2) & 1::2, (s >> 1) & 1::2, s & 1::2].reshape(-1, 3) for s in range(8)])
    for J2 in (0.0, 0.4):
        b = oracle.Oracle(*shape, structure="sc_nnn", J=0.9, J2=J2, Ku=0.2, eu=(1, 1, 0), seed=1); b.set_spins(mapped)
        nnn = 0.0
        for ax1, ax2 in ((0, 1), (0, 2), (1, 2)):                 # each next-nearest pair once: (+,+) and (+,-) along two axes
            for sg in (1, -1):
                nnn += np.einsum("zyxa,zyxa->", S, np.roll(np.roll(S, -1, axis=ax1), -sg, axis=ax2))
        assert abs(b.total_energy() - (sc.total_energy() - J2 * nnn)) < 1e-9


@pytest.mark.parametrize("structure,shape", CASES[:2] + CASES[4:6])
def test_local_energy_difference_is_the_full_recomputation(structure, shape):
    n = 8 * shape[0] * shape[1] * shape[2]
    o = oracle.Oracle(*shape, structure=structure, J=1.0, J2=0.35, Ku=0.3, eu=(1, 2, 2), Kc=0.2, B=(0.1, -0.2, 0.3), seed=2)
    S = _rand_spins(n, 5); o.set_spins(S)
    for s in np.random.default_rng(6).integers(0, n, 12):
        new = _rand_spins(1, int(s) + 50)[0]
        dE_local = o.site_energy(int(s), new) - o.site_energy(int(s), S[s])
        E0 = o.total_energy(); S2 = S.copy(); S2[s] = new; o.set_spins(S2)
        assert abs((o.total_energy() - E0) - dE_local) < 1e-12
        o.set_spins(S)


@pytest.mark.parametrize("structure,E0", [("hcp", -6.0), ("sc_nnn", -3.0 - 6 * 0.25)])
def test_ground_state_and_eight_colours(structure, E0):
    o = oracle.Oracle(2, 2, 2, structure=structure, J2=0.25, Ku=0.05, seed=3)
    ob = o.observables()
    assert abs(ob.E_total - (E0 - 0.05)) < 1e-12 and abs(ob.m - 1) < 1e-15
    S = o.get_spins()
    for colour in range(8):                                       # a pass of colour c moves sublattice c only
        n = o.half_sweep(1.5, colour); S2 = o.get_spins()
        moved = (S2 != S).any(axis=1)
        assert n > 0 and moved[colour * 8:(colour + 1) * 8].any() and not np.delete(moved, np.s_[colour * 8:(colour + 1) * 8]).any()
        S = S2
    assert abs(np.linalg.norm(S, axis=1) - 1).max() < 1e-12
    o.sweep(1.5, 3)                                               # a sweep = eight passes: the acceptance counts every site once
    assert 0.0 < o.observables().last_acceptance <= 1.0
    with pytest.raises(ValueError):
        o.constrained_sweep(1.0, 0.3, 0.0, 1)
    with pytest.raises(ValueError):
        oracle.Oracle(2, 2, 2, structure=structure, periodic=(1, 1, 0))


def test_uniforms_pair_the_x_neighbours_of_a_sublattice():
    """As on bcc / fcc (C-30): cells i and i ^ 1 of a sublattice row share one Philox block keyed on the even one's site id."""
    o = oracle.Oracle(4, 2, 2, structure="hcp", seed=9)
    for sub in (0, 5, 7):
        for (i, j, k) in ((0, 0, 0), (2, 1, 1)):
            first = sub * 16 + i + 4 * (j + 2 * k)
            r = oracle.philox4x32_10((first, 0 | (sub << 8), 7, 0), (9, 0))
            for half in (0, 1):
                u = o.site_uniforms(i + half, j, k, sub, 7)
                w0, w1 = r[2 * half], r[2 * half + 1]
                assert u == (oracle.uniform(w0), oracle.uniform_azimuth(w0, w1), oracle.uniform(w1))


_POOL = ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1))


def _trace(structure, shape, T, n_eq, n_s, seed, **kw):
    o = oracle.Oracle(*shape, structure=structure, seed=seed, **kw)
    o.set_sampling(False); o.sweep(T, n_eq); o.set_sampling(True); o.sweep(T, n_s)
    return o.trace()


@pytest.mark.parametrize("structure,shape,J2", [("hcp", (3, 2, 2), 0.0), ("sc_nnn", (2, 2, 2), 0.3)])
def test_low_temperature_spin_waves_and_equipartition(structure, shape, J2):
    """Linear spin-wave theory on the ACTUAL lattice: A = (sum_j J_ij + 2K) 1 - (J W1 + J2 W2); 1 - m_l = (T/N) sum over the
    eigenvalues of A except the uniform mode's (2K); E/N = E_0 + T."""
    K = 0.01
    W1, W2 = _bond_matrices(structure, shape); n = len(W1)
    Wj = W1 + J2 * W2
    z = Wj.sum(axis=1)[0]
    lam = np.linalg.eigvalsh((z + 2 * K) * np.eye(n) - Wj)
    assert abs(lam[0] - 2 * K) < 1e-9 and lam[1] > 0.5
    futs = {T: _POOL.submit(_trace, structure, shape, T, 1500, 8000, 11, Ku=K, J2=J2, cone0=0.3) for T in (0.03, 0.15)}
    for T, tol in ((0.03, 2e-4), (0.15, 2e-3)):
        tr = futs[T].result()
        m, se = blocked_mean_se(np.linalg.norm(tr[:, 2:5], axis=1))
        assert abs((1 - m) - T * (1 / lam[1:]).sum() / n) < tol + 3 * se
        E, seE = blocked_mean_se(tr[:, 5])
        assert abs(E - (-z / 2 - K + T)) < 2e-3 + 3 * seE


def test_cubic_basis_mode_samples_the_simple_cubic_ensemble():
    """J2 = 0: m(T) and E(T) of the eight-colour sweep on 4^3 cells against the two-colour sweep of the sc mode on the same 8^3
    lattice, below T_C (1.0) and near it (1.4): the order of the colour passes does not change the ensemble."""
    for T in (1.0, 1.4):
        fa = _POOL.submit(_trace, "sc_nnn", (4, 4, 4), T, 1000, 6000, 5, cone0=1.0)
        fb = _POOL.submit(_trace, "sc", (8, 8, 8), T, 1000, 6000, 6, cone0=1.0)
        ta, tb = fa.result(), fb.result()
        for f in (lambda t: np.linalg.norm(t[:, 2:5], axis=1), lambda t: t[:, 5]):
            a, sa = blocked_mean_se(f(ta)); b, sb = blocked_mean_se(f(tb))
            assert abs(a - b) < 3.5 * np.hypot(sa, sb) + 1e-3, (T, a, b)


def test_hcp_orders_like_a_twelve_neighbour_lattice():
    """The classical hcp Heisenberg model (z = 12) orders close to the fcc value k_B T_C / J = 3.18: strongly ordered at T = 2.2,
    disordered at T = 4.4 (a lattice with 6 or 8 bonds per site would be disordered at 2.2)."""
    lo = _POOL.submit(_trace, "hcp", (3, 2, 2), 2.2, 1000, 4000, 7, cone0=1.0)
    hi = _POOL.submit(_trace, "hcp", (3, 2, 2), 4.4, 1000, 4000, 8, cone0=1.5)
    m_lo = np.linalg.norm(lo.result()[:, 2:5], axis=1).mean(); m_hi = np.linalg.norm(hi.result()[:, 2:5], axis=1).mean()
    assert m_lo > 0.55 and m_hi < 0.25
