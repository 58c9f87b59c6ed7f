"""Pins for the oracle's bcc mode ("2 simple cubic sub-lattices for bcc"; reading C-30).  No GPU.

What fixes the mode with nothing to compare against: the GEOMETRY of the bcc lattice (built here from coordinates, not
from the oracle's index arithmetic), the classical ground state and equipartition, linear spin-wave theory on the
actual finite lattice (eigenvalues of the geometric bond matrix), local dE = full recomputation, and the known Curie
temperature of the classical bcc Heisenberg model, k_B T_C / J = 2.0542 (z = 8).
"""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

import oracle
from stats_util import blocked_mean_se


def _positions(nx, ny, nz):
    """Site s = sub*Ncell + i + nx*(j + ny*k): A (sub 0) at the cell corner, B (sub 1) at the cell centre."""
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    A = np.stack([i.ravel(), j.ravel(), k.ravel()], axis=1).astype(float)
    return np.concatenate([A, A + 0.5])


def _bond_matrix(shape, periodic):
    """W[s, t] = number of nearest-neighbour bonds (length sqrt(3)/2) between sites s and t, from coordinates and the
    periodic images alone (a pair can be joined through several images when a periodic dimension is 1 or 2 cells)."""
    r = _positions(*shape); n = len(r)
    W = np.zeros((n, n))
    shifts = [np.array([a * shape[0] if periodic[0] else 0, b * shape[1] if periodic[1] else 0, c * shape[2] if periodic[2] else 0], float)
              for a in (-1, 0, 1) for b in (-1, 0, 1) for c in (-1, 0, 1)]
    shifts = list({tuple(s) for s in shifts})
    for t in shifts:
        d = r[None, :, :] + np.array(t)[None, None, :] - r[:, None, :]
        W += np.isclose((d ** 2).sum(axis=2), 0.75)
    return W


def _rand_spins(n, seed):
    v = np.random.default_rng(seed).standard_normal((n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


CASES = [((4, 4, 4), (1, 1, 1)), ((3, 5, 2), (1, 1, 1)), ((2, 2, 2), (1, 1, 1)), ((1, 3, 4), (1, 1, 1)),
         ((4, 3, 3), (1, 0, 1)), ((3, 3, 3), (0, 0, 0)), ((5, 1, 2), (0, 1, 0))]


@pytest.mark.parametrize("shape,periodic", CASES)
def test_bonds_are_the_geometric_nearest_neighbours(shape, periodic):
    """Total energy (the oracle's bond enumeration) against -J sum over geometric bonds, exchange field against W S, the
    per-site bond count (8 in a periodic box), and bipartiteness: no bond inside a sublattice."""
    W = _bond_matrix(shape, periodic); n = len(W); nc = n // 2
    assert np.allclose(W, W.T) and not W[:nc, :nc].any() and not W[nc:, nc:].any()
    if all(periodic):
        assert (W.sum(axis=1) == 8).all()
    o = oracle.Oracle(*shape, periodic=periodic, structure="bcc", J=0.7, Ku=0.0, seed=1)
    S = _rand_spins(n, 3); o.set_spins(S)
    E_geo = -0.7 * 0.5 * np.einsum("st,sa,ta->", W, S, S)
    assert abs(o.total_energy() - E_geo) < 1e-10 * max(1.0, abs(E_geo))
    assert abs(o.observables().E_exch * n - E_geo) < 1e-10 * max(1.0, abs(E_geo))
    h = 0.7 * W @ S                                               # E_i(S) = -S.h_i with J = 0.7, no on-site terms
    for s in (0, nc - 1, nc, n - 1, n // 3):
        v = _rand_spins(1, 100 + s)[0]
        assert abs(o.site_energy(s, v) + v @ h[s]) < 1e-12


@pytest.mark.parametrize("shape,periodic", CASES[:5])
def test_local_energy_difference_is_the_full_recomputation(shape, periodic):
    """P-5 on the bcc lattice, all four terms on, tilted axis: moving one spin changes the total energy by E_i(S') - E_i(S)."""
    n = 2 * shape[0] * shape[1] * shape[2]
    o = oracle.Oracle(*shape, periodic=periodic, structure="bcc", J=1.0, Ku=0.3, eu=(1, 2, 2), Kc=0.2, B=(0.1, -0.2, 0.3), seed=2)
    S = _rand_spins(n, 5); o.set_spins(S)
    rng = np.random.default_rng(6)
    for s in rng.integers(0, n, 12):
        new = _rand_spins(1, int(s) + 50)[0]
        dE_local = o.site_energy(int(s), new) - o.site_energy(int(s), S[s])
        E0 = o.total_energy(); S2 = S.copy(); S2[s] = new; o.set_spins(S2)
        assert abs((o.total_energy() - E0) - dE_local) < 1e-12
        o.set_spins(S)


def test_ground_state_and_sublattice_colours():
    o = oracle.Oracle(4, 4, 4, structure="bcc", Ku=0.05, seed=3)
    ob = o.observables()
    assert abs(ob.E_total - (-4.0 - 0.05)) < 1e-12 and abs(ob.m - 1) < 1e-15     # z/2 = 4 bonds per spin
    # a half-sweep of colour c moves sublattice c only (the other one is bit-identical)
    S0 = o.get_spins(); n0 = o.half_sweep(1.0, 0); S1 = o.get_spins()
    assert n0 > 0 and (S1[64:] == S0[64:]).all() and (S1[:64] != S0[:64]).any()
    n1 = o.half_sweep(1.0, 1); S2 = o.get_spins()
    assert n1 > 0 and (S2[:64] == S1[:64]).all() and (S2[64:] != S1[64:]).any()
    assert abs(np.linalg.norm(S2, axis=1) - 1).max() < 1e-12


def test_uniforms_pair_the_x_neighbours_of_a_sublattice():
    """Reading C-30: cells i and i ^ 1 of a sublattice row share one Philox block (words 0,1 / 2,3), keyed on the even one."""
    o = oracle.Oracle(4, 2, 2, structure="bcc", seed=9)
    for sub in (0, 1):
        for (i, j, k) in ((0, 0, 0), (2, 1, 1)):
            first = sub * 16 + i + 4 * (j + 2 * k)
            r = oracle.philox4x32_10((first, 0 | (sub << 8), 7, 0), (9, 0))
            for half in (0, 1):
                u = o.site_uniforms(i + half, j, k, sub, 7)
                w0, w1 = r[2 * half], r[2 * half + 1]
                assert u == (oracle.uniform(w0), oracle.uniform_azimuth(w0, w1), oracle.uniform(w1))


_POOL = ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1))


def _trace(shape, T, n_eq, n_s, seed, **kw):
    o = oracle.Oracle(*shape, structure="bcc", seed=seed, **kw)
    o.set_sampling(False); o.sweep(T, n_eq); o.set_sampling(True); o.sweep(T, n_s)
    return o.trace()


def test_low_temperature_spin_waves_and_equipartition():
    """Linear spin-wave theory on the ACTUAL lattice: with A = (8 J + 2 K) 1 - J W (W the geometric bond matrix),
    1 - m_l = (T / N) sum over the eigenvalues of A except the uniform mode's (K > 0 shifts it to 2 K; m_l = |M|/N is blind to
    a uniform tilt), and E/N = -4 J - K + T (two quadratic modes per spin)."""
    shape, K = (6, 6, 6), 0.01
    lam = np.linalg.eigvalsh((8.0 + 2 * K) * np.eye(432) - _bond_matrix(shape, (1, 1, 1)))
    assert abs(lam[0] - 2 * K) < 1e-9
    futs = {T: _POOL.submit(_trace, shape, T, 1500, 6000, 11, Ku=K, cone0=0.3) for T in (0.02, 0.1)}
    for T, tol in ((0.02, 1.5e-4), (0.1, 1.5e-3)):
        tr = futs[T].result()
        m, se = blocked_mean_se(np.linalg.norm(tr[:, 2:5], axis=1))
        assert abs((1 - m) - T * (1 / lam[1:]).sum() / 432) < tol + 3 * se
        E, seE = blocked_mean_se(tr[:, 5])
        assert abs(E - (-4 - K + T)) < 2e-3 + 3 * seE


def _binder(L, T):
    tr = _trace((L, L, L), T, 2000, 24000, 7, cone0=1.2)
    m = np.linalg.norm(tr[:, 2:5], axis=1)
    nb = 20; mb = m[: (len(m) // nb) * nb].reshape(nb, -1)
    m2, m4 = (mb ** 2).mean(axis=1), (mb ** 4).mean(axis=1)
    U = 1 - m4.mean() / (3 * m2.mean() ** 2)
    Uj = np.array([1 - np.delete(m4, i).mean() / (3 * np.delete(m2, i).mean() ** 2) for i in range(nb)])
    return U, np.sqrt((nb - 1) * Uj.var())


def test_curie_temperature_of_the_bcc_heisenberg_model():
    """k_B T_C / J = 2.0542 for the classical Heisenberg model on the bcc lattice (z = 8; high-precision Monte Carlo value,
    e.g. Peczak, Ferrenberg and Landau 1991: K_c = J / k_B T_C = 0.4868).  The Binder cumulant of the two sizes orders
    below, crosses at, and inverts above T_C, at the universal 3-D Heisenberg value ~0.62 -- a wrong coordination number
    (6 or 12 bonds) would put the crossing at ~1.44 or ~3.2."""
    Ts = (1.9, 2.0542, 2.22)
    futs = {(L, T): _POOL.submit(_binder, L, T) for L in (5, 8) for T in Ts}
    U = {k: f.result() for k, f in futs.items()}
    err = lambda T: np.hypot(U[(8, T)][1], U[(5, T)][1])
    assert U[(8, Ts[0])][0] - U[(5, Ts[0])][0] > 3 * err(Ts[0])
    assert U[(5, Ts[2])][0] - U[(8, Ts[2])][0] > 3 * err(Ts[2])
    assert abs(U[(8, Ts[1])][0] - U[(5, Ts[1])][0]) < 3 * err(Ts[1]) + 0.008
    assert abs(U[(8, Ts[1])][0] - 0.62) < 0.03


# ------------------------------------------------------------------------------ constrained MC (Table A2) on the bcc lattice
def test_constrained_pairing_on_a_sublattice():
    """The analytic pairing (C-11) acts on the cell order of a sublattice: a perfect matching inside the colour, roles
    randomised, partner varying; colour-linear index a <-> site = sublattice*Ncell + a."""
    o = oracle.Oracle(8, 4, 4, structure="bcc")
    Nc = o.N // 2
    lead_count = np.zeros(Nc); seen = [set() for _ in range(8)]
    for colour in (0, 1):
        assert [o.site_of(colour, a) for a in (0, 5, Nc - 1)] == [colour * Nc, colour * Nc + 5, colour * Nc + Nc - 1]
        for s in range(200):
            partner, lead = o.pairing(s, colour)
            a = np.arange(Nc)
            assert (partner[partner] == a).all() and (partner != a).all()
            assert lead.sum() == Nc // 2 and (lead[partner] == 1 - lead).all()
            lead_count += lead
            for i in range(8): seen[i].add(int(partner[i]))
    assert np.all(np.abs(lead_count / 400 - 0.5) < 5 * np.sqrt(0.25 / 400)) and min(len(x) for x in seen) > 3
    with pytest.raises(ValueError):
        oracle.Oracle(3, 3, 3, structure="bcc").pairing(0, 0)     # odd colour population (C-15)
    with pytest.raises(ValueError):
        oracle.Oracle(4, 4, 4, structure="fcc").constrained_sweep(1.0, 0.3, 0.0, 1)   # four colours: not a two-pass constrained sweep


def _ctrace(shape, T, theta, n_eq, n_s, seed, **kw):
    o = oracle.Oracle(*shape, structure="bcc", seed=seed, **kw)
    o.set_sampling(False); o.constrained_sweep(T, theta, 0.0, n_eq); o.set_sampling(True); o.constrained_sweep(T, theta, 0.0, n_s)
    return o.trace(), o.observables(), o.get_spins()


def test_constrained_direction_is_held_and_isotropic_ensemble_is_unchanged():
    """P-16 / P-17 on bcc: M/|M| = e_C to 1e-12 and the transverse sum conserved; with an isotropic Hamiltonian the constrained
    chain samples the unconstrained distribution of |M| and E (8^3 cells = 1024 spins, T = 1.5; the stale-M_L bias is O(1/N))."""
    th = 0.9; e = np.array([np.sin(th), 0.0, np.cos(th)])
    fc = _POOL.submit(_ctrace, (8, 8, 8), 1.5, th, 400, 3000, 5, cone0=1.0)
    fu = _POOL.submit(_trace, (8, 8, 8), 1.5, 400, 3000, 6, cone0=1.0)
    trc, ob, S = fc.result(); tru = fu.result()
    M = S.sum(axis=0)
    assert np.abs(M / np.linalg.norm(M) - e).max() < 1e-12
    assert np.abs(M - (M @ e) * e).max() < 1e-9
    for f in (lambda t: np.linalg.norm(t[:, 2:5], axis=1), lambda t: t[:, 5]):
        a, sa = blocked_mean_se(f(trc)); b, sb = blocked_mean_se(f(tru))
        assert abs(a - b) < 3 * np.hypot(sa, sb) + 1.5e-3


def test_constrained_torque_gives_the_anisotropy_constant():
    """P-18 on bcc: restoring torque per spin = K(T) sin 2 theta, K(T -> 0) = K_u (Table A2 with the bcc field)."""
    th = np.pi / 4
    tr, ob, _ = _ctrace((6, 6, 6), 0.01, th, 300, 600, 8, Ku=0.05, cone0=0.2)
    K = -(ob.sum_torque[1] / ob.n_samples) / np.sin(2 * th)
    m = np.linalg.norm(tr[:, 2:5], axis=1).mean()
    assert abs(K / (0.05 * m ** 3) - 1) < 0.02 and abs(K / 0.05 - 1) < 0.02
