"""Pins of the oracle's rigid rotation (reading C-12: ``orc_align_to``) and of the rules around it.

The rotation that takes M/|M| = u onto e_C is fixed by three properties, none of which retypes the oracle's formula:
  (i)   it is RIGID and PROPER: every pairwise dot product S_i.S_j (hence the exchange energy) and every triple product
        S_i.(S_j x S_k) of a scattered state is unchanged to 1e-12;
  (ii)  it maps u onto e_C: M/|M| = e_C afterwards, |M| unchanged;
  (iii) it is the MINIMAL rotation: the axis k = u x e_C is left where it is (R k = k).
A rotation with R u = e_C and R k = k is unique, so a dropped Rodrigues term (the k (k.S)(1 - cos) term is exercised
only by states with k.S != 0), a wrong sign of the angle or a transposed matrix fails one of them.  The matrix is
recovered from the before / after states by least squares (numpy), not from the oracle's source.
"""
import numpy as np
import pytest

import oracle
from paper_2103_03517_b200 import inputs


def _direction(theta, phi):
    return np.array([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)])


def _recover_rotation(before, after):
    """least-squares 3x3 matrix with after_i = R before_i"""
    X, *_ = np.linalg.lstsq(before, after, rcond=None)
    return X.T


@pytest.mark.parametrize("theta,phi,mdir", [(1.1, -0.7, (0.3, -0.2, 0.9)), (2.6, 2.0, (-0.5, 0.1, 0.2)), (0.0, 0.0, (0.0, 1.0, 0.05))])
def test_align_is_the_minimal_rigid_rotation_onto_eC(theta, phi, mdir):
    shape = (8, 6, 4)
    N = shape[0] * shape[1] * shape[2]
    o = oracle.Oracle(*shape, Ku=0.05, Kc=0.1)
    S0 = inputs.thermal_like_spins(N, seed=4, spread=0.8, direction=mdir).astype(np.float64)
    S0 /= np.linalg.norm(S0, axis=1, keepdims=True)
    o.set_spins(S0)
    e = _direction(theta, phi)
    iso = oracle.Oracle(*shape)                # isotropic Hamiltonian: its total energy is the exchange energy alone
    iso.set_spins(S0); E0 = iso.total_energy()
    assert o.align_to(e) == 0
    S1 = o.get_spins()
    # (i) rigid and proper
    assert np.abs(S1 @ S1.T - S0 @ S0.T).max() < 1e-12
    idx = np.random.default_rng(1).integers(0, N, size=(200, 3))
    tp0 = np.einsum("ij,ij->i", S0[idx[:, 0]], np.cross(S0[idx[:, 1]], S0[idx[:, 2]]))
    tp1 = np.einsum("ij,ij->i", S1[idx[:, 0]], np.cross(S1[idx[:, 1]], S1[idx[:, 2]]))
    assert np.abs(tp1 - tp0).max() < 1e-12
    iso.set_spins(S1); assert abs(iso.total_energy() - E0) < 1e-10 * N
    assert np.abs(np.linalg.norm(S1, axis=1) - 1).max() < 1e-14
    # (ii) M/|M| = e_C, |M| kept
    M0, M1 = S0.sum(axis=0), S1.sum(axis=0)
    assert np.abs(M1 / np.linalg.norm(M1) - e).max() < 1e-12
    assert abs(np.linalg.norm(M1) - np.linalg.norm(M0)) < 1e-10
    # (iii) minimal rotation: the recovered matrix fixes k = u x e_C
    R = _recover_rotation(S0, S1)
    assert np.abs(R @ R.T - np.eye(3)).max() < 1e-12 and abs(np.linalg.det(R) - 1) < 1e-12
    u = M0 / np.linalg.norm(M0)
    k = np.cross(u, e); k /= np.linalg.norm(k)
    assert np.abs(R @ u - e).max() < 1e-12 and np.abs(R @ k - k).max() < 1e-12
    # the state is genuinely scattered about k (the k (k.S)(1 - cos) term matters): without it the check above fails
    assert np.abs(S0 @ k).mean() > 0.1


def test_align_from_the_exactly_antiparallel_state():
    """u = -e_C exactly (k = u x e_C = 0): a rotation by pi about an axis perpendicular to u.  The state is built from
    mirror pairs (sx, sy, sz), (-sx, -sy, sz) on consecutive sites, so the transverse sums cancel exactly in fp64."""
    shape = (8, 4, 4)
    N = shape[0] * shape[1] * shape[2]
    rng = np.random.default_rng(3)
    half = rng.standard_normal((N // 2, 3)) * 0.6 + np.array([0, 0, -1.0])
    half /= np.linalg.norm(half, axis=1, keepdims=True)
    S0 = np.empty((N, 3)); S0[0::2] = half; S0[1::2] = half * np.array([-1.0, -1.0, 1.0])
    o = oracle.Oracle(*shape)
    o.set_spins(S0)
    M0 = S0.sum(axis=0)
    assert M0[0] == 0.0 and M0[1] == 0.0 and M0[2] < 0
    e = np.array([0.0, 0.0, 1.0])
    assert o.align_to(e) == 0
    S1 = o.get_spins()
    assert np.abs(S1 @ S1.T - S0 @ S0.T).max() < 1e-12
    M1 = S1.sum(axis=0)
    assert np.abs(M1 / np.linalg.norm(M1) - e).max() < 1e-12 and abs(np.linalg.norm(M1) - np.linalg.norm(M0)) < 1e-10
    R = _recover_rotation(S0, S1)
    assert np.abs(R @ R.T - np.eye(3)).max() < 1e-12 and abs(np.linalg.det(R) - 1) < 1e-12
    assert abs(np.trace(R) + 1) < 1e-12                       # rotation angle pi: trace = 1 + 2 cos(pi)


def test_align_refuses_a_state_without_magnetisation():
    shape = (4, 4, 2)
    N = 32
    S = np.zeros((N, 3)); S[0::2, 2] = 1.0; S[1::2, 2] = -1.0
    o = oracle.Oracle(*shape)
    o.set_spins(S)
    assert o.align_to(np.array([0.0, 0.0, 1.0])) == -1       # |M|/N < 1e-6 (C-12)


def test_unconstrained_sweeps_invalidate_the_alignment():
    """constrained(theta, phi) -> unconstrained sweeps -> constrained(same theta, phi): M has drifted off e_C in between
    (the unconstrained move does not hold it), and the transverse component of M is conserved by every pair move, so the
    second constrained run must re-align first (C-12, "once per change" read as: whenever M/|M| may have left e_C)."""
    shape, T, theta, phi = (8, 8, 8), 1.0, 0.6, 0.3
    e = _direction(theta, phi)
    o = oracle.Oracle(*shape, Ku=0.05, cone0=0.6, seed=5)
    o.constrained_sweep(T, theta, phi, 20)
    ob = o.observables()
    assert np.abs(np.array(ob.M) / ob.m - e).max() < 1e-12                # pin P-16
    o.sweep(T, 30)
    ob = o.observables()
    drift = np.abs(np.array(ob.M) / ob.m - e).max()
    assert drift > 1e-3                                                    # the unconstrained sweeps moved M off e_C
    o.constrained_sweep(T, theta, phi, 1)
    ob = o.observables()
    assert np.abs(np.array(ob.M) / ob.m - e).max() < 1e-12                # re-aligned, then held


def test_torque_is_accumulated_by_constrained_sweeps_only():
    """the torque on M is the observable of the constrained method; unconstrained sweeps leave sum_torque alone."""
    o = oracle.Oracle(8, 8, 8, Ku=0.05, cone0=0.6, seed=2)
    o.sweep(0.5, 5)
    assert list(o.observables().sum_torque) == [0.0, 0.0, 0.0] and o.observables().n_samples == 5
    o.constrained_sweep(0.5, 0.7, 0.0, 5)
    ob = o.observables()
    assert ob.n_samples == 10 and abs(ob.sum_torque[1]) > 0


def test_cone_frame_uses_the_sign_bit_of_sz():
    """Reading C-29: sigma of the Duff frame is the SIGN BIT of S_z.  For S_z = -0.0 the two candidate frames differ by a
    rotation of the azimuth, so the trial spin tells them apart; both are unit vectors inside the cone."""
    theta, u0, u1 = 0.7, 0.35, 0.2
    Sp = np.array([0.6, 0.8, 0.0]); Sm = np.array([0.6, 0.8, -0.0])
    a, b = oracle.cone_move(Sp, theta, u0, u1), oracle.cone_move(Sm, theta, u0, u1)
    for v in (a, b):
        assert abs(np.linalg.norm(v) - 1) < 1e-14 and v @ Sp >= np.cos(theta) - 1e-14
    assert abs(a @ Sp - b @ Sp) < 1e-14                                   # same polar angle ...
    assert np.abs(a - b).max() > 1e-2                                     # ... different azimuth: the frames differ
    # sigma = -1 continues the S_z < 0 side: the trial spin is continuous across S_z -> 0-
    eps = np.array([0.6, 0.8, -1e-13]); eps /= np.linalg.norm(eps)
    assert np.abs(oracle.cone_move(eps, theta, u0, u1) - b).max() < 1e-10
    eps = np.array([0.6, 0.8, +1e-13]); eps /= np.linalg.norm(eps)
    assert np.abs(oracle.cone_move(eps, theta, u0, u1) - a).max() < 1e-10
