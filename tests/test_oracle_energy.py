"""Deterministic pins for the oracle's energies, fields, decision variable, controller and pairing.

P-4 (|S| = 1), P-5 (local dE == full-lattice recomputation), torque == -dE/d(rotation), the wiring of one
Metropolis update (which Philox words feed which step), P-19 (controller), P-20 (determinism), and the
requirements R1-R4 on the constrained pairing (reading C-11).
"""
import numpy as np
import pytest

import oracle
from paper_2103_03517_b200 import inputs


def _tilted_axis():
    e = np.array([0.3, -0.5, 0.81]); return e / np.linalg.norm(e)


CASES = [
    dict(shape=(6, 4, 4), periodic=(1, 1, 1)),
    dict(shape=(2, 2, 2), periodic=(1, 1, 1)),          # every distinct neighbour counted twice
    dict(shape=(6, 5, 3), periodic=(1, 0, 0)),          # odd open dims
    dict(shape=(8, 4, 4), periodic=(1, 1, 0), masked=True),
    dict(shape=(2, 1, 1), periodic=(0, 0, 0)),          # the dimer
    dict(shape=(6, 4, 4), periodic=(2, 1, 1)),          # anti-periodic along x (domain-wall box)
    dict(shape=(2, 2, 2), periodic=(2, 1, 1)),          # L = 2 with an anti-periodic wrap: the two x-bonds cancel
    dict(shape=(8, 4, 4), periodic=(2, 1, 0), masked=True),
]


def _make(case, seed=3, **kw):
    nx, ny, nz = case["shape"]
    mask = inputs.random_bond_mask(nx, ny, nz, case["periodic"], seed=9, p_cut=0.3) if case.get("masked") else None
    o = oracle.Oracle(nx, ny, nz, periodic=case["periodic"], J=0.7, Ku=0.11, eu=_tilted_axis(), Kc=0.23,
                      B=(0.05, -0.02, 0.13), bond_mask=mask, seed=seed, **kw)
    o.set_spins(inputs.random_unit_spins(o.N, seed=seed, dtype=np.float64))
    return o


@pytest.mark.parametrize("case", CASES)
def test_p5_local_delta_e_equals_full_lattice_recomputation(case):
    o = _make(case)
    rng = np.random.default_rng(1)
    S = o.get_spins()
    for site in rng.integers(0, o.N, size=min(o.N, 12)):
        new = rng.standard_normal(3); new /= np.linalg.norm(new)
        e0 = o.total_energy()
        dE_local = o.site_energy(site, new) - o.site_energy(site, S[site])
        S2 = S.copy(); S2[site] = new
        o.set_spins(S2)
        dE_full = o.total_energy() - e0
        o.set_spins(S)
        assert abs(dE_local - dE_full) < 1e-12 * max(1.0, abs(e0))


@pytest.mark.parametrize("case", CASES)
def test_observable_energy_matches_bond_sum_and_terms_add_up(case):
    o = _make(case)
    ob = o.observables()
    assert abs(ob.E_total * o.N - o.total_energy()) < 1e-11 * o.N
    assert abs(ob.E_total - (ob.E_exch + ob.E_aniso + ob.E_zeeman)) < 1e-14
    S = o.get_spins()
    assert np.allclose(np.array(ob.M), S.mean(axis=0), atol=1e-14)
    assert abs(ob.m - np.linalg.norm(S.mean(axis=0))) < 1e-14
    assert abs(ob.E_zeeman + S.mean(axis=0) @ np.array([0.05, -0.02, 0.13])) < 1e-14


def test_energy_special_values_from_the_paper():
    # cubic easy axes are the Cartesian axes (E = 0) and the hard axis is the long cube diagonal (E = Kc/3)
    o = oracle.Oracle(4, 4, 4, J=0.0, Kc=0.7)
    for d, want in (((1, 0, 0), 0.0), ((0, 1, 0), 0.0), ((0, 0, 1), 0.0), ((1, 1, 1), 0.7 / 3), ((1, 1, 0), 0.7 / 4)):
        o.init_uniform(d)
        assert abs(o.observables().E_aniso - want) < 1e-15
    # uniaxial: E = -Ku along the easy axis, 0 perpendicular;  ferromagnet: E_exch = -3J per site (z = 6, bonds once, C-1)
    o = oracle.Oracle(4, 4, 4, J=1.3, Ku=0.2, eu=(0, 0, 1))
    o.init_uniform((0, 0, 1)); ob = o.observables()
    assert abs(ob.E_aniso + 0.2) < 1e-15 and abs(ob.E_exch + 3 * 1.3) < 1e-14
    o.init_uniform((1, 0, 0)); assert abs(o.observables().E_aniso) < 1e-15
    # open cube L^3: bonds = 3 L^2 (L-1)
    o = oracle.Oracle(4, 4, 4, periodic=(0, 0, 0), J=1.0)
    assert abs(o.observables().E_exch * 64 + 3 * 16 * 3) < 1e-12


def test_torque_is_minus_dE_by_rotation_angle():
    # rotate ALL spins rigidly by a small angle about axis a: dE/d(delta) = - N tau_a  (exchange drops out for symmetric bonds)
    o = _make(CASES[0])
    S = o.get_spins()
    tau = np.array(o.observables().torque)
    d = 1e-6
    for a in range(3):
        k = np.zeros(3); k[a] = 1.0
        def rot(sign):
            ang = sign * d
            return S * np.cos(ang) + np.cross(k, S) * np.sin(ang) + np.outer(S @ k, k) * (1 - np.cos(ang))
        o.set_spins(rot(+1)); ep = o.total_energy()
        o.set_spins(rot(-1)); em = o.total_energy()
        o.set_spins(S)
        assert abs(-(ep - em) / (2 * d) / o.N - tau[a]) < 1e-8
    # uniform state at polar angle t about y, easy axis z: tau_y = -K sin(2t)  (P:54 torque route, config c4)
    o = oracle.Oracle(4, 4, 4, Ku=0.05)
    t = 0.6
    o.init_uniform((np.sin(t), 0, np.cos(t)))
    assert np.allclose(o.observables().torque, (0, -0.05 * np.sin(2 * t), 0), atol=1e-15)


@pytest.mark.parametrize("case", CASES[:4])
def test_half_sweep_wiring_decision_variable_and_stream(case):
    """x = dE/T + ln u2; S' = cone(S,u0,u1); the uniforms follow reading C-26: sites x and x^2 of a row share the block
    Philox(key=seed, ctr=(index of the one with bit 1 of x clear, colour<<8, sweep)), two words each:
    u0 = top 23 bits of w0, u2 = top 23 bits of w1 (+ half), u1 = the 9 + 9 low bits (retyped here in integer arithmetic)."""
    seed = (7 << 32) | 123
    o = _make(case, seed=seed, cone0=0.9, adaptive=False)
    o.set_sweep((5 << 32) | 17)
    T = 0.8
    S = o.get_spins()
    for colour in (0, 1):
        before = o.get_spins()
        n, x, acc = o.half_sweep(T, colour, want_detail=True)
        after = o.get_spins()
        xs, ys, zs = inputs.site_coords(*o.shape)
        col = (xs + ys + zs) & 1
        assert n == acc.sum()
        assert np.isnan(x[col != colour]).all() and not np.isnan(x[col == colour]).any()
        assert (after[col != colour] == before[col != colour]).all()
        chk = oracle.Oracle(*o.shape, periodic=case["periodic"], J=0.7, Ku=0.11, eu=_tilted_axis(), Kc=0.23,
                            B=(0.05, -0.02, 0.13), bond_mask=o._mask)
        chk.set_spins(before)
        for site in np.nonzero(col == colour)[0][:40]:
            x_site = int(xs[site])
            first = int(site) - (x_site & 2)
            r = [int(v) for v in oracle.philox4x32_10([first, colour << 8, 17, 5], [123, 7])]
            w0, w1 = (r[2], r[3]) if (x_site & 2) else (r[0], r[1])
            u = [((w0 >> 9) + 0.5) / 2**23, (((w0 & 511) << 9) | (w1 & 511)) / 2**18, ((w1 >> 9) + 0.5) / 2**23]
            assert u == list(o.site_uniforms(x_site, int(ys[site]), int(zs[site]), colour, (5 << 32) | 17))
            Sn = oracle.cone_move(before[site], 0.9, u[0], u[1])
            xd = (chk.site_energy(site, Sn) - chk.site_energy(site, before[site])) / T + np.log(u[2])
            assert abs(xd - x[site]) < 1e-12
            assert acc[site] == (xd < 0)
            assert np.allclose(after[site], Sn if xd < 0 else before[site], atol=0)


def test_p4_unit_norm_is_invariant():
    o = oracle.Oracle(8, 8, 8, Ku=0.01, Kc=0.02, seed=1)
    o.set_spins(inputs.random_unit_spins(o.N, seed=2, dtype=np.float64))
    o.set_sampling(False)
    o.sweep(0.7, 300)
    assert np.abs(np.linalg.norm(o.get_spins(), axis=1) - 1).max() < 1e-12
    o.constrained_sweep(0.7, 0.4, 0.3, 200)
    assert np.abs(np.linalg.norm(o.get_spins(), axis=1) - 1).max() < 1e-12


def test_p19_controller_steps_clamps_and_rule():
    deg = np.pi / 180
    # exact +-1 degree steps, decided by 2*count > N (equality decreases: C-9)
    o = oracle.Oracle(4, 4, 4, cone0=0.5)
    N = o.N
    o.end_sweep(N // 2 + 1); assert o.observables().cone_rad == 0.5 + deg
    o.end_sweep(N // 2);     assert o.observables().cone_rad == 0.5 + deg - deg
    o.end_sweep(0);          assert abs(o.observables().cone_rad - (0.5 - deg)) < 1e-15
    # clamps at [1 deg, 180 deg]
    for _ in range(400): o.end_sweep(N)
    assert o.observables().cone_rad == np.pi
    for _ in range(400): o.end_sweep(0)
    assert o.observables().cone_rad == deg
    # non-adaptive: never moves
    o = oracle.Oracle(4, 4, 4, cone0=0.5, adaptive=False)
    o.end_sweep(N); assert o.observables().cone_rad == 0.5
    # closed loop: T >> J saturates at pi with acceptance > 0.5; moderate T settles near 0.5
    o = oracle.Oracle(8, 8, 8, cone0=0.5, seed=3); o.sweep(50.0, 200)
    ob = o.observables(); assert ob.cone_rad == np.pi and ob.last_acceptance > 0.5
    o = oracle.Oracle(8, 8, 8, Ku=0.01, cone0=0.5, seed=3); o.sweep(1.0, 600)
    tr = o.trace()
    assert abs(tr[200:, 0].mean() - 0.5) < 0.02
    steps = np.abs(np.diff(tr[:, 1])); assert np.allclose(steps, deg, atol=1e-14)


def test_p20_determinism_and_split_invariance():
    def run(splits, seed=42):
        o = oracle.Oracle(6, 6, 6, Ku=0.01, cone0=0.5, seed=seed)
        for n in splits: o.sweep(1.1, n)
        return o.get_spins(), o.trace()
    s1, t1 = run([30]); s2, t2 = run([30]); s3, t3 = run([1] * 30); s4, t4 = run([7, 23])
    assert (s1 == s2).all() and (t1 == t2).all() and (s1 == s3).all() and (t1 == t3).all() and (s1 == s4).all()
    s5, _ = run([30], seed=43)
    assert (s1 != s5).any()


# ---------------------------------------------------------------------------------------- pairing (C-11)
@pytest.mark.parametrize("shape", [(16, 16, 16), (8, 8, 8), (4, 4, 4), (2, 2, 2), (6, 6, 2), (12, 4, 2)])
def test_pairing_is_a_role_randomised_perfect_matching(shape):
    o = oracle.Oracle(*shape)
    Nc = o.N // 2
    lead_count = np.zeros(Nc); partners_seen = [set() for _ in range(min(Nc, 16))]
    n_sweeps = 200
    for colour in (0, 1):
        for s in range(n_sweeps):
            partner, lead = o.pairing(s, colour)
            assert (partner >= 0).all() and (partner < Nc).all()
            a = np.arange(Nc)
            assert (partner[partner] == a).all() and (partner != a).all()      # R1: involution without fixed points
            assert lead.sum() == Nc // 2 and (lead[partner] == 1 - lead).all()  # one leader per pair
            lead_count += lead
            for i in range(len(partners_seen)): partners_seen[i].add(int(partner[i]))
    p = lead_count / (2 * n_sweeps)
    assert np.all(np.abs(p - 0.5) < 5 * np.sqrt(0.25 / (2 * n_sweeps)))        # R3: every site leads with prob 1/2
    if Nc >= 16:
        assert min(len(s) for s in partners_seen) > 3                          # R4: partner varies
    # pure function of (seed, sweep, colour): R2
    q1, l1 = o.pairing(7, 1); q2, l2 = o.pairing(7, 1)
    assert (q1 == q2).all() and (l1 == l2).all()
    o2 = oracle.Oracle(*shape, seed=43)
    if Nc >= 64:
        assert any((o2.pairing(s, 0)[0] != o.pairing(s, 0)[0]).any() for s in range(4))


def test_pairing_same_colour_sites_and_colour_linear_index():
    o = oracle.Oracle(6, 4, 2)
    xs, ys, zs = inputs.site_coords(6, 4, 2)
    for colour in (0, 1):
        sites = [o.site_of(colour, a) for a in range(o.N // 2)]
        assert sorted(sites) == sorted(np.nonzero(((xs + ys + zs) & 1) == colour)[0].tolist())
        # a = (x>>1) + (nx/2)(y + ny z)
        for a, s in enumerate(sites):
            assert a == (xs[s] >> 1) + 3 * (ys[s] + 4 * zs[s])
    with pytest.raises(ValueError):
        oracle.Oracle(6, 3, 1, periodic=(1, 0, 0)).pairing(0, 0)               # odd colour population (C-15)
