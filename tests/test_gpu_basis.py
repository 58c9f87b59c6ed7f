"""GPU parity for the eight-colour lattices (reading C-32): hcp and simple cubic with next-nearest neighbours --
the CUDA pass (bond table derived in mc_api.cu) against the oracle's basis mode (bonds derived in mc_oracle.c), element by element
through the C ABI, same bar as the sc lattice (C-14)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

X_BAND, SPIN_TOL = 1e-5, 1e-4


@pytest.fixture(scope="module")
def mods():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    import oracle
    from paper_2103_03517_b200 import binding, build, inputs
    build.build()
    return oracle, binding, inputs


def _pair(mods, structure, shape, seed=42, cone=0.5, sweep=0, adaptive=False, **ham):
    oracle, binding, inputs = mods
    o = oracle.Oracle(*shape, seed=seed, cone0=cone, adaptive=adaptive, structure=structure, **ham)
    g = binding.Lattice(*shape, seed=seed, cone0=cone, adaptive=adaptive, structure=structure, **ham)
    o.set_sweep(sweep); g.set_sweep(sweep)
    return o, g


def _half(o, g, T, colour):
    before = g.get_spins()
    o.set_spins(before)
    n_o, x_o, acc_o = o.half_sweep(T, colour, want_detail=True)
    x_g, acc_g = g.half_sweep(T, colour, want_detail=True)
    after_g = g.get_spins().astype(np.float64); after_o = o.get_spins()
    nc = g.N // 8
    mine = (np.arange(g.N) // nc) == colour                  # colour = sublattice, stored contiguously
    assert (after_g[~mine] == before[~mine].astype(np.float64)).all()
    assert not np.isnan(x_g[mine]).any()
    differ = mine & (acc_g != acc_o)
    assert (np.abs(x_o[differ]) < X_BAND).all()
    agree = mine & ~differ
    assert np.abs(after_g[agree] - after_o[agree]).max() < SPIN_TOL
    changed = (after_g != before.astype(np.float64)).any(axis=1)
    assert (changed[mine] == (acc_g[mine] == 1)).all()
    assert np.abs(np.linalg.norm(after_g, axis=1) - 1).max() < 2e-7
    near = mine & (np.abs(x_o) < 2.0)
    return int(differ.sum()), float(np.abs(x_g[near] - x_o[near]).max()) if near.any() else 0.0


CASES = [
    ("hcp", (16, 12, 8), 3.0, 0.8, dict(Ku=0.05)),                                                   # near the ordering temperature
    ("hcp", (4, 1, 1), 1.0, 1.5, dict()),                                                             # one-cell-thick: neighbours counted several times
    ("hcp", (8, 2, 2), 4.0, np.pi, dict(Kc=0.2)),                                                     # 2-cell periodic dims
    ("hcp", (12, 5, 7), 1.3, 1.0, dict(Ku=0.2, eu=(0.3, -0.5, 0.81), Kc=0.1, B=(0.1, -0.05, 0.2))),   # odd dims, ragged grid, every term
    ("hcp", (32, 24, 20), 0.4, 0.4, dict(Ku=0.01)),                                                   # several CTAs per SM, low T
    ("sc_nnn", (16, 12, 8), 2.0, 0.8, dict(J2=0.3, Ku=0.05)),
    ("sc_nnn", (4, 1, 1), 1.0, 1.5, dict(J2=-0.2)),
    ("sc_nnn", (8, 2, 2), 2.5, np.pi, dict(J2=0.5, Kc=0.2)),
    ("sc_nnn", (12, 5, 7), 1.3, 1.0, dict(J2=0.25, Ku=0.2, eu=(0.3, -0.5, 0.81), Kc=0.1, B=(0.1, -0.05, 0.2))),
    ("sc_nnn", (32, 24, 20), 0.4, 0.4, dict(J2=0.1, Ku=0.01)),
]


@pytest.mark.parametrize("structure,shape,T,cone,ham", [CASES[0], CASES[3], CASES[5], CASES[8]])
def test_basis_half_sweep_parity_with_the_run_time_bond_table(mods, structure, shape, T, cone, ham):
    """The sweep passes default to the instantiations with compile-time bond tables; MC_PATH_GENERIC forces the one that reads
    the table mc_create uploaded (the stand-alone measurement always does)."""
    test_basis_half_sweep_parity(mods, structure, shape, T, cone, ham, path=1)


@pytest.mark.parametrize("structure,shape,T,cone,ham", CASES)
def test_basis_half_sweep_parity(mods, structure, shape, T, cone, ham, path=None):
    oracle, binding, inputs = mods
    o, g = _pair(mods, structure, shape, cone=cone, sweep=(5 << 32) | 777, **ham)
    if path is not None: g.debug_set_path(path)
    g.set_spins(inputs.random_unit_spins(g.N, seed=8))
    worst = 0.0
    for colour in (0, 1, 2, 3, 4, 5, 6, 7, 2, 5):
        f, dx = _half(o, g, T, colour)
        worst = max(worst, dx)
    assert worst < X_BAND
    g.set_spins(inputs.thermal_like_spins(g.N, 9, 0.2))
    for colour in range(8):
        f, dx = _half(o, g, T, colour)
        assert dx < X_BAND
    with pytest.raises(binding.McError):
        g.half_sweep(T, 8)
    g.close()


@pytest.mark.parametrize("structure,E0,ham", [("hcp", -6.0, dict()), ("sc_nnn", -3.0 - 6 * 0.25, dict(J2=0.25))])
def test_basis_observables_and_ground_state(mods, structure, E0, ham):
    oracle, binding, inputs = mods
    shape = (12, 6, 10)
    o, g = _pair(mods, structure, shape, Ku=0.1, eu=(1, 1, 0), Kc=0.05, B=(0.02, 0.0, -0.03), **ham)
    ob = g.observables()
    assert abs(ob.E_exch - E0) < 1e-6 and abs(ob.m - 1) < 1e-6
    s = inputs.random_unit_spins(g.N, seed=4); g.set_spins(s); o.set_spins(g.get_spins())
    a, b = g.observables(), o.observables()
    for name in ("m", "E_total", "E_exch", "E_aniso", "E_zeeman"):
        assert abs(getattr(a, name) - getattr(b, name)) < 3e-6, name
    assert np.abs(np.array(a.M) - np.array(b.M)).max() < 2e-6
    assert np.abs(np.array(a.torque) - np.array(b.torque)).max() < 2e-6
    with pytest.raises(binding.McError):
        g.constrained_sweep(1.0, 0.3, 0.0, 1)
    g.close()


@pytest.mark.parametrize("structure,ham", [("hcp", dict()), ("sc_nnn", dict(J2=0.3))])
def test_basis_sweep_equals_hooks_and_fused_energy(mods, structure, ham):
    """mc_sweep(T, n) = n x (eight hooks, end_sweep), bit for bit; the fused sums of the last sweep -- the exchange energy counted
    bond by bond in the pass of the bond's higher colour -- equal a fresh measurement of the final state."""
    oracle, binding, inputs = mods
    shape, T = (16, 8, 8), 2.5
    s0 = inputs.random_unit_spins(8 * 16 * 8 * 8, seed=5)
    o, a = _pair(mods, structure, shape, cone=0.5, adaptive=True, Ku=0.05, **ham); a.set_spins(s0)
    o2, b = _pair(mods, structure, shape, cone=0.5, adaptive=True, Ku=0.05, **ham); b.set_spins(s0)
    a.sweep(T, 6)
    for _ in range(6):
        for colour in range(8): b.half_sweep(T, colour)
        b.end_sweep()
    assert (a.get_spins() == b.get_spins()).all() and (a.trace() == b.trace()).all()
    ob = a.observables(); tr = a.trace()
    assert np.abs(tr[-1, 2:5] - np.array(ob.M)).max() < 1e-6 and abs(tr[-1, 5] - ob.E_total) < 1e-5
    assert (tr[:, 0] > 0).all() and (tr[:, 0] <= 1).all()
    assert np.allclose(np.abs(np.diff(tr[:, 1])), np.pi / 180, atol=1e-12)
    a.close(); b.close()


@pytest.mark.parametrize("structure,shape,ham,points", [
    ("hcp", (4, 3, 4), dict(), ((2.4, 0.45, 0.85), (4.2, 0.0, 0.2))),
    ("sc_nnn", (4, 4, 4), dict(J2=0.0), ((1.0, 0.55, 0.8), (1.9, 0.0, 0.2))),          # J2 = 0: the simple cubic lattice, T_C = 1.443
])
def test_basis_ensemble_matches_oracle(mods, structure, shape, ham, points):
    """m(T) of an equilibrated run: GPU against the oracle within 3 standard errors, in the ordered and in the disordered phase."""
    from stats_util import blocked_mean_se
    oracle, binding, inputs = mods
    for T, lo, hi in points:
        o, g = _pair(mods, structure, shape, seed=3, cone=1.0, adaptive=True, Ku=0.01, **ham)
        o.set_sampling(False); o.sweep(T, 500); o.set_sampling(True); o.sweep(T, 3000)
        g.sweep(T, 500); g.reset_accumulators(); g.sweep(T, 6000)
        mo, so = blocked_mean_se(np.linalg.norm(o.trace()[:, 2:5], axis=1))
        mg, sg = blocked_mean_se(np.linalg.norm(g.trace(6000)[:, 2:5], axis=1))
        assert abs(mo - mg) < 3 * np.hypot(so, sg) + 2e-3, (T, mo, mg)
        assert lo < mg < hi, (T, mg)
        g.close()
