"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element, on seeded inputs.

The bar (BASELINE.json north_star; reading C-14): ONE colour pass from an identical fp32 state --
  * spins agree to 1e-4 max abs wherever the decisions agree;
  * accept/reject decisions may differ only where the oracle's |x| < 1e-5, x = dE/T + ln u2 (constrained: the
    log form of P:193);
and (measured, not required) the GPU's own fp32 x stays within a few 1e-6 of the oracle's.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

X_BAND = 1e-5       # decisions may differ only inside this band of the oracle's decision variable
SPIN_TOL = 1e-4     # max abs spin difference where decisions agree


@pytest.fixture(scope="module")
def mods():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    import oracle
    from paper_2103_03517_b200 import binding, build, inputs
    build.build()
    return oracle, binding, inputs


def _colour(shape):
    nx, ny, nz = shape
    s = np.arange(nx * ny * nz)
    return ((s % nx) + (s // nx) % ny + s // (nx * ny)) & 1


def _pair(mods, shape, seed=42, cone=0.5, sweep=0, path=None, **ham):
    oracle, binding, inputs = mods
    o = oracle.Oracle(*shape, seed=seed, cone0=cone, adaptive=False, **ham)
    g = binding.Lattice(*shape, seed=seed, cone0=cone, adaptive=False, **ham)
    if path is not None:
        g.debug_set_path(path)                              # documented test hook of include/mc.h (no environment variables)
    o.set_sweep(sweep); g.set_sweep(sweep)
    return o, g


def _check_half_sweep(o, g, T, colour, shape, allow_flips=True):
    """One colour pass on both sides from the GPU's current fp32 state.  Returns (n_flips, max |x_gpu - x_oracle|)."""
    before = g.get_spins()
    o.set_spins(before)                                  # identical state: the oracle takes the fp32 values
    n_o, x_o, acc_o = o.half_sweep(T, colour, want_detail=True)
    x_g, acc_g = g.half_sweep(T, colour, want_detail=True)
    after_g = g.get_spins().astype(np.float64); after_o = o.get_spins()
    col = _colour(shape)
    mine = col == colour
    # the other colour is untouched, bit for bit
    assert (after_g[~mine] == before[~mine].astype(np.float64)).all()
    # every site of this colour got a decision variable
    assert not np.isnan(x_g[mine]).any()
    differ = mine & (acc_g != acc_o)
    assert (np.abs(x_o[differ]) < X_BAND).all(), f"decision differs outside the band: {np.abs(x_o[differ]).max()}"
    if not allow_flips:
        assert differ.sum() == 0
    agree = mine & ~differ
    assert np.abs(after_g[agree] - after_o[agree]).max() < SPIN_TOL
    # accepted <=> changed, rejected <=> bit-identical
    changed = (after_g != before.astype(np.float64)).any(axis=1)
    assert (changed[mine] == (acc_g[mine] == 1)).all()
    # unit norm (pin P-4, GPU bound)
    assert np.abs(np.linalg.norm(after_g, axis=1) - 1).max() < 2e-7
    # accuracy of the GPU's own fp32 decision variable where it matters: near the decision boundary
    near = mine & (np.abs(x_o) < 2.0)
    return int(differ.sum()), float(np.abs(x_g[near] - x_o[near]).max()) if near.any() else 0.0


CASES = [
    # (shape, T, cone, ham kwargs)                                         what it covers
    ((16, 16, 16), 1.0, 0.5, dict(Ku=0.01)),                              # c1: VEC=4, one CTA row tiles
    ((24, 10, 6), 0.7, 1.2, dict(Kc=0.3, B=(0.1, -0.05, 0.2))),           # VEC=4, ragged rows (R=12), cubic + field
    ((40, 12, 10), 1.44, 2.0, dict(Kc=0.01)),                              # c3 parameters, several CTAs + tail
    ((6, 4, 4), 1.0, 0.8, dict(Ku=0.2, eu=(0.3, -0.5, 0.81))),            # VEC=1 path (nx % 8 != 0), tilted axis
    ((2, 2, 2), 3.0, np.pi, dict(Ku=0.1)),                                 # L = 2: every neighbour counted twice
    ((8, 6, 5), 0.9, 1.0, dict(periodic=(1, 0, 0), Ku=0.05, Kc=0.1)),      # open faces, odd open dims, both anisotropies
    ((2, 1, 1), 1.0, 1.5, dict(periodic=(0, 0, 0))),                       # the dimer
    ((64, 64, 64), 0.1, 0.3, dict(Ku=0.01)),                               # c2 first T-point (low T, random state = worst case)
    ((24, 8, 6), 0.8, 0.7, dict(periodic=(2, 1, 1), Ku=0.1)),              # anti-periodic x (domain-wall box), VEC=4
    ((6, 4, 4), 1.1, 1.0, dict(periodic=(2, 1, 0), Kc=0.2)),               # anti-periodic x, VEC=1 path, open z
    ((2, 2, 2), 2.0, 2.5, dict(periodic=(2, 1, 1), Ku=0.1)),               # L = 2 with an anti-periodic wrap: the x-bonds cancel
    ((96, 40, 36), 1.2, 0.9, dict(Kc=0.2, Ku=0.1, eu=(0.5, 0.5, 0.7), B=(0.05, 0.1, -0.2))),   # tiled pass, run-time row length (R = 48), two slabs, ragged z-segments, every term
    ((96, 40, 36), 0.9, 0.8, dict(periodic=(2, 1, 1), Ku=0.1, Kc=0.05)),     # tiled pass with the anti-periodic x wrap (ANTI instantiation)
    ((80, 30, 58), 0.6, 0.4, dict(Ku=0.05)),                               # tiled pass, one slab = all of y (halo wraps on both sides), R = 40
]


# lattices on which the tiled pass is not the default (no compile-time row length, or anti-periodic) but must stay correct
TILED_CASES = [c for c in CASES if c[0] in ((96, 40, 36), (80, 30, 58))]


@pytest.mark.parametrize("shape,T,cone,ham", TILED_CASES)
def test_half_sweep_parity_forced_staged_pass(mods, shape, T, cone, ham):
    test_half_sweep_parity_random_state(mods, shape, T, cone, ham, path=2)      # MC_PATH_STAGED


@pytest.mark.parametrize("shape,T,cone,ham", [c for c in CASES if c[0] == (64, 64, 64)] + TILED_CASES)
def test_half_sweep_parity_forced_generic_pass(mods, shape, T, cone, ham):
    test_half_sweep_parity_random_state(mods, shape, T, cone, ham, path=1)      # MC_PATH_GENERIC


# the register-carried march (MC_PATH_MARCH = 3): bulk z-march, ragged segments, masked / open faces, and the thin-film y-march
MARCH_CASES = [
    ((40, 12, 18), 1.44, 2.0, dict(Kc=0.01)),                                                # z-march, 4 segments + remainder
    ((24, 10, 16), 0.7, 1.2, dict(Kc=0.3, Ku=0.1, eu=(0.5, 0.5, 0.7), B=(0.1, -0.05, 0.2))),  # every term
    ((64, 64, 64), 0.1, 0.3, dict(Ku=0.01)),                                                 # low T
    ((16, 6, 17), 0.9, 1.0, dict(periodic=(1, 0, 0), Ku=0.05, Kc=0.1)),                      # masked: open y and z faces, odd nz
    ((512, 24, 4), 0.8, 0.9, dict(periodic=(1, 1, 0), Ku=0.1)),                              # thin film: y-march (a block = 64 items x 4 planes), open z
    ((256, 9, 8), 1.0, 1.2, dict(periodic=(0, 0, 1), Kc=0.2)),                               # y-march with open x and y, periodic z, odd ny
]


@pytest.mark.parametrize("shape,T,cone,ham", MARCH_CASES)
def test_half_sweep_parity_forced_march_pass(mods, shape, T, cone, ham):
    test_half_sweep_parity_random_state(mods, shape, T, cone, ham, path=3)      # MC_PATH_MARCH


def test_march_pass_is_bit_identical_to_the_generic_pass(mods):
    """Same packed arithmetic in the same order: after sweeps on both paths the spins are equal bit for bit (the fused sums are
    not: their fp32 partial sums group the sites differently before the exact fixed-point reduction)."""
    oracle, binding, inputs = mods
    cases = [((64, 48, 40), dict(Kc=0.05, Ku=0.02)), ((32, 16, 24), dict(periodic=(1, 0, 1), Ku=0.1)), ((512, 16, 4), dict(periodic=(1, 1, 0), Ku=0.1))]
    mask, region, axes = inputs.voronoi_film(512, 16, 4, mean_diameter=12, seed=3)
    cases.append(((512, 16, 4), dict(periodic=(1, 1, 0), Ku=0.02, bond_mask=mask, region=region, region_axis=axes)))
    for shape, ham in cases:
        out = []
        for path in (1, 3):
            g = binding.Lattice(*shape, cone0=0.8, adaptive=True, seed=11, **ham)
            g.debug_set_path(path)
            g.set_spins(inputs.random_unit_spins(g.N, seed=2)); g.sweep(0.9, 7)
            out.append((g.get_spins(), g.trace()[:, :2])); g.close()
        assert (out[0][0] == out[1][0]).all() and (out[0][1] == out[1][1]).all(), shape      # spins; acceptance and cone per sweep


@pytest.mark.parametrize("shape,T,cone,ham", CASES)
def test_half_sweep_parity_random_state(mods, shape, T, cone, ham, path=None):
    oracle, binding, inputs = mods
    o, g = _pair(mods, shape, cone=cone, sweep=(3 << 32) | 12345, path=path, **ham)
    g.set_spins(inputs.random_unit_spins(g.N, seed=7))
    worst = 0.0; flips = 0
    for colour in (0, 1, 0, 1):
        f, dx = _check_half_sweep(o, g, T, colour, shape)
        flips += f; worst = max(worst, dx)
    print(f"\n{shape} T={T}: decision flips {flips}, max |x_gpu - x_oracle| = {worst:.2e}")
    assert worst < X_BAND      # |x_gpu - x_oracle| over the sites with |x_oracle| < 2 (where a decision can flip)
    g.close()


def test_half_sweep_parity_masked_and_grain_axes(mods):
    """config c5 at reduced size: Voronoi film, J = 0 across grain boundaries, per-grain easy axes, open top/bottom."""
    oracle, binding, inputs = mods
    shape = (64, 48, 4)
    mask, region, axes = inputs.voronoi_film(*shape, mean_diameter=12, seed=3)
    ham = dict(periodic=(1, 1, 0), Ku=0.02, bond_mask=mask, region=region, region_axis=axes)
    for T, cone, state in ((0.1, 0.25, "ordered"), (1.0, 1.0, "random")):
        o, g = _pair(mods, shape, cone=cone, sweep=99, **ham)
        g.set_spins(inputs.thermal_like_spins(g.N, 5, 0.15) if state == "ordered" else inputs.random_unit_spins(g.N, 5))
        for colour in (0, 1):
            f, dx = _check_half_sweep(o, g, T, colour, shape)
            print(f"\nfilm {state} T={T} colour {colour}: flips {f}, max dx {dx:.2e}")
        g.close()
    # random symmetric dilution on a periodic lattice, scalar path
    shape = (6, 6, 4)
    m2 = inputs.random_bond_mask(*shape, (1, 1, 1), seed=4, p_cut=0.3)
    o, g = _pair(mods, shape, cone=1.0, Ku=0.1, bond_mask=m2)
    g.set_spins(inputs.random_unit_spins(g.N, 6))
    for colour in (0, 1):
        _check_half_sweep(o, g, 0.8, colour, shape)
    g.close()


@pytest.mark.parametrize("T,spread,cone", [(0.1, 0.15, 0.25), (0.02, 0.06, 0.1), (0.5, 0.4, 0.6)])
def test_low_temperature_decision_accuracy(mods, T, spread, cone):
    """the fp32 decision variable must stay inside the 1e-5 band at low T on thermal-looking states."""
    oracle, binding, inputs = mods
    shape = (32, 32, 32)
    o, g = _pair(mods, shape, cone=cone, sweep=5, Ku=0.01)
    g.set_spins(inputs.thermal_like_spins(g.N, seed=11, spread=spread))
    worst = 0.0
    for colour in (0, 1):
        f, dx = _check_half_sweep(o, g, T, colour, shape)
        worst = max(worst, dx)
    print(f"\nT={T}: max |x_gpu - x_oracle| = {worst:.2e}")
    # T >= 0.1 is BASELINE's range: the GPU's fp32 x itself must stay inside the band.  T = 0.02 is outside it; there the
    # fp32 resolution of dE/T (~1e-7 |h||d| / T) is the limit and only the decision rule (checked above) is required.
    assert worst < (X_BAND if T >= 0.1 else 3e-5)
    g.close()


def test_sweep_equals_hooks_and_is_deterministic(mods):
    oracle, binding, inputs = mods
    shape = (24, 16, 8)
    s0 = inputs.random_unit_spins(24 * 16 * 8, seed=1)
    def run(kind):
        g = binding.Lattice(*shape, Ku=0.01, cone0=0.5, adaptive=True, seed=42)
        g.set_spins(s0)
        if kind == "one":
            g.sweep(1.0, 12)
        elif kind == "split":
            for n in (1, 5, 6): g.sweep(1.0, n)
        else:
            for _ in range(12):
                g.half_sweep(1.0, 0); g.half_sweep(1.0, 1); g.end_sweep()
        out = g.get_spins(), g.trace(), g.observables()
        g.close()
        return out
    a, ta, oa = run("one"); b, tb, ob = run("split"); c, tc, oc = run("hooks"); d, td, od = run("one")
    assert (a == b).all() and (a == c).all() and (a == d).all()          # P-20: bit-identical spins
    assert (ta == tb).all() and (ta == tc).all() and (ta == td).all()    # bitwise reproducible reductions
    assert oa.sweep == 12 and len(ta) == 12
    assert np.allclose(np.abs(np.diff(ta[:, 1])), np.pi / 180, atol=1e-14)   # controller: exact 1 degree steps (P-19)


def test_observables_match_oracle(mods):
    oracle, binding, inputs = mods
    shape = (16, 12, 6)
    mask = inputs.boundary_mask(*shape, (1, 1, 0))
    kw = dict(periodic=(1, 1, 0), J=0.8, Ku=0.3, eu=(0.2, 0.1, 0.9), Kc=0.4, B=(0.1, 0.2, -0.3))
    o, g = _pair(mods, shape, **kw)
    s = inputs.random_unit_spins(g.N, 3)
    g.set_spins(s); o.set_spins(g.get_spins())
    a, b = g.observables(), o.observables()
    for name in ("m", "E_total", "E_exch", "E_aniso", "E_zeeman"):
        assert abs(getattr(a, name) - getattr(b, name)) < 2e-6, name
    assert np.allclose(list(a.M), list(b.M), atol=1e-6) and np.allclose(list(a.torque), list(b.torque), atol=1e-6)
    # fused per-sweep values (trace) agree with a fresh measurement of the post-sweep state
    g.sweep(0.9, 3)
    tr = g.trace(); ob = g.observables()
    assert np.allclose(tr[-1, 2:5], list(ob.M), atol=1e-6) and abs(tr[-1, 5] - ob.E_total) < 2e-6
    assert ob.n_samples == 3 and abs(ob.sum_E - tr[:, 5].sum()) < 1e-12
    g.close()


@pytest.mark.parametrize("shape", [(64, 64, 64), (128, 32, 32), (192, 32, 24)])
def test_compile_time_row_length_instantiations_match_the_checked_one(mods, shape):
    """R = 32, 64, 96 (R = 112: the 224^3 test): the instantiation mc_sweep launches writes no decision variable, so it is
    compared bit for bit with the run-time-row-length instantiation that does and that the oracle parity cases go through."""
    oracle, binding, inputs = mods
    s0 = inputs.random_unit_spins(shape[0] * shape[1] * shape[2], seed=21)
    g = binding.Lattice(*shape, Ku=0.02, Kc=0.1, B=(0.05, 0.0, -0.1), cone0=0.8, adaptive=False, seed=3)
    out = []
    for detail in (False, True):
        g.set_spins(s0); g.set_sweep(41)
        for colour in (0, 1):
            g.half_sweep(0.9, colour, want_detail=detail)
        out.append(g.get_spins())
    assert (out[0] == out[1]).all() and not (out[0] == s0).all()
    o = oracle.Oracle(*shape, Ku=0.02, Kc=0.1, B=(0.05, 0.0, -0.1), cone0=0.8, adaptive=False, seed=3)
    g.set_spins(s0); g.set_sweep(41); o.set_sweep(41); o.set_spins(g.get_spins())
    _, x_o, _ = o.half_sweep(0.9, 0, want_detail=True)
    g.half_sweep(0.9, 0)
    bad = np.abs(g.get_spins().astype(np.float64) - o.get_spins()).max(axis=1) >= SPIN_TOL
    assert (np.abs(x_o[bad]) < X_BAND).all()
    g.close()


def test_tiled_pass_fused_sums_match_a_fresh_measurement(mods):
    """The tiled pass forms the on-site energies of the final spin from the dE terms (s4 identity, (S.e)^2 difference form)
    and sums in 64-bit fixed point: its per-sweep M and E must equal a standalone measurement of the same state, and the
    oracle's energy of that state."""
    oracle, binding, inputs = mods
    shape = (64, 64, 64)
    kw = dict(J=0.9, Ku=0.3, eu=(0.2, 0.1, 0.9), Kc=0.4, B=(0.1, 0.2, -0.3))
    g = binding.Lattice(*shape, seed=5, cone0=0.7, adaptive=True, **kw)
    g.set_spins(inputs.random_unit_spins(g.N, 11))
    g.sweep(0.8, 4)
    tr = g.trace()
    fused = g.observables()                                   # what the black pass left
    g.set_spins(g.get_spins())                                # invalidates the fused sums: the next call measures afresh
    fresh = g.observables()
    o = oracle.Oracle(*shape, seed=5, **kw); o.set_spins(g.get_spins()); ref = o.observables()
    for name in ("m", "E_total", "E_exch", "E_aniso", "E_zeeman"):
        assert abs(getattr(fused, name) - getattr(fresh, name)) < 2e-6, name
        assert abs(getattr(fresh, name) - getattr(ref, name)) < 2e-6, name
    assert np.allclose(tr[-1, 2:5], list(fresh.M), atol=1e-6) and abs(tr[-1, 5] - fresh.E_total) < 2e-6
    g.close()


def test_domain_wall_box_profile_and_energy_match_oracle(mods):
    """anti-periodic x + slice profile.  A tanh wall (Eq. 5) with thermal scatter: mc_profile_x against the
    oracle's slice average, the exchange energy (wrap bonds counted with -S_j) against the oracle's, then whole sweeps
    keep the wall in the box (m_z changes sign once along x and the total M_z stays near 0)."""
    oracle, binding, inputs = mods
    shape = (48, 16, 12)
    kw = dict(periodic=(2, 1, 1), J=1.0, Ku=0.05)
    o, g = _pair(mods, shape, **kw)
    nx, ny, nz = shape
    x = np.arange(nx * ny * nz) % nx
    rng = np.random.default_rng(4)
    S = np.zeros((nx * ny * nz, 3)); S[:, 2] = np.tanh(-(x - 23.5) / np.sqrt(1.0 / (2 * 0.05))); S[:, 1] = np.sqrt(1 - S[:, 2] ** 2)
    S += 0.15 * rng.standard_normal(S.shape); S /= np.linalg.norm(S, axis=1, keepdims=True)
    g.set_spins(S.astype(np.float32)); o.set_spins(g.get_spins())
    pg, po = g.profile_x(), o.profile_x()
    assert pg.shape == (nx, 3) and np.abs(pg - po).max() < 1e-6
    a, b = g.observables(), o.observables()
    for name in ("E_total", "E_exch", "E_aniso", "m"):
        assert abs(getattr(a, name) - getattr(b, name)) < 2e-6, name
    assert (g.profile_x() == pg).all()                       # exact fixed-point sums: bitwise reproducible
    for colour in (0, 1):
        _check_half_sweep(o, g, 0.5, colour, shape)
    g2 = binding.Lattice(*shape, seed=9, cone0=0.4, adaptive=True, **kw)
    g2.set_spins(g.get_spins()); g2.sweep(0.4, 300)
    mz = g2.profile_x()[:, 2]
    assert mz[:8].mean() > 0.8 and mz[-8:].mean() < -0.8 and (np.diff(np.sign(mz)) != 0).sum() == 1
    g.close(); g2.close()


def test_set_get_roundtrip_and_init(mods):
    oracle, binding, inputs = mods
    g = binding.Lattice(8, 6, 4, periodic=(1, 1, 1))
    s = inputs.random_unit_spins(g.N, 9)
    g.set_spins(s)
    assert np.abs(g.get_spins() - s).max() < 1.2e-7
    g.init_spins(1, (1, 1, 0))
    assert np.allclose(g.get_spins(), np.array([1, 1, 0]) / np.sqrt(2), atol=1e-7)
    assert abs(g.observables().m - 1) < 1e-6
    g.close()


def test_random_start_matches_oracle(mods):
    oracle, binding, inputs = mods
    for shape in ((24, 20, 16), (6, 4, 4)):
        g = binding.Lattice(*shape, seed=11); g.init_spins(2)
        o = oracle.Oracle(*shape, seed=11); o.init_random()
        assert np.abs(g.get_spins() - o.get_spins()).max() < 2e-6
        g.close()


def test_error_paths(mods):
    oracle, binding, inputs = mods
    g = binding.Lattice(8, 4, 4)
    with pytest.raises(binding.McError): g.sweep(0.0, 1)                 # C-16
    with pytest.raises(binding.McError): g.sweep(-1.0, 1)
    with pytest.raises(binding.McError): g.set_cone(0.0)
    g.set_spins(inputs.random_unit_spins(g.N, 1) * np.array([1, 1, 0], np.float32) + np.array([0, 0, 1e-9], np.float32))
    bad = binding.Lattice(6, 3, 1, periodic=(1, 0, 0))                   # 9 sites per colour: odd (C-15)
    with pytest.raises(binding.McError): bad.constrained_sweep(1.0, 0.0, 0.0, 1)
    m = inputs.boundary_mask(8, 4, 4, (1, 1, 1)); m[0] &= 0xFE            # asymmetric mask
    with pytest.raises(binding.McError): binding.Lattice(8, 4, 4, bond_mask=m)
    with pytest.raises(binding.McError): binding.Lattice(8, 4, 4, periodic=(1, 2, 1))     # anti-periodic along x only
    g.close(); bad.close()


# ------------------------------------------------------------------------------------------ constrained path
CCASES = [
    ((16, 16, 16), 0.8, 0.6, dict(Ku=0.05)),            # VEC=4, B=32
    ((8, 8, 8), 1.0, 1.0, dict(Ku=0.05, Kc=0.02)),      # VEC=4, B=32, H=8
    ((12, 4, 2), 0.9, 0.9, dict(Ku=0.1)),               # VEC=1, B=8
    ((6, 6, 2), 0.9, 0.9, dict()),                      # VEC=1, B=2
    ((32, 16, 8), 0.3, 0.3, dict(Ku=0.05)),             # lower T
    ((16, 8, 8), 0.7, 0.6, dict(periodic=(2, 1, 1), Ku=0.1)),              # pair pass in the domain-wall box (anti-periodic x)
]


@pytest.mark.parametrize("shape,T,cone,ham", CCASES)
def test_constrained_half_sweep_parity(mods, shape, T, cone, ham):
    oracle, binding, inputs = mods
    theta, phi = 0.7, 0.4
    e = np.array([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)])
    o, g = _pair(mods, shape, cone=cone, sweep=77, **ham)
    g.set_spins(inputs.thermal_like_spins(g.N, seed=2, spread=0.5, direction=e))
    col = _colour(shape)
    worst = 0.0
    for colour in (0, 1):
        before = g.get_spins()
        o.set_spins(before)
        ML = float((before.astype(np.float64) @ e).sum())
        n_o, ml_o, x_o, acc_o = o.constrained_half_sweep(T, e, colour, ML, want_detail=True)
        x_g, acc_g = g.constrained_half_sweep(T, theta, phi, colour, ML, want_detail=True)
        after_g = g.get_spins().astype(np.float64); after_o = o.get_spins()
        mine = col == colour
        assert (after_g[~mine] == before[~mine].astype(np.float64)).all()
        # same pairing: leaders are exactly the sites that carry a decision variable
        partner, lead = o.pairing(77, colour)
        lead_sites = np.array([o.site_of(colour, a) for a in np.nonzero(lead)[0]])
        foll_sites = np.array([o.site_of(colour, partner[a]) for a in np.nonzero(lead)[0]])
        assert not np.isnan(x_g[lead_sites]).any() and np.isnan(x_g[foll_sites]).all()
        assert (acc_g[lead_sites] == acc_g[foll_sites]).all()
        differ = acc_g[lead_sites] != acc_o[lead_sites]
        xo = x_o[lead_sites]
        assert (np.abs(xo[differ]) < X_BAND).all(), np.abs(xo[differ]).max()
        ok_pairs = ~differ
        for sites in (lead_sites[ok_pairs], foll_sites[ok_pairs]):
            assert np.abs(after_g[sites] - after_o[sites]).max() < SPIN_TOL
        fin = np.isfinite(xo) & np.isfinite(x_g[lead_sites])
        assert (np.isfinite(xo) == np.isfinite(x_g[lead_sites])).mean() > 0.999
        worst = max(worst, float(np.abs(x_g[lead_sites][fin] - xo[fin]).max()))
        assert np.abs(np.linalg.norm(after_g, axis=1) - 1).max() < 3e-7
        # transverse magnetisation is conserved by every accepted pair (P-16, fp32)
        Mb = before.astype(np.float64).sum(axis=0); Ma = after_g.sum(axis=0)
        perp = (Ma - Mb) - ((Ma - Mb) @ e) * e
        assert np.abs(perp).max() < 1e-6 * np.sqrt(g.N) + 1e-5
    print(f"\nconstrained {shape} T={T}: max |x_gpu - x_oracle| = {worst:.2e}")
    g.close()


def test_align_rotation_matches_oracle(mods):
    oracle, binding, inputs = mods
    shape = (16, 8, 8)
    o, g = _pair(mods, shape, Ku=0.05)
    s = inputs.thermal_like_spins(g.N, seed=4, spread=0.6, direction=(0.3, -0.2, 0.9))
    g.set_spins(s); o.set_spins(g.get_spins())
    theta, phi = 1.1, -0.7
    e = np.array([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)])
    g.align_to(theta, phi); assert o.align_to(e) == 0
    assert np.abs(g.get_spins() - o.get_spins()).max() < 1e-6
    ob = g.observables()
    assert np.allclose(np.array(ob.M) / ob.m, e, atol=1e-6)
    g.close()


# ------------------------------------------------------------------------------------------ whole constrained sweeps (a-10)
def test_constrained_sweep_equals_hooks_and_fused_ML_is_exact(mods):
    """Constrained twin of test_sweep_equals_hooks_and_is_deterministic.  mc_constrained_sweep(T, theta, phi, 3) takes M_L of
    every sweep from the fused fixed-point sums of the previous one (SURVEY a-10); the hook-assembled twin is handed
    M_L = the fp64 sum of S_i.e_C of the same state (computed here with NumPy from mc_get_spins).
      * the fused M (hence M_L = N M.e_C) of every sweep, read from the trace, equals the fp64 value of the post-sweep state
        to 2e-7 per site -- an O(1/N) slip (one spin dropped or counted twice: 2.4e-4 per site here) fails;
      * the two runs end in bit-identical spins (16^3: a decision inside the ~1e-7 band that the last-bit difference of the
        two M_L values opens has probability ~1e-3 over the 6144 pair decisions; the seeds are fixed, so the outcome is too);
      * acceptance and cone trace agree exactly."""
    oracle, binding, inputs = mods
    shape, T, theta, phi = (16, 16, 16), 0.8, 0.7, 0.4
    N = 16 ** 3
    e = np.array([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)])
    s0 = inputs.thermal_like_spins(N, seed=2, spread=0.5, direction=e)
    a = binding.Lattice(*shape, Ku=0.05, cone0=0.6, adaptive=True, seed=42); a.set_spins(s0)
    b = binding.Lattice(*shape, Ku=0.05, cone0=0.6, adaptive=True, seed=42); b.set_spins(s0)
    a.align_to(theta, phi); b.align_to(theta, phi)
    assert (a.get_spins() == b.get_spins()).all()
    states = []
    for k in range(3):
        a.constrained_sweep(T, theta, phi, 1)
        states.append(a.get_spins())
    tr = a.trace()
    assert len(tr) == 3
    for k in range(3):
        M64 = states[k].astype(np.float64).sum(axis=0) / N
        assert np.abs(tr[k, 2:5] - M64).max() < 2e-7, (k, tr[k, 2:5], M64)
    for k in range(3):
        cur = b.get_spins().astype(np.float64)
        ML = float((cur @ e).sum())
        b.constrained_half_sweep(T, theta, phi, 0, ML)
        b.constrained_half_sweep(T, theta, phi, 1, ML)                    # stale M_L: the same value for both colours
        b.end_sweep()
        assert (b.get_spins() == states[k]).all(), k
    tb = b.trace()
    assert (tb[:, :2] == tr[:, :2]).all() and np.abs(tb[:, 2:] - tr[:, 2:]).max() < 1e-9
    # one call of 3 sweeps = three calls of 1 sweep, bitwise (P-20 for the constrained path)
    c = binding.Lattice(*shape, Ku=0.05, cone0=0.6, adaptive=True, seed=42); c.set_spins(s0)
    c.constrained_sweep(T, theta, phi, 3)
    assert (c.get_spins() == states[2]).all() and (c.trace() == tr).all()
    a.close(); b.close(); c.close()


def test_unconstrained_sweeps_invalidate_the_alignment_on_the_gpu(mods):
    """constrained -> mc_sweep -> constrained with the same (theta, phi): the library re-aligns (C-12), as the oracle does
    (tests/test_oracle_align.py).  Without the re-alignment M stays tilted: the pair move conserves its transverse part."""
    oracle, binding, inputs = mods
    shape, T, theta, phi = (16, 16, 16), 1.0, 0.6, 0.3
    e = np.array([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)])
    g = binding.Lattice(*shape, Ku=0.05, cone0=0.6, adaptive=True, seed=5)
    g.constrained_sweep(T, theta, phi, 20)
    ob = g.observables(); assert np.abs(np.array(ob.M) / ob.m - e).max() < 2e-6
    g.sweep(T, 40)
    ob = g.observables(); assert np.abs(np.array(ob.M) / ob.m - e).max() > 1e-3
    g.constrained_sweep(T, theta, phi, 5)
    ob = g.observables(); assert np.abs(np.array(ob.M) / ob.m - e).max() < 2e-6
    g.half_sweep(T, 0); g.half_sweep(T, 1); g.end_sweep()                 # the hooks invalidate it as well
    g.constrained_sweep(T, theta, phi, 1)
    ob = g.observables(); assert np.abs(np.array(ob.M) / ob.m - e).max() < 2e-6
    g.close()


def test_a_hook_without_end_sweep_does_not_leak_into_the_next_sweep(mods):
    """include/mc.h: a half-sweep hook leaves its count and fused sums pending; mc_sweep discards them."""
    oracle, binding, inputs = mods
    shape = (16, 16, 16)
    s0 = inputs.random_unit_spins(16 ** 3, seed=3)
    a = binding.Lattice(*shape, Ku=0.01, cone0=2.5, adaptive=True, seed=7); a.set_spins(s0)
    a.half_sweep(3.0, 0)                                                  # never closed: ~4096 * 0.5 * 0.9 accepted moves pending
    snap = a.get_spins()
    a.set_spins(snap)                                                     # the upload renormalises: both handles take the same one
    b = binding.Lattice(*shape, Ku=0.01, cone0=2.5, adaptive=True, seed=7); b.set_spins(snap)            # a clean handle, same spins
    a.sweep(3.0, 2); b.sweep(3.0, 2)
    ta, tb = a.trace(), b.trace()
    assert (a.get_spins() == b.get_spins()).all()
    assert (ta == tb).all() and (ta[:, 0] <= 1.0).all()                   # acceptance, cone, M, E: nothing of the hook's pass is left
    ob = a.observables()
    assert np.abs(ta[-1, 2:5] - np.array(ob.M)).max() < 1e-6              # the fused M of the last sweep holds one sweep only
    a.close(); b.close()


def test_negative_zero_sz_takes_the_sign_bit_frame_on_every_path(mods):
    """Reading C-29: sigma of the Duff frame is the sign bit of S_z.  Spins with S_z = -0.0 (and +0.0) on the scalar path
    (VEC = 1), the packed generic path (VEC = 4) and the staged pass propose the oracle's trial spins."""
    oracle, binding, inputs = mods
    for shape, path in (((6, 4, 4), None), ((16, 16, 16), None), ((96, 40, 36), 2)):
        N = shape[0] * shape[1] * shape[2]
        s = inputs.random_unit_spins(N, seed=12)
        s[0::3, 2] = -0.0; s[1::3, 2] = 0.0
        s /= np.linalg.norm(s.astype(np.float64), axis=1, keepdims=True).astype(np.float32)
        assert np.signbit(s[0::3, 2]).all() and not np.signbit(s[1::3, 2]).any()
        o, g = _pair(mods, shape, cone=1.0, sweep=5, path=path, Ku=0.05)
        g.set_spins(s)
        got = g.get_spins()
        assert np.signbit(got[0::3, 2]).all()                            # the upload keeps the sign bit
        for colour in (0, 1):
            _check_half_sweep(o, g, 1.0, colour, shape)
        g.close()


def test_no_kernel_writes_outside_the_workspace(mods):
    """Canary zones of 1 MiB on both sides of the caller's workspace stay intact through every kernel of the library, on
    lattices whose sizes are not multiples of any tile (the last plane / row / item is where an index error would land):
    colour passes (generic, staged, masked, bcc), pair passes, upload / readback, hooks, measurement, rotation, profile."""
    oracle, binding, inputs = mods
    G = 1 << 20
    runs = [dict(shape=(16, 16, 16), ham=dict(Ku=0.01)), dict(shape=(2, 2, 2), ham=dict(Ku=0.1)), dict(shape=(6, 4, 4), ham=dict(Kc=0.2)),
            dict(shape=(2, 1, 1), ham=dict(periodic=(0, 0, 0))), dict(shape=(8, 6, 5), ham=dict(periodic=(1, 0, 0), Ku=0.05)),
            dict(shape=(64, 64, 64), ham=dict(Kc=0.01)), dict(shape=(96, 40, 36), ham=dict(Ku=0.1), path=2),
            dict(shape=(80, 30, 58), ham=dict(periodic=(2, 1, 1), Ku=0.05), path=2),
            dict(shape=(12, 5, 7), ham=dict(Ku=0.2, structure="bcc")), dict(shape=(4, 1, 1), ham=dict(structure="bcc")),
            dict(shape=(12, 5, 7), ham=dict(Kc=0.1, structure="fcc")), dict(shape=(4, 1, 1), ham=dict(structure="fcc"))]
    for r in runs:
        g = binding.Lattice(*r["shape"], cone0=0.8, adaptive=True, seed=3, guard_bytes=G, **r["ham"])
        if "path" in r: g.debug_set_path(r["path"])
        g.set_spins(inputs.random_unit_spins(g.N, seed=1)); g.sweep(1.0, 3)
        g.half_sweep(1.0, 0, want_detail=True); g.half_sweep(1.0, 1); g.end_sweep()
        g.init_spins(0); g.sweep(0.5, 2)
        sc = r["ham"].get("structure", "sc") == "sc"
        if sc and (g.N // 2) % 2 == 0:
            try:
                g.constrained_sweep(0.5, 0.4, 0.2, 3)
            except binding.McError:
                pass                                            # lattices the pairing does not cover
        if sc: g.profile_x()
        g.observables(); g.get_spins(); g.trace()
        assert g.check_guards(), r
        g.close()
    shape = (64, 48, 4)                                         # the film: bond mask + grain table + open faces
    mask, region, axes = inputs.voronoi_film(*shape, mean_diameter=12, seed=3)
    g = binding.Lattice(*shape, periodic=(1, 1, 0), Ku=0.02, bond_mask=mask, region=region, region_axis=axes, guard_bytes=G)
    g.sweep(0.5, 3); g.observables()
    assert g.check_guards()
    g.close()


def test_checkpoint_restore_in_the_middle_of_a_run(mods):
    """a run interrupted after 7 of 15 sweeps and restored into a fresh handle from (spins, sweep counter, cone)
    continues bit for bit -- the RNG is counter-based, the upload of a downloaded state is the identity.  Unconstrained
    (staged, march and generic lattices) and constrained."""
    oracle, binding, inputs = mods
    for shape, ham, constrained in (((64, 64, 64), dict(Kc=0.01), False), ((64, 48, 40), dict(Ku=0.05), False),
                                    ((24, 10, 6), dict(Ku=0.1, B=(0.0, 0.1, 0.0)), False), ((32, 16, 16), dict(Ku=0.05), True)):
        step = (lambda g, n: g.constrained_sweep(0.8, 0.5, 0.2, n)) if constrained else (lambda g, n: g.sweep(1.1, n))
        a = binding.Lattice(*shape, cone0=0.7, adaptive=True, seed=9, **ham)
        if not constrained: a.set_spins(inputs.random_unit_spins(a.N, seed=4))
        step(a, 7)
        snap, ob = a.get_spins(), a.observables()
        step(a, 8)
        b = binding.Lattice(*shape, cone0=0.7, adaptive=True, seed=9, **ham)
        b.set_spins(snap); b.set_sweep(ob.sweep); b.set_cone(ob.cone_rad)
        assert (b.get_spins() == snap).all()                                # the upload changed nothing
        step(b, 8)                                                          # constrained: M already lies along e_C, the library does not rotate
        assert (a.get_spins() == b.get_spins()).all(), shape
        assert (a.trace()[-8:] == b.trace()).all()
        a.close(); b.close()
