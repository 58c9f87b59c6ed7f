"""GPU parity for the bcc lattice (reading C-30): the CUDA pass against the oracle's bcc mode, element by
element through the C ABI, with the same bar as the sc lattice (C-14): decisions may differ only where the oracle's
|x| < 1e-5, spins agree to 1e-4 where the decisions agree."""
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


def _pair(mods, shape, seed=42, cone=0.5, sweep=0, adaptive=False, path=None, **ham):
    oracle, binding, inputs = mods
    o = oracle.Oracle(*shape, seed=seed, cone0=cone, adaptive=adaptive, structure="bcc", **ham)
    g = binding.Lattice(*shape, seed=seed, cone0=cone, adaptive=adaptive, structure="bcc", **ham)
    if path is not None:
        g.debug_set_path(path)
    o.set_sweep(sweep); g.set_sweep(sweep)
    return o, g


def _half(o, g, T, colour):
    before = g.get_spins()
    o.set_spins(before)
    n_o, x_o, acc_o = o.half_sweep(T, colour, want_detail=True)
    x_g, acc_g = g.half_sweep(T, colour, want_detail=True)
    after_g = g.get_spins().astype(np.float64); after_o = o.get_spins()
    nc = g.N // 2
    mine = (np.arange(g.N) >= nc) == bool(colour)            # colour = sublattice, stored contiguously
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
    ((16, 16, 16), 2.0, 0.8, dict(Ku=0.05)),                                                  # near T_C of the bcc lattice
    ((4, 1, 1), 1.0, 1.5, dict()),                                                            # one-cell-thick: neighbours counted 4 times
    ((8, 2, 2), 3.0, np.pi, dict(Kc=0.2)),                                                    # 2-cell periodic dims: each neighbour twice
    ((12, 5, 7), 0.9, 1.0, dict(Ku=0.2, eu=(0.3, -0.5, 0.81), Kc=0.1, B=(0.1, -0.05, 0.2))),  # odd dims, ragged grid, every term
    ((64, 40, 24), 0.3, 0.4, dict(Ku=0.01)),                                                  # several CTAs per SM, low T
]


MARCH_CASES = [
    ((16, 16, 16), 2.0, 0.8, dict(Ku=0.05)),
    ((12, 5, 9), 0.9, 1.0, dict(Ku=0.2, eu=(0.3, -0.5, 0.81), Kc=0.1, B=(0.1, -0.05, 0.2))),  # odd ny and nz, two segments + remainder
    ((64, 40, 24), 0.3, 0.4, dict(Ku=0.01)),
    ((8, 2, 8), 3.0, np.pi, dict(Kc=0.2)),                                                    # 2-cell periodic y: the two rows of a plane coincide
]


@pytest.mark.parametrize("shape,T,cone,ham", MARCH_CASES)
def test_bcc_half_sweep_parity_forced_march_pass(mods, shape, T, cone, ham):
    test_bcc_half_sweep_parity(mods, shape, T, cone, ham, path=3)                               # MC_PATH_MARCH


def test_bcc_march_pass_is_bit_identical_to_the_generic_pass(mods):
    oracle, binding, inputs = mods
    for shape, ham in (((32, 24, 20), dict(Ku=0.05, Kc=0.02)), ((16, 7, 11), dict(B=(0.0, 0.1, 0.2)))):
        out = []
        for path in (1, 3):
            g = binding.Lattice(*shape, cone0=0.8, adaptive=True, seed=11, structure="bcc", **ham)
            g.debug_set_path(path)
            g.set_spins(inputs.random_unit_spins(g.N, seed=2)); g.sweep(1.7, 7)
            out.append((g.get_spins(), g.trace()[:, :2])); g.close()
        assert (out[0][0] == out[1][0]).all() and (out[0][1] == out[1][1]).all(), shape


@pytest.mark.parametrize("shape,T,cone,ham", CASES)
def test_bcc_half_sweep_parity(mods, shape, T, cone, ham, path=None):
    oracle, binding, inputs = mods
    o, g = _pair(mods, shape, cone=cone, sweep=(5 << 32) | 777, path=path, **ham)
    g.set_spins(inputs.random_unit_spins(g.N, seed=8))
    worst = 0.0
    for colour in (0, 1, 0, 1):
        f, dx = _half(o, g, T, colour)
        worst = max(worst, dx)
    assert worst < X_BAND
    g.set_spins(inputs.thermal_like_spins(g.N, 9, 0.2))                                        # an ordered state: the low-T regime of dE
    for colour in (0, 1):
        f, dx = _half(o, g, T, colour)
        assert dx < X_BAND
    g.close()


def test_bcc_observables_and_ground_state(mods):
    oracle, binding, inputs = mods
    shape = (12, 6, 10)
    o, g = _pair(mods, shape, Ku=0.1, eu=(1, 1, 0), Kc=0.05, B=(0.02, 0.0, -0.03))
    ob = g.observables()
    assert abs(ob.E_exch + 4.0) < 1e-6 and abs(ob.m - 1) < 1e-6                                # +z start: 4 bonds per spin
    s = inputs.random_unit_spins(g.N, seed=4); g.set_spins(s); o.set_spins(g.get_spins())
    a, b = g.observables(), o.observables()
    for name in ("m", "E_total", "E_exch", "E_aniso", "E_zeeman"):
        assert abs(getattr(a, name) - getattr(b, name)) < 2e-6, name
    assert np.abs(np.array(a.M) - np.array(b.M)).max() < 2e-6
    assert np.abs(np.array(a.torque) - np.array(b.torque)).max() < 2e-6
    g.close()
    odd = binding.Lattice(4, 3, 1, structure="bcc")                                            # 12 cells: not a multiple of 8
    with pytest.raises(binding.McError):
        odd.constrained_sweep(1.0, 0.3, 0.0, 1)
    odd.close()


def test_bcc_sweep_equals_hooks_and_controller(mods):
    """mc_sweep(T, n) = n x (hook colour 0, hook colour 1, end_sweep), bit for bit; the fused sums of the last sweep equal a
    fresh measurement; the cone follows the +-1 degree controller of the oracle while decisions agree."""
    oracle, binding, inputs = mods
    shape, T = (16, 8, 8), 1.5
    s0 = inputs.random_unit_spins(2 * 16 * 8 * 8, seed=5)
    o, a = _pair(mods, shape, cone=0.5, adaptive=True, Ku=0.05); a.set_spins(s0)
    o2, b = _pair(mods, shape, cone=0.5, adaptive=True, Ku=0.05); b.set_spins(s0)
    a.sweep(T, 6)
    for _ in range(6):
        b.half_sweep(T, 0); b.half_sweep(T, 1); b.end_sweep()
    assert (a.get_spins() == b.get_spins()).all() and (a.trace() == b.trace()).all()
    ob = a.observables(); tr = a.trace()
    assert np.abs(tr[-1, 2:5] - np.array(ob.M)).max() < 1e-6 and abs(tr[-1, 5] - ob.E_total) < 1e-5
    assert np.allclose(np.abs(np.diff(tr[:, 1])), np.pi / 180, atol=1e-12)
    a.close(); b.close()


def test_bcc_ensemble_matches_oracle_and_orders_below_tc(mods):
    """m(T) of an equilibrated run: GPU against the oracle within 3 standard errors at T = 1.6 (ordered: a simple cubic lattice is
    already disordered there, T_C = 1.44) and at T = 2.4 (above the bcc T_C = 2.054)."""
    from stats_util import blocked_mean_se
    oracle, binding, inputs = mods
    shape = (8, 8, 8)
    for T, lo, hi in ((1.6, 0.5, 0.8), (2.4, 0.0, 0.2)):
        o, g = _pair(mods, shape, seed=3, cone=1.0, adaptive=True, Ku=0.01)
        o.set_sampling(False); o.sweep(T, 500); o.set_sampling(True); o.sweep(T, 3000)
        g.sweep(T, 500); g.reset_accumulators(); g.sweep(T, 6000)
        mo, so = blocked_mean_se(np.linalg.norm(o.trace()[:, 2:5], axis=1))
        mg, sg = blocked_mean_se(np.linalg.norm(g.trace(6000)[:, 2:5], axis=1))
        assert abs(mo - mg) < 3 * np.hypot(so, sg) + 2e-3, (T, mo, mg)
        assert lo < mg < hi
        g.close()


# ------------------------------------------------------------------------------------------ constrained path (Table A2) on bcc
CCASES = [
    ((16, 16, 16), 1.2, 0.6, dict(Ku=0.05)),                                                  # B = 32, many chunks
    ((8, 2, 2), 1.0, 1.0, dict(Ku=0.05, Kc=0.02)),                                            # 32 cells: B = 16, H = 2; 2-cell periodic dims
    ((4, 2, 1), 0.9, 0.9, dict()),                                                            # 8 cells: B = 4, one leader group per colour
    ((12, 5, 8), 0.9, 0.9, dict(Ku=0.1, eu=(0.3, -0.5, 0.81), B=(0.05, 0.0, 0.1))),           # 480 cells: B = 16, odd ny
    ((64, 40, 24), 0.3, 0.3, dict(Ku=0.05)),                                                  # several CTAs per SM, low T
]


@pytest.mark.parametrize("shape,T,cone,ham", CCASES)
def test_bcc_constrained_half_sweep_parity(mods, shape, T, cone, ham):
    """Pair pass against the oracle's constrained bcc mode (same bar as the sc lattice): same pairing (leaders carry the decision
    variable, followers none), decisions differ only inside the band, both members agree to 1e-4, transverse M conserved."""
    oracle, binding, inputs = mods
    theta, phi = 0.7, 0.4
    e = np.array([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)])
    o, g = _pair(mods, shape, cone=cone, sweep=77, **ham)
    g.set_spins(inputs.thermal_like_spins(g.N, seed=2, spread=0.5, direction=e))
    nc = g.N // 2
    worst, q99 = 0.0, 0.0
    for colour in (0, 1):
        before = g.get_spins()
        o.set_spins(before)
        ML = float((before.astype(np.float64) @ e).sum())
        n_o, ml_o, x_o, acc_o = o.constrained_half_sweep(T, e, colour, ML, want_detail=True)
        x_g, acc_g = g.constrained_half_sweep(T, theta, phi, colour, ML, want_detail=True)
        after_g = g.get_spins().astype(np.float64); after_o = o.get_spins()
        mine = (np.arange(g.N) >= nc) == bool(colour)
        assert (after_g[~mine] == before[~mine].astype(np.float64)).all()
        partner, lead = o.pairing(77, colour)
        lead_sites = colour * nc + np.nonzero(lead)[0]
        foll_sites = colour * nc + partner[np.nonzero(lead)[0]]
        assert not np.isnan(x_g[lead_sites]).any() and np.isnan(x_g[foll_sites]).all()
        assert (acc_g[lead_sites] == acc_g[foll_sites]).all()
        differ = acc_g[lead_sites] != acc_o[lead_sites]
        xo = x_o[lead_sites]
        assert (np.abs(xo[differ]) < X_BAND).all()
        ok_pairs = ~differ
        for sites in (lead_sites[ok_pairs], foll_sites[ok_pairs]):
            assert np.abs(after_g[sites] - after_o[sites]).max() < SPIN_TOL
        assert (np.isfinite(xo) == np.isfinite(x_g[lead_sites])).mean() > 0.999
        near = np.isfinite(x_g[lead_sites]) & (np.abs(xo) < 2.0)                              # the decision variable where it decides
        if near.any():
            # ln|S_j,par / S'_j,par| is ill-conditioned where the radicand of P:189 is small (a follower turned almost
            # perpendicular to e_C: fp32 rounding 1e-7 of the radicand over a radicand of 1e-4), so the maximum is reported
            # and the 99th percentile bounded; the decisions above are the bar
            dx = np.abs(x_g[lead_sites][near] - xo[near])
            worst = max(worst, float(dx.max())); q99 = max(q99, float(np.quantile(dx, 0.99)))
        assert np.abs(np.linalg.norm(after_g, axis=1) - 1).max() < 3e-7
        Mb = before.astype(np.float64).sum(axis=0); Ma = after_g.sum(axis=0)
        perp = (Ma - Mb) - ((Ma - Mb) @ e) * e
        assert np.abs(perp).max() < 1e-6 * np.sqrt(g.N) + 1e-5
    print(f"\nbcc constrained {shape} T={T}: |x_gpu - x_oracle| over |x| < 2: max {worst:.2e}, 99th percentile {q99:.2e}")
    assert q99 < 2e-5 and worst < 1e-2
    g.close()


def test_bcc_constrained_sweep_equals_hooks_and_holds_the_direction(mods):
    """mc_constrained_sweep on bcc: the fused M of every sweep equals the fp64 sum of the post-sweep state (2e-7 per site), the
    hook-assembled twin (M_L handed in from NumPy) ends in bit-identical spins, M stays along e_C, and the mean torque of an
    equilibrated run agrees with the oracle's within 3 standard errors."""
    from stats_util import blocked_mean_se
    oracle, binding, inputs = mods
    shape, T, theta, phi = (16, 8, 8), 1.0, 0.7, 0.4
    N = 2 * 16 * 8 * 8
    e = np.array([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)])
    s0 = inputs.thermal_like_spins(N, seed=2, spread=0.5, direction=e)
    kw = dict(Ku=0.05, cone0=0.6, adaptive=True, seed=42, structure="bcc")
    a = binding.Lattice(*shape, **kw); a.set_spins(s0)
    b = binding.Lattice(*shape, **kw); b.set_spins(s0)
    a.align_to(theta, phi); b.align_to(theta, phi)
    states = []
    for k in range(3):
        a.constrained_sweep(T, theta, phi, 1); states.append(a.get_spins())
    tr = a.trace()
    for k in range(3):
        M64 = states[k].astype(np.float64).sum(axis=0) / N
        assert np.abs(tr[k, 2:5] - M64).max() < 2e-7
        assert np.abs(M64 / np.linalg.norm(M64) - e).max() < 2e-6
    for k in range(3):
        ML = float((b.get_spins().astype(np.float64) @ e).sum())
        b.constrained_half_sweep(T, theta, phi, 0, ML); b.constrained_half_sweep(T, theta, phi, 1, ML); b.end_sweep()
        assert (b.get_spins() == states[k]).all(), k
    assert (b.trace()[:, :2] == tr[:, :2]).all()
    a.close(); b.close()
    # ensemble: |M|, E and the mean torque of an equilibrated run (Ku = 0.1, theta = pi/4), GPU against the oracle
    th = np.pi / 4
    o = oracle.Oracle(8, 8, 8, structure="bcc", Ku=0.1, cone0=0.8, adaptive=True, seed=3)
    g = binding.Lattice(8, 8, 8, structure="bcc", Ku=0.1, cone0=0.8, adaptive=True, seed=4)
    o.set_sampling(False); o.constrained_sweep(1.0, th, 0.0, 300); o.set_sampling(True); o.constrained_sweep(1.0, th, 0.0, 2000)
    g.constrained_sweep(1.0, th, 0.0, 300); g.reset_accumulators(); g.constrained_sweep(1.0, th, 0.0, 8000)
    to, tg = o.trace(), g.trace(8000)
    for f in (lambda t: np.linalg.norm(t[:, 2:5], axis=1), lambda t: t[:, 5]):
        x, sx = blocked_mean_se(f(tg)); y, sy = blocked_mean_se(f(to))
        assert abs(x - y) < 3 * np.hypot(sx, sy) + 1e-3
    og, oo = g.observables(), o.observables()
    ty_g = og.sum_torque[1] / og.n_samples; ty_o = oo.sum_torque[1] / oo.n_samples
    assert abs(ty_g - ty_o) < 0.03 * abs(ty_o), (ty_g, ty_o)
    assert -0.1 < ty_g < -0.03                                                                # a restoring torque of order K_u m^3
    g.close()
