"""GPU ensemble parity and full-size checks (BASELINE.json configs c1-c5 through the C ABI).

  * ensemble m(T), susceptibility, acceptance and cone agree with the oracle within 3 standard errors (north_star);
  * the physics pins of SURVEY section 8(c) re-run on the GPU path at sizes the oracle cannot reach;
  * one colour pass at BASELINE's FULL sizes (224^3, 2048x2048x4, 128^3 constrained), in the launch configuration
    bench.py times, compared with the oracle site by site.
"""
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

from stats_util import blocked_mean_se

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mods():
    import torch
    assert torch.cuda.is_available()
    import oracle
    from paper_2103_03517_b200 import binding, build, inputs
    build.build()
    return oracle, binding, inputs


def _mag(tr):
    return np.linalg.norm(tr[:, 2:5], axis=1)


def _chi(m, N, T, nb=20):
    """reduced susceptibility (N/T)(<m^2> - <m>^2) (Eq. 6, C-18) with a jackknife error over blocks."""
    n = (len(m) // nb) * nb
    b = m[:n].reshape(nb, -1)
    m1, m2 = b.mean(axis=1), (b ** 2).mean(axis=1)
    full = N / T * (m2.mean() - m1.mean() ** 2)
    jk = np.array([N / T * (np.delete(m2, i).mean() - np.delete(m1, i).mean() ** 2) for i in range(nb)])
    return full, np.sqrt((nb - 1) * jk.var())


def test_c1_trace_acceptance_cone_and_m(mods):
    """config c1: 16^3, K=0.01, T=1, +z start, 1000 adaptive sweeps from cone 0.5 rad, seed 42."""
    oracle, binding, inputs = mods
    g = binding.Lattice(16, 16, 16, Ku=0.01, cone0=0.5, adaptive=True, seed=42)
    g.sweep(1.0, 1000)
    tg = g.trace()
    o = oracle.Oracle(16, 16, 16, Ku=0.01, cone0=0.5, adaptive=True, seed=42)
    o.sweep(1.0, 1000)
    to = o.trace()
    assert len(tg) == 1000
    # the first sweep starts from the identical state with the identical stream: same acceptance up to marginal sites
    assert abs(tg[0, 0] - to[0, 0]) < 5 / 4096 and tg[0, 1] == to[0, 1] == 0.5
    for col, tol in ((0, 0.01), (1, np.radians(1.5))):
        assert abs(tg[300:, col].mean() - to[300:, col].mean()) < tol
    mg, sg = blocked_mean_se(_mag(tg[300:])); mo, so = blocked_mean_se(_mag(to[300:]))
    assert abs(mg - mo) < 3 * np.hypot(sg, so)
    Eg, sg = blocked_mean_se(tg[300:, 5]); Eo, so = blocked_mean_se(to[300:, 5])
    assert abs(Eg - Eo) < 3 * np.hypot(sg, so)
    assert abs(tg[300:, 0].mean() - 0.5) < 0.02
    print(f"\nc1: acceptance {tg[300:,0].mean():.4f} cone {np.degrees(tg[300:,1].mean()):.2f} deg m {mg:.4f} (oracle {mo:.4f}) E {Eg:.4f} (oracle {Eo:.4f})")
    g.close()


def test_ensemble_m_and_susceptibility_match_oracle(mods):
    """config c2's Hamiltonian at 16^3: m(T), chi_l and chi_z from the GPU and from the oracle within 3 SE."""
    oracle, binding, inputs = mods
    Ts = (0.6, 1.2, 1.5, 1.8)
    n_eq, n_s, L = 1000, 6000, 16
    def run_oracle(T):
        o = oracle.Oracle(L, L, L, Ku=0.01, cone0=0.5, seed=100 + int(10 * T))
        o.set_sampling(False); o.sweep(T, n_eq); o.set_sampling(True); o.sweep(T, n_s)
        return o.trace()
    with ThreadPoolExecutor(4) as ex:
        futs = [ex.submit(run_oracle, T) for T in Ts]
        gtr = []
        for T in Ts:
            g = binding.Lattice(L, L, L, Ku=0.01, cone0=0.5, seed=200 + int(10 * T))
            g.sweep(T, n_eq); g.reset_accumulators(); g.sweep(T, n_s)
            gtr.append((g.trace(n_s), g.observables())); g.close()
        otr = [f.result() for f in futs]
    for T, (tg, ob), to in zip(Ts, gtr, otr):
        assert len(tg) == n_s and ob.n_samples == n_s
        mg, sg = blocked_mean_se(_mag(tg)); mo, so = blocked_mean_se(_mag(to))
        assert abs(mg - mo) < 3 * np.hypot(sg, so), (T, mg, mo)
        cg, scg = _chi(_mag(tg), L ** 3, T); co, sco = _chi(_mag(to), L ** 3, T)
        assert abs(cg - co) < 3 * np.hypot(scg, sco), (T, cg, co)
        # accumulators (Eq. 6) reproduce the trace
        assert abs(ob.sum_m[0] / n_s - _mag(tg).mean()) < 1e-12
        assert abs(ob.sum_m2[3] / n_s - (tg[:, 4] ** 2).mean()) < 1e-12
        print(f"\nT={T}: m gpu {mg:.4f}+-{sg:.4f} oracle {mo:.4f}+-{so:.4f}; chi_l gpu {cg:.3f}+-{scg:.3f} oracle {co:.3f}+-{sco:.3f}")


def test_gpu_physics_pins(mods):
    oracle, binding, inputs = mods
    # P-6 Langevin at 64^3: J = 0, field along z
    g = binding.Lattice(64, 64, 64, J=0.0, B=(0, 0, 1.0), cone0=1.0, seed=1)
    g.sweep(0.5, 100); g.sweep(0.5, 300)
    m, se = blocked_mean_se(g.trace(300)[:, 4]); x = 2.0
    assert abs(m - (1 / np.tanh(x) - 1 / x)) < 3 * se + 1e-4
    g.close()
    # P-10 / P-11 spin waves at 32^3, T = 0.02
    L, K, T = 32, 0.01, 0.02
    g = binding.Lattice(L, L, L, Ku=K, cone0=0.5, seed=2)
    g.sweep(T, 3000); g.sweep(T, 3000)
    tr = g.trace(3000)
    k = 2 * np.pi * np.arange(L) / L
    kx, ky, kz = np.meshgrid(k, k, k, indexing="ij")
    eps = (2 * (3 - np.cos(kx) - np.cos(ky) - np.cos(kz)) + 2 * K).ravel()[1:]
    assert abs(_mag(tr).mean() - (1 - T * np.sum(1 / eps) / L ** 3)) < 1e-4
    assert abs(tr[:, 5].mean() - (-3 - K + T)) < 1e-3
    s = g.get_spins()
    assert np.abs(np.linalg.norm(s.astype(np.float64), axis=1) - 1).max() < 2e-7      # P-4 after 6000 sweeps
    g.close()
    # P-9 open chain
    g = binding.Lattice(4096, 1, 1, periodic=(0, 0, 0), cone0=1.0, seed=3)
    g.sweep(1.0, 300); g.sweep(1.0, 3000)
    m, se = blocked_mean_se(g.trace(3000)[:, 5])
    assert abs(m - (-(4095 / 4096) * (1 / np.tanh(1.0) - 1))) < 3 * se + 1e-4
    g.close()


def test_c2_temperature_sweep_tc_from_susceptibility_peak(mods):
    """config c2: 64^3, K=0.01, T = 0.1..1.6 in 16 steps, +z start at every T.  (Sweep counts reduced 5x from
    BASELINE's 5000+5000 to keep the test short; the schedule is otherwise the config's.)"""
    oracle, binding, inputs = mods
    L, n_eq, n_s = 64, 1000, 1000
    Ts = [0.1 * k for k in range(1, 17)]
    m, chi = [], []
    for k, T in enumerate(Ts, start=1):
        g = binding.Lattice(L, L, L, Ku=0.01, cone0=0.5, seed=42 + k)
        g.sweep(T, n_eq); g.reset_accumulators(); g.sweep(T, n_s)
        ob = g.observables()
        ml = ob.sum_m[0] / ob.n_samples
        m.append(ml); chi.append(L ** 3 / T * (ob.sum_m2[0] / ob.n_samples - ml ** 2))
        g.close()
    m, chi = np.array(m), np.array(chi)
    print("\nc2 m(T):", np.round(m, 4)); print("c2 chi_l(T):", np.round(chi, 3))
    assert np.all(np.diff(m) < 0)                                   # m decreases monotonically with T
    # Bloch law with the paper's fit up to T = 1.2 (pin P-15)
    for T, v in zip(Ts[:12], m[:12]):
        assert abs(v - (1 - T / 1.4451) ** 0.340) < 0.03, (T, v)
    ipk = int(np.argmax(chi))
    assert ipk in (13, 14)                                          # chi_l peaks at T = 1.4 or 1.5: T_c = 1.443 on a 0.1 grid (P-14, C-19)
    a, b, c = np.polyfit(Ts[ipk - 1: ipk + 2], chi[ipk - 1: ipk + 2], 2)
    assert abs(-b / (2 * a) - 1.443) < 0.06
    assert chi[0] < 0.05 * chi[ipk]                                 # chi_l -> 0 as T -> 0


def test_c4_constrained_torque_on_gpu(mods):
    """config c4 at 64^3 (one theta, three T): direction held (P-16), torque -> K(T) = K_u m^3 (P-18)."""
    oracle, binding, inputs = mods
    L, Ku, theta = 64, 0.05, np.pi / 4
    e = np.array([np.sin(theta), 0, np.cos(theta)])
    for T in (0.3, 0.8, 1.2):
        g = binding.Lattice(L, L, L, Ku=Ku, cone0=0.5, seed=42)
        g.constrained_sweep(T, theta, 0.0, 600); g.reset_accumulators(); g.constrained_sweep(T, theta, 0.0, 800)
        ob = g.observables(); tr = g.trace(800)
        assert np.abs(tr[:, 2:5] / _mag(tr)[:, None] - e).max() < 2e-6
        tq = np.array(ob.sum_torque) / ob.n_samples
        K = -tq[1] / np.sin(2 * theta) / Ku
        m = ob.sum_m[0] / ob.n_samples
        print(f"\nc4 T={T}: m={m:.4f} K(T)/Ku={K:.4f} m^3={m**3:.4f} acceptance={tr[:,0].mean():.3f}")
        # Callen-Callen K(T)/K_u = m^3 is the LOW-temperature law; the paper's fit over its whole range gives
        # the smaller exponent 2.95.  Up to T = 0.8 the m^3 law must hold to 3 %; at T = 1.2 (0.83 T_c) only the effective
        # exponent ln K / ln m is pinned to the window around the paper's fit.
        if T <= 0.8:
            assert abs(K - m ** 3) < 0.03 * m ** 3 + 2e-3
        else:
            assert 2.7 < np.log(K) / np.log(m) < 3.05
        assert abs(tr[200:, 0].mean() - 0.5) < 0.03
        g.close()


def test_constrained_ensemble_matches_oracle(mods):
    oracle, binding, inputs = mods
    L, T, theta = 16, 0.8, np.pi / 4
    def run_oracle():
        o = oracle.Oracle(L, L, L, Ku=0.05, cone0=0.5, seed=7)
        o.set_sampling(False); o.constrained_sweep(T, theta, 0.0, 1000); o.set_sampling(True); o.constrained_sweep(T, theta, 0.0, 4000)
        return o.trace(), o.observables()
    with ThreadPoolExecutor(1) as ex:
        fut = ex.submit(run_oracle)
        g = binding.Lattice(L, L, L, Ku=0.05, cone0=0.5, seed=8)
        g.constrained_sweep(T, theta, 0.0, 1000); g.reset_accumulators(); g.constrained_sweep(T, theta, 0.0, 4000)
        tg, og = g.trace(4000), g.observables(); g.close()
        to, oo = fut.result()
    for f in (_mag, lambda t: t[:, 5]):
        a, sa = blocked_mean_se(f(tg)); b, sb = blocked_mean_se(f(to))
        assert abs(a - b) < 3 * np.hypot(sa, sb)
    ty_g = og.sum_torque[1] / og.n_samples; ty_o = oo.sum_torque[1] / oo.n_samples
    assert abs(ty_g - ty_o) < 0.02 * abs(ty_o)


# ---------------------------------------------------------------------------------------------- full sizes
def _full_size_half_sweep(mods, shape, T, cone, state_seed, ham, colour=0):
    oracle, binding, inputs = mods
    N = shape[0] * shape[1] * shape[2]
    g = binding.Lattice(*shape, seed=42, cone0=cone, adaptive=False, **ham)
    o = oracle.Oracle(*shape, seed=42, cone0=cone, adaptive=False, **ham)
    g.set_spins(inputs.random_unit_spins(N, seed=state_seed))
    g.set_sweep(1234); o.set_sweep(1234)
    before = g.get_spins()
    o.set_spins(before)
    _, x_o, acc_o = o.half_sweep(T, colour, want_detail=True)
    x_g, acc_g = g.half_sweep(T, colour, want_detail=True)
    after_g = g.get_spins(); after_o = o.get_spins()
    s = np.arange(N); col = ((s % shape[0]) + (s // shape[0]) % shape[1] + s // (shape[0] * shape[1])) & 1
    mine = col == colour
    differ = mine & (acc_g != acc_o)
    assert (np.abs(x_o[differ]) < 1e-5).all()
    agree = mine & ~differ
    assert np.abs(after_g[agree].astype(np.float64) - after_o[agree]).max() < 1e-4
    assert (after_g[~mine] == before[~mine]).all()
    dx = np.abs(x_g[mine] - x_o[mine]).max()
    print(f"\nfull size {shape}: {mine.sum()} updates, accepted {acc_g[mine].mean():.3f}, marginal flips {differ.sum()}, max |dx| {dx:.2e}")
    g.close()


def test_full_size_c3_half_sweep_parity(mods):
    """config c3: 224^3 = 11.24 M spins, Kc = 0.01, T = 1.2, random-sphere start -- the headline launch configuration."""
    _full_size_half_sweep(mods, (224, 224, 224), 1.2, 1.0, 42, dict(Kc=0.01), colour=1)


def test_full_size_c3_timed_kernels_match_the_checked_ones(mods):
    """The kernels bench.py times at c3 are the compile-time-row-length instantiation launched back to back with
    programmatic dependent launch; the parity test above goes through the instantiation that also writes the decision
    variable.  Same state, same sweep counter: (i) one colour pass of the timed instantiation against the oracle
    (a spin may differ only where the oracle's decision was marginal), and bit for bit against the checked one;
    (ii) mc_sweep(T, 2) = four dependent launches against the same four passes issued one by one with a
    synchronisation after each: bitwise equal spins, sums and controller state."""
    oracle, binding, inputs = mods
    shape, T = (224, 224, 224), 1.2
    N = 224 ** 3
    s0 = inputs.random_unit_spins(N, seed=42)
    ham = dict(Kc=0.01)
    g = binding.Lattice(*shape, seed=42, cone0=1.0, adaptive=False, **ham)
    o = oracle.Oracle(*shape, seed=42, cone0=1.0, adaptive=False, **ham)
    g.set_spins(s0); g.set_sweep(77); o.set_sweep(77)
    before = g.get_spins(); o.set_spins(before)
    _, x_o, acc_o = o.half_sweep(T, 0, want_detail=True)
    g.half_sweep(T, 0)                                                     # no detail: the timed instantiation
    fast = g.get_spins()
    g.set_spins(s0); g.set_sweep(77)
    g.half_sweep(T, 0, want_detail=True)                                   # the checked instantiation
    assert (g.get_spins() == fast).all()
    after_o = o.get_spins()
    bad = np.abs(fast.astype(np.float64) - after_o).max(axis=1) >= 1e-4
    assert (np.abs(x_o[bad]) < 1e-5).all() and bad.sum() < 50
    g.close()
    a = binding.Lattice(*shape, seed=42, cone0=0.5, adaptive=True, **ham); a.set_spins(s0)
    b = binding.Lattice(*shape, seed=42, cone0=0.5, adaptive=True, **ham); b.set_spins(s0)
    a.sweep(T, 2)
    for _ in range(2):
        b.half_sweep(T, 0); b.observables(); b.half_sweep(T, 1); b.end_sweep(); b.observables()
    oa, ob = a.observables(), b.observables()
    assert (a.get_spins() == b.get_spins()).all()
    assert oa.sweep == ob.sweep == 2 and oa.cone_rad == ob.cone_rad and oa.E_total == ob.E_total and list(oa.M) == list(ob.M)
    assert (a.trace() == b.trace()).all()
    a.close(); b.close()


@pytest.mark.parametrize("T", [0.5, 1.44])
def test_full_size_c3_parity_at_the_points_bench_times(mods, T):
    """bench.py cycles T through {0.5, 1.2, 1.44} with the adaptive cone from a random-sphere start.  Here the library
    itself runs 60 such sweeps at T (the controller settles near 0.67 rad at T = 0.5 and near 1.6 rad at T = 1.44), then
    BOTH colour passes from that state, with that cone and sweep counter, are compared with the oracle site by site."""
    oracle, binding, inputs = mods
    shape = (224, 224, 224); N = 224 ** 3
    ham = dict(Kc=0.01)
    g = binding.Lattice(*shape, seed=42, cone0=0.5, adaptive=True, **ham)
    g.set_spins(inputs.random_unit_spins(N, seed=42))
    g.sweep(T, 60)
    ob = g.observables()
    o = oracle.Oracle(*shape, seed=42, cone0=ob.cone_rad, adaptive=False, **ham)
    o.set_sweep(ob.sweep)
    s = np.arange(N); col = ((s % 224) + (s // 224) % 224 + s // (224 * 224)) & 1
    for colour in (0, 1):
        before = g.get_spins(); o.set_spins(before)
        _, x_o, acc_o = o.half_sweep(T, colour, want_detail=True)
        x_g, acc_g = g.half_sweep(T, colour, want_detail=True)
        after_g = g.get_spins(); after_o = o.get_spins()
        mine = col == colour
        differ = mine & (acc_g != acc_o)
        assert (np.abs(x_o[differ]) < 1e-5).all()
        agree = mine & ~differ
        assert np.abs(after_g[agree].astype(np.float64) - after_o[agree]).max() < 1e-4
        assert (after_g[~mine] == before[~mine]).all()
        near = mine & (np.abs(x_o) < 2.0)
        print(f"\n224^3 T={T} cone={ob.cone_rad:.3f} colour {colour}: accepted {acc_g[mine].mean():.3f}, marginal flips {differ.sum()}, "
              f"max |dx| near the boundary {np.abs(x_g[near] - x_o[near]).max():.2e}")
        assert np.abs(x_g[near] - x_o[near]).max() < 1e-5
    g.close()


@pytest.mark.parametrize("colour", [0, 1])
def test_full_size_c5_half_sweep_parity(mods, colour):
    """config c5: 2048 x 2048 x 4 granular film (16.8 M spins), Voronoi grains, per-grain axes, open z."""
    oracle, binding, inputs = mods
    shape = (2048, 2048, 4)
    mask, region, axes = inputs.voronoi_film(*shape, mean_diameter=40, seed=42)
    _full_size_half_sweep(mods, shape, 0.5, 0.8, 43, dict(periodic=(1, 1, 0), Ku=0.02, bond_mask=mask, region=region, region_axis=axes), colour=colour)


@pytest.mark.parametrize("colour", [0, 1])
@pytest.mark.parametrize("L", [128, 224])
def test_full_size_c4_constrained_half_sweep_parity(mods, L, colour):
    """config c4: 128^3, K_u = 0.05, constrained pass at theta = 45 deg; and the same pass on the 224^3 lattice on which
    bench.py times the constrained sweeps (other_paths)."""
    oracle, binding, inputs = mods
    shape, T, theta = (L, L, L), 0.8, np.pi / 4
    N = L ** 3
    e = np.array([np.sin(theta), 0.0, np.cos(theta)])
    g = binding.Lattice(*shape, Ku=0.05, cone0=0.6, adaptive=False, seed=42)
    o = oracle.Oracle(*shape, Ku=0.05, cone0=0.6, adaptive=False, seed=42)
    g.set_spins(inputs.thermal_like_spins(N, seed=5, spread=0.5, direction=e))
    g.set_sweep(9); o.set_sweep(9)
    before = g.get_spins(); o.set_spins(before)
    ML = float((before.astype(np.float64) @ e).sum())
    _, _, x_o, acc_o = o.constrained_half_sweep(T, e, colour, ML, want_detail=True)
    x_g, acc_g = g.constrained_half_sweep(T, theta, 0.0, colour, ML, want_detail=True)
    after_g = g.get_spins().astype(np.float64); after_o = o.get_spins()
    lead = ~np.isnan(x_o)
    assert (lead == ~np.isnan(x_g)).all()                                  # identical pairing roles at full size
    differ = lead & (acc_g != acc_o)
    assert (np.abs(x_o[differ]) < 1e-5).all()
    s = np.arange(N); col = ((s % L) + (s // L) % L + s // (L * L)) & 1
    same = (acc_g == acc_o) & (col == colour)
    assert np.abs(after_g[same] - after_o[same]).max() < 1e-4
    fin = lead & np.isfinite(x_o) & np.isfinite(x_g)
    print(f"\nfull size {L}^3 constrained: pairs {lead.sum()}, accepted {acc_g[lead].mean():.3f}, flips {differ.sum()}, max |dx| {np.abs(x_g[fin]-x_o[fin]).max():.2e}")
    g.close()


def test_full_size_march_pass_half_sweep_parity(mods):
    """256^3 = 16.8 M spins: the lattice size class whose default kernel is the register-carried march pass (9 z-segments per
    column, one resident wave) -- one colour pass against the oracle, in the launch configuration mc_sweep uses."""
    oracle, binding, inputs = mods
    g = binding.Lattice(256, 256, 256, Kc=0.01); assert g.debug_get_path() == binding.MC_PATH_MARCH; g.close()
    _full_size_half_sweep(mods, (256, 256, 256), 1.2, 1.2, 7, dict(Kc=0.01), colour=1)


# ---------------------------------------------------------------------------------------------- f-1 domain-wall workload
def test_domain_wall_workload_gives_the_exchange_stiffness(mods):
    """SURVEY 8f-1 end to end: anti-periodic box, slice profiles, tanh fits, K(T) from the constrained torque,
    A(T) = K Delta^2 / pi^2.  Checks against what the model fixes: A(T -> 0) = J/2 per lattice spacing (sc, nearest neighbours),
    Delta(T -> 0) = pi sqrt(J / 2 K_u), and an exponent of A ~ m^k between the paper's low-temperature values and mean field
    (Table I: 1.48 ... 1.79; MFA: 2)."""
    from paper_2103_03517_b200 import configs
    out = configs.dw(shape=(96, 32, 32), Ku=0.05, temps=(0.2, 0.5, 0.8, 1.0), equil=1500, snapshots=120, every=10)
    pts = out["points"]
    assert all(p["fits"] > 100 for p in pts)
    assert abs(pts[0]["Delta"] / out["expected_T0"]["Delta"] - 1) < 0.06            # T = 0.2: a few per cent wider than at T = 0
    assert all(a["Delta"] < b["Delta"] for a, b in zip(pts, pts[1:]))               # the wall widens with T (Fig. 2)
    assert abs(out["A0_extrapolated"] / 0.5 - 1) < 0.08
    # four points and short runs: the slope is good to about +-0.25 (the full schedule of configs.dw gives 1.76)
    assert 1.1 < out["A_over_m_exponent_m_gt_0.6"] < 2.1, out["A_over_m_exponent_m_gt_0.6"]


# ---------------------------------------------------------------------------------------------- f-4 second anisotropy route
def test_easy_axis_route_of_eq4_follows_the_callen_callen_law(mods):
    """SURVEY 8f-4 end to end: K(T)/K(0) from the easy-axis anisotropy energy of a standard run (Eq. (4)) against the
    l = 2 Callen-Callen law the paper measures (m^2.95) and against the constrained torque route ("identical results")."""
    from paper_2103_03517_b200 import configs
    out = configs.f4(L=32, Ku=0.05, temps=(0.3, 0.6, 0.9), equil=1500, samples=150, every=10)
    for p in out["points"]:
        assert abs(p["k_eq4"] - p["m^2.95"]) < 0.02, p
        assert abs(p["k_torque"] - p["k_eq4"]) < 0.06, p
        assert 0.3 < p["chi_perp_eq6"] / p["chi_perp_eq7"] < 3.0, p             # Eq. (7): same order (the macrospin mode is slow to sample)


# ---------------------------------------------------------------------------------------------- f-2 lattices at bench size
@pytest.mark.parametrize("structure,L,T,colour,ham", [
    ("bcc", 176, 1.8, 1, dict()),                    # 10.9 M spins, 8 neighbours
    ("fcc", 140, 2.8, 3, dict()),                    # 11.0 M spins, 12 neighbours, four colours
    ("hcp", 176, 2.8, 5, dict()),                    # 43.6 M spins, 12 neighbours through the bond table, eight colours
    ("sc_nnn", 176, 2.0, 2, dict(J2=0.3)),           # 43.6 M spins, 6 + 12 neighbours
])
def test_full_size_sublattice_lattices_at_the_sizes_bench_times(mods, structure, L, T, colour, ham):
    """The lattices of bench.py's `other_paths` at the sizes and in the launch configuration it times: the library
    runs 12 sweeps at T from the seeded random-sphere start with the adaptive cone (as the bench does), then ONE colour pass from
    that state, with that cone and sweep counter, is compared with the oracle site by site (C-14 bar)."""
    oracle, binding, inputs = mods
    g = binding.Lattice(L, L, L, Ku=0.01, cone0=0.5, adaptive=True, seed=42, structure=structure, **ham)
    g.init_spins(2); g.sweep(T, 12)
    ob = g.observables()
    o = oracle.Oracle(L, L, L, Ku=0.01, cone0=ob.cone_rad, adaptive=False, seed=42, structure=structure, **ham)
    o.set_sweep(ob.sweep)
    before = g.get_spins(); o.set_spins(before)
    _, x_o, acc_o = o.half_sweep(T, colour, want_detail=True)
    x_g, acc_g = g.half_sweep(T, colour, want_detail=True)
    after_g = g.get_spins(); after_o = o.get_spins()
    nc = L ** 3
    mine = np.zeros(g.N, bool); mine[colour * nc:(colour + 1) * nc] = True
    differ = mine & (acc_g != acc_o)
    assert (np.abs(x_o[differ]) < 1e-5).all()
    agree = mine & ~differ
    assert np.abs(after_g[agree].astype(np.float64) - after_o[agree]).max() < 1e-4
    assert (after_g[~mine] == before[~mine]).all()
    near = mine & (np.abs(x_o) < 2.0)
    dx = np.abs(x_g[near] - x_o[near]).max()
    print(f"\n{structure} {L}^3 cells T={T} cone={ob.cone_rad:.3f} colour {colour}: {nc} updates, accepted {acc_g[mine].mean():.3f}, "
          f"marginal flips {differ.sum()}, max |dx| near the boundary {dx:.2e}")
    assert dx < 1e-5 and differ.sum() < 50
    g.close()


def test_full_size_bcc_constrained_half_sweep_parity(mods):
    """The constrained pair pass on the 176^3-cell bcc lattice bench.py times (Table A2 with the 8-bond field): after 12
    constrained sweeps of the library, one pair pass of sublattice B against the oracle: same pairs decided the same way outside
    the band, both members of every agreeing pair to 1e-4."""
    oracle, binding, inputs = mods
    L, T, theta, phi = 176, 0.8, 0.6, 0.0
    e = np.array([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)])
    g = binding.Lattice(L, L, L, Ku=0.01, cone0=0.5, adaptive=True, seed=42, structure="bcc")
    g.constrained_sweep(T, theta, phi, 12)
    ob = g.observables()
    o = oracle.Oracle(L, L, L, Ku=0.01, cone0=ob.cone_rad, adaptive=False, seed=42, structure="bcc")
    o.set_sweep(ob.sweep)
    before = g.get_spins(); o.set_spins(before)
    ML = float((before.astype(np.float64) @ e).sum())
    colour, nc = 1, L ** 3
    _, _, x_o, acc_o = o.constrained_half_sweep(T, e, colour, ML, want_detail=True)
    x_g, acc_g = g.constrained_half_sweep(T, theta, phi, colour, ML, want_detail=True)
    after_g = g.get_spins().astype(np.float64); after_o = o.get_spins()
    partner, lead = o.pairing(int(ob.sweep), colour)
    la = np.nonzero(lead)[0]
    lead_sites, foll_sites = colour * nc + la, colour * nc + partner[la]
    assert not np.isnan(x_g[lead_sites]).any() and np.isnan(x_g[foll_sites]).all()
    assert (acc_g[lead_sites] == acc_g[foll_sites]).all()
    differ = acc_g[lead_sites] != acc_o[lead_sites]
    assert (np.abs(x_o[lead_sites][differ]) < 1e-5).all() and differ.sum() < 50
    for sites in (lead_sites[~differ], foll_sites[~differ]):
        assert np.abs(after_g[sites] - after_o[sites]).max() < 1e-4
    assert (after_g[:nc] == before[:nc].astype(np.float64)).all()
    print(f"\nbcc constrained 176^3 cells: {len(la)} pairs, accepted {acc_g[lead_sites].mean():.3f}, marginal flips {differ.sum()}")
    g.close()


# ---------------------------------------------------------------------------------------------- maximum size
def test_maximum_size_lattice_sampled_parity_and_path_equality(mods):
    """The largest lattice the boundary accepts (N < 2^31, include/mc.h): 1280 x 1280 x 1310 = 2 146 304 000 spins, 25.8 GB of state
    plus the staging area in one 51.5 GB workspace -- a quarter of a B200's HBM (the paper: "100 M spins in 6 GB").
      * sampled parity: from the +z start, one red and one black pass (march pass); the oracle recomputes SAMPLED sites one by
        one -- uniforms of the true site index (top of the 32-bit site-id range included), cone move, dE from the site's six
        neighbours as the GPU left them -- and the GPU's spin must be the oracle's outcome (decisions inside the band skipped);
      * any-size property: the same two passes through the gather (other index arithmetic, same counters) give the same
        accepted count (exact), M and E of the trace row to 2e-7 per site, and bit-identical spins on the sampled sites."""
    import torch
    oracle, binding, inputs = mods
    if torch.cuda.mem_get_info()[0] < 60e9:
        pytest.skip("needs 52 GB of free device memory")
    shape = (1280, 1280, 1310)
    nx, ny, nz = shape
    N = nx * ny * nz
    assert 2 ** 31 - 2_000_000 < N < 2 ** 31
    ham = dict(Ku=0.05, eu=(0.3, -0.5, 0.81), Kc=0.01, B=(0.02, 0.0, -0.01))
    T, cone, sweep0 = 1.0, 0.6, (7 << 32) | 123
    g = binding.Lattice(*shape, seed=42, cone0=cone, adaptive=False, **ham)
    assert g.debug_get_path() == binding.MC_PATH_MARCH
    ob = g.observables()
    assert abs(ob.E_exch + 3.0) < 1e-6 and abs(ob.m - 1.0) < 1e-6
    g.set_sweep(sweep0)
    g.half_sweep(T, 0); g.half_sweep(T, 1); g.end_sweep()
    S = g.get_spins()
    row_march = g.trace(1)[0].copy()
    assert 0.2 < row_march[0] < 0.8

    # sampled sites: the corners of the index range, the planes at the periodic wrap, around site ids 2^30 and N - 1, random ones
    rng = np.random.default_rng(5)
    sites = [0, 1, nx - 1, nx, nx * ny - 1, N - 1, N - 2, N - nx, N - nx * ny, 2 ** 30 - 1, 2 ** 30, 2 ** 30 + 1, N // 2, N // 2 + 1]
    sites += [int(v) for v in rng.integers(0, N, 300)] + [int(v) for v in rng.integers(N - 4 * nx * ny, N, 100)]
    U = oracle.Oracle(nx, ny, 2, seed=42, cone0=cone, adaptive=False, **ham)          # the uniforms depend on nx, ny and the site index only
    E = oracle.Oracle(4, 4, 4, seed=42, cone0=cone, adaptive=False, **ham)            # the energy of a site given its six neighbours
    centre = 1 + 4 * (1 + 4 * 1)
    nb_small = [2 + 4 * (1 + 4 * 1), 0 + 4 * (1 + 4 * 1), 1 + 4 * (2 + 4 * 1), 1 + 4 * (0 + 4 * 1), 1 + 4 * (1 + 4 * 2), 1 + 4 * (1 + 4 * 0)]
    zhat = np.array([0.0, 0.0, 1.0])
    checked = skipped = 0
    expect = {}
    for s in sites:
        x, y, z = s % nx, (s // nx) % ny, s // (nx * ny)
        colour = (x + y + z) & 1
        u0, u1, u2 = U.site_uniforms(x, y, z, colour, sweep0)
        Sn = oracle.cone_move(zhat, cone, u0, u1)
        nb_big = [((x + 1) % nx) + nx * (y + ny * z), ((x - 1) % nx) + nx * (y + ny * z), x + nx * (((y + 1) % ny) + ny * z),
                  x + nx * (((y - 1) % ny) + ny * z), x + nx * (y + ny * ((z + 1) % nz)), x + nx * (y + ny * ((z - 1) % nz))]
        patch = np.tile(zhat, (64, 1))
        if colour == 1:                                                                # the black pass sees the red sites as the red pass left them
            for a, b in zip(nb_small, nb_big): patch[a] = S[b].astype(np.float64)
        E.set_spins(patch)
        xd = (E.site_energy(centre, Sn) - E.site_energy(centre, zhat)) / T + np.log(u2)
        if abs(xd) < 1e-5:
            skipped += 1; continue
        want = Sn if xd < 0 else zhat
        assert np.abs(S[s].astype(np.float64) - want).max() < 1e-4, (s, x, y, z, colour, xd)
        expect[s] = S[s].copy(); checked += 1
    assert checked > 400 and skipped < 5

    # the same two passes through the gather
    g.init_spins(0); g.set_sweep(sweep0); g.set_cone(cone); g.debug_set_path(binding.MC_PATH_GENERIC)
    g.half_sweep(T, 0); g.half_sweep(T, 1); g.end_sweep()
    row_gen = g.trace(1)[0].copy()
    # accepted count and cone: exact; M and E: the per-thread fp32 partial sums group the sites differently (2e-7 per site)
    assert (row_gen[:2] == row_march[:2]).all() and np.abs(row_gen[2:] - row_march[2:]).max() < 2e-7, (row_gen, row_march)
    S2 = g.get_spins()
    for s, v in expect.items():
        assert (S2[s] == v).all()
    del S, S2
    g.close()
