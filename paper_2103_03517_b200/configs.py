"""The five workloads of BASELINE.json, run in full through the library (python -m paper_2103_03517_b200.configs).

Every schedule is the one BASELINE.json / SURVEY.md 8(d) states (no shortening: on a B200 all five together take well
under a minute of device time); inputs are seeded and synthetic (paper_2103_03517_b200/inputs.py).  Prints one JSON
object per config with the outputs the config names (per-sweep acceptance and m; m(T), susceptibilities and T_C from the
susceptibility peak; throughput; torque versus theta and K(T); film m(T)) next to what the paper prints for the same
physics where it prints something (P:44 T_C and beta, P:52 anisotropy exponent).  Host analysis: analysis.py.
"""
from __future__ import annotations

import json
import sys
import time

import numpy as np

from . import analysis, binding, inputs, replicas


def _sync():
    import torch
    torch.cuda.synchronize()


def c1(device="cuda:0"):
    g = binding.Lattice(16, 16, 16, Ku=0.01, cone0=0.5, adaptive=True, seed=42, device=device)
    g.sweep(1.0, 1000)
    tr = g.trace()
    out = {"config": "c1 16^3, Ku=0.01, T=1.0, 1000 sweeps, +z start, adaptive cone from 0.5 rad",
           "acceptance_first_10": [round(v, 4) for v in tr[:10, 0]], "acceptance_last_500_mean": float(tr[-500:, 0].mean()),
           "cone_rad_final": float(g.observables().cone_rad),
           "m_last_500_mean": float(np.linalg.norm(tr[-500:, 2:5], axis=1).mean())}
    g.close()
    return out


def _c2_point(point, seed, device):
    """One temperature point of c2: its own handle, +z start, `seed` = 42 + k (replicas.point_seed)."""
    T, L, equil, sample = point
    g = binding.Lattice(L, L, L, Ku=0.01, cone0=0.5, adaptive=True, seed=seed, device=device)
    g.sweep(T, equil); g.reset_accumulators(); g.sweep(T, sample)
    ob = g.observables()
    chi = analysis.susceptibilities(ob, T)
    g.close()
    return {"m": ob.sum_m[0] / ob.n_samples, "chi_l": float(chi[0]), "chi_t": float(0.5 * (chi[1] + chi[2]))}


def _c2_create(point, seed, device, stream):
    T, L, equil, sample = point
    return binding.Lattice(L, L, L, Ku=0.01, cone0=0.5, adaptive=True, seed=seed, device=device, stream=stream)


def _c2_phases(point):
    T, L, equil, sample = point
    return [("sweep", T, equil), ("reset",), ("sweep", T, sample)]


def _c2_collect(g, point):
    ob = g.observables()
    chi = analysis.susceptibilities(ob, point[0])
    g.close()
    return {"m": ob.sum_m[0] / ob.n_samples, "chi_l": float(chi[0]), "chi_t": float(0.5 * (chi[1] + chi[2]))}


def c2(device=None, L=64, equil=5000, sample=5000, dist=None, concurrent=True):
    """16 independent temperature points: dealt over the ranks by replicas.run_points (several ranks), or -- one process, the default
    -- all at once on one device, one stream each, their sweeps replayed as CUDA graphs (replicas.run_points_concurrent; the same
    numbers bit for bit)."""
    Ts = [0.1 * k for k in range(1, 17)]
    pts = [(T, L, equil, sample) for T in Ts]
    if dist is None and concurrent:
        res = replicas.run_points_concurrent(pts, _c2_create, _c2_phases, _c2_collect, device=device or "cuda:0", base_seed=42)
    else:
        res = replicas.run_points(pts, _c2_point, base_seed=42, dist=dist, device=device)
    if res is None:
        return None                                           # not rank 0
    m, chi_l, chi_t = [r["m"] for r in res], [r["chi_l"] for r in res], [r["chi_t"] for r in res]
    tc_peak = Ts[int(np.argmax(chi_l))]
    below = [i for i, T in enumerate(Ts) if T < tc_peak and m[i] > 0.3]
    tc_fit, beta, _ = analysis.fit_bloch([Ts[i] for i in below], [m[i] for i in below])
    return {"config": f"c2 {L}^3, Ku=0.01, T=0.1..1.6, {equil}+{sample} sweeps per point", "T": Ts, "m": m, "chi_longitudinal": chi_l,
            "chi_transverse": chi_t, "Tc_from_chi_peak": tc_peak, "bloch_fit": {"Tc": tc_fit, "beta": beta},
            "paper": {"kB_Tc_over_J": 1.4451, "beta": 0.340, "where": "P:44 (50 nm^3 mesh, 8 M spins)"}}


def c3(device="cuda:0", L=224, sweeps=2000):
    import torch
    N = L ** 3
    out = {"config": f"c3 {L}^3, Kc=0.01, T in (0.5, 1.2, 1.44), {sweeps} sweeps each from a seeded random-sphere start", "points": []}
    for T in (0.5, 1.2, 1.44):
        g = binding.Lattice(L, L, L, Kc=0.01, cone0=0.5, adaptive=True, seed=42, device=device)
        g.init_spins(2)
        g.sweep(T, sweeps // 2); _sync()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); g.sweep(T, sweeps - sweeps // 2); e1.record(); _sync()
        ob = g.observables()
        out["points"].append({"T": T, "m": ob.m, "E_per_site": ob.E_total, "acceptance": ob.last_acceptance, "cone_rad": ob.cone_rad,
                              "updates_per_s_last_half": N * (sweeps - sweeps // 2) / (e0.elapsed_time(e1) * 1e-3)})
        g.close()
    return out


def _c4_point(point, seed, device):
    """One (T, theta) point of c4: +z start rotated onto e_C (C-12), seed 42 at every point as BASELINE.json states."""
    T, th, L, sweeps, discard = point
    g = binding.Lattice(L, L, L, Ku=0.05, cone0=0.5, adaptive=True, seed=42, device=device)
    g.constrained_sweep(T, th, 0.0, discard); g.reset_accumulators(); g.constrained_sweep(T, th, 0.0, sweeps - discard)
    ob = g.observables()
    g.close()
    return {"tau_y": ob.sum_torque[1] / ob.n_samples, "m": ob.sum_m[0] / ob.n_samples}


def _c4_create(point, seed, device, stream):
    return binding.Lattice(point[2], point[2], point[2], Ku=0.05, cone0=0.5, adaptive=True, seed=42, device=device, stream=stream)


def _c4_phases(point):
    T, th, L, sweeps, discard = point
    return [("constrained", T, th, 0.0, discard), ("reset",), ("constrained", T, th, 0.0, sweeps - discard)]


def _c4_collect(g, point):
    ob = g.observables()
    g.close()
    return {"tau_y": ob.sum_torque[1] / ob.n_samples, "m": ob.sum_m[0] / ob.n_samples}


def c4(device=None, L=128, sweeps=5000, discard=1000, dist=None, concurrent=True):
    """33 independent (T, theta) points through replicas.run_points (several ranks) or, one process, concurrently on one device
    (replicas.run_points_concurrent, 11 at a time)."""
    thetas = np.deg2rad(np.arange(0, 91, 9))                  # 0..90 deg in 10 steps (C-20)
    temps = (0.3, 0.8, 1.2)
    pts = [(T, float(th), L, sweeps, discard) for T in temps for th in thetas]
    if dist is None and concurrent:
        res = replicas.run_points_concurrent(pts, _c4_create, _c4_phases, _c4_collect, device=device or "cuda:0", base_seed=42, max_concurrent=11)
    else:
        res = replicas.run_points(pts, _c4_point, base_seed=42, dist=dist, device=device)
    if res is None:
        return None
    out = {"config": f"c4 {L}^3, Ku=0.05, constrained, theta=0..90 deg (11 points), T in (0.3, 0.8, 1.2), {sweeps} sweeps per point", "points": []}
    Ks, ms = [], []
    for i, T in enumerate(temps):
        tau = [r["tau_y"] for r in res[i * len(thetas):(i + 1) * len(thetas)]]
        mm = [r["m"] for r in res[i * len(thetas):(i + 1) * len(thetas)]]
        fit = thetas <= np.deg2rad(45.5)                     # towards the hard plane the uniform state of so large a lattice is not
        K = analysis.anisotropy_from_torque(thetas[fit], np.array(tau)[fit])   # stable over 5000 sweeps (|M| drops, domains): fit the stable branch
        Ks.append(K); ms.append(float(np.mean(np.array(mm)[fit])))
        out["points"].append({"T": T, "torque_y": tau, "m_of_theta": mm, "m": ms[-1], "K_fit_theta_le_45deg": K})
    k, K0 = analysis.power_law_exponent(np.array(ms), np.array(Ks))
    out["K_over_m_exponent"] = k; out["K0_extrapolated"] = K0
    out["paper"] = {"uniaxial_exponent": 2.95, "where": "P:52 (Callen-Callen: 3)"}
    return out


def c5(device="cuda:0", nx=2048, ny=2048, nz=4, sweeps=3000):
    mask, region, axes = inputs.voronoi_film(nx, ny, nz, 40, seed=42)
    g = binding.Lattice(nx, ny, nz, periodic=(1, 1, 0), Ku=0.02, bond_mask=mask, region=region, region_axis=axes,
                        cone0=0.5, adaptive=True, seed=42, device=device)
    Ts, m = [0.1 * k for k in range(1, 16)], []
    for T in Ts:                                              # increasing sweep, state and cone carried over
        g.sweep(T, sweeps - 1000); g.reset_accumulators(); g.sweep(T, 1000)
        ob = g.observables(); m.append(ob.sum_m[0] / ob.n_samples)
    g.close()
    out = {"config": f"c5 {nx}x{ny}x{nz} granular film, {axes.shape[0]} grains, Ku=0.02 per-grain axes, T=0.1..1.5, {sweeps} sweeps each", "T": Ts, "m": m}
    # Eq. (8): multi-Bloch fit of the film's m(T) (normalised to its lowest-T value: the random per-grain axes cap m
    # near 0.55) for an increasing number of terms; the weighted mean T_C is the film's average Curie temperature
    try:
        mm = np.array(m) / m[0]
        out["multi_bloch_mean_Tc"] = {str(nb): round(analysis.fit_multi_bloch(Ts, mm, nb)[3], 4) for nb in (1, 2, 4, 8)}
    except Exception as exc:                                  # a fit that does not converge must not lose the measured curve
        out["multi_bloch_mean_Tc"] = f"fit failed: {exc}"
    return out


def dw(device="cuda:0", shape=(160, 48, 48), Ku=0.05, temps=(0.2, 0.4, 0.6, 0.8, 0.9, 1.0, 1.1, 1.2), equil=3000, snapshots=300, every=10):
    """SURVEY 8f-1, the paper's domain-wall workload (Eq. (5), Fig. 2-3, Table I): a 180 degree wall held in the box by the
    anti-periodic boundary along x; per temperature the wall width Delta(T) from tanh fits of the slice profile m_z(x) (one fit per
    snapshot, the box re-centred on the wall first: it diffuses), the bulk m(T) from the same fits, K(T) from a constrained run at
    theta = 45 degrees on a periodic lattice, A(T) = K(T) Delta(T)^2 / pi^2 and the exponent k of A ~ m^k over m > 0.6
    (paper: 1.48 ... 1.79, rising with the anisotropy)."""
    nx, ny, nz = shape
    N = nx * ny * nz
    x = (np.arange(N) % nx).astype(np.float64)
    d0 = np.sqrt(1.0 / (2.0 * Ku))                            # T = 0 continuum wall parameter sqrt(A/K), A = J/2 per lattice spacing
    out = {"config": f"domain wall {nx}x{ny}x{nz}, anti-periodic x, Ku={Ku}, {equil} + {snapshots}x{every} sweeps per T", "points": []}
    ms, As = [], []
    for i, T in enumerate(temps):
        g = binding.Lattice(nx, ny, nz, periodic=(2, 1, 1), Ku=Ku, cone0=0.5, adaptive=True, seed=42 + i, device=device)
        S = np.zeros((N, 3)); S[:, 2] = np.tanh(-(x - (nx / 2 - 0.5)) / d0); S[:, 1] = np.sqrt(1.0 - S[:, 2] ** 2)
        g.set_spins(S.astype(np.float32)); g.sweep(T, equil)
        mfit, widths = [], []
        for _ in range(snapshots):
            g.sweep(T, every)
            mz = g.profile_x()[:, 2]
            c = int(np.argmin(np.abs(np.convolve(mz, np.ones(5) / 5, mode="same"))))      # the wall: where the smoothed profile crosses zero
            sft = (c - nx // 2) % nx
            mz = np.concatenate([mz[sft:], -mz[:sft]])        # re-centre; a slice that wraps the anti-periodic boundary changes sign
            try:
                m, _, D = analysis.fit_domain_wall(mz)
            except Exception:
                continue
            if 1.0 < D < nx / 2:
                mfit.append(m); widths.append(D)
        g.close()
        L = 32
        c4 = binding.Lattice(L, L, L, Ku=Ku, cone0=0.5, adaptive=True, seed=142 + i, device=device)
        c4.constrained_sweep(T, np.pi / 4, 0.0, 1500); c4.reset_accumulators(); c4.constrained_sweep(T, np.pi / 4, 0.0, 3000)
        ob = c4.observables(); c4.close()
        K = -ob.sum_torque[1] / ob.n_samples                  # tau_y = -K sin(2 theta), theta = 45 degrees
        D = float(np.mean(widths)); m = float(np.mean(mfit))
        A = analysis.exchange_stiffness(K, D)
        ms.append(m); As.append(A)
        out["points"].append({"T": T, "m_bulk": m, "Delta": D, "Delta_se": float(np.std(widths) / np.sqrt(len(widths))), "fits": len(widths),
                              "K": float(K), "A": float(A)})
    k, A0 = analysis.power_law_exponent(np.array(ms), np.array(As), m_min=0.6)
    out["A_over_m_exponent_m_gt_0.6"] = k; out["A0_extrapolated"] = A0
    out["expected_T0"] = {"Delta": float(np.pi * d0), "A": 0.5}
    out["paper"] = {"k": "1.48 +- 0.02 ... 1.79 +- 0.02 with rising anisotropy (Table I, P:90); mean field 2", "where": "P:76-90"}
    return out


def f4(device="cuda:0", L=48, Ku=0.05, temps=(0.2, 0.4, 0.6, 0.8, 1.0, 1.2), equil=3000, samples=300, every=20):
    """SURVEY 8f-4, the paper's second anisotropy route and its susceptibility check on observables the library already returns:
    Eq. (4) -- K(T)/K(0) from the easy-axis anisotropy energy of a STANDARD run -- against the constrained torque route
    ("identical results"), and Eq. (7) -- chi_perp = m^2 / (2 K(T)) -- against the transverse susceptibility of
    Eq. (6) accumulated by the same standard run."""
    out = {"config": f"f-4 {L}^3, Ku={Ku} along z, {equil} + {samples}x{every} sweeps per T (standard), 32^3 constrained at 45 deg", "points": []}
    for i, T in enumerate(temps):
        g = binding.Lattice(L, L, L, Ku=Ku, cone0=0.5, adaptive=True, seed=42 + i, device=device)
        g.sweep(T, equil); g.reset_accumulators()
        Ea = []
        for _ in range(samples):
            g.sweep(T, every); Ea.append(g.observables().E_aniso)
        ob = g.observables(); g.close()
        chi = analysis.susceptibilities(ob, T)
        m = ob.sum_m[0] / ob.n_samples
        k4 = analysis.anisotropy_scaling_easy_axis(float(np.mean(Ea)), Ku=Ku)
        c = binding.Lattice(32, 32, 32, Ku=Ku, cone0=0.5, adaptive=True, seed=142 + i, device=device)
        c.constrained_sweep(T, np.pi / 4, 0.0, 1500); c.reset_accumulators(); c.constrained_sweep(T, np.pi / 4, 0.0, 4000)
        oc = c.observables(); c.close()
        kt = -oc.sum_torque[1] / oc.n_samples / Ku
        out["points"].append({"T": T, "m": float(m), "k_eq4": float(k4), "k_torque": float(kt), "m^2.95": float(m ** 2.95),
                              "chi_perp_eq6": float(0.5 * (chi[1] + chi[2])), "chi_perp_eq7": float(analysis.chi_perp_uniaxial(m, Ku * k4)),
                              "chi_l": float(chi[0])})
    ms = np.array([p["m"] for p in out["points"]])
    out["exponent_eq4"] = analysis.power_law_exponent(ms, np.array([p["k_eq4"] for p in out["points"]]))[0]
    out["exponent_torque"] = analysis.power_law_exponent(ms, np.array([p["k_torque"] for p in out["points"]]))[0]
    # the cubic case of Eq. (4): k_c = 1 - 5 K_easy / (3 K_0,hard) from a standard run with Kc > 0 (easy axes <100>), against m^9.90
    cub = []
    for i, T in enumerate((0.1, 0.2, 0.3, 0.4, 0.6, 0.8)):
        g = binding.Lattice(L, L, L, Kc=Ku, cone0=0.5, adaptive=True, seed=242 + i, device=device)
        g.sweep(T, equil); g.reset_accumulators()
        Ea = []
        for _ in range(samples):
            g.sweep(T, every); Ea.append(g.observables().E_aniso)
        ob = g.observables(); g.close()
        m = ob.sum_m[0] / ob.n_samples
        cub.append({"T": T, "m": float(m), "k_eq4": float(analysis.anisotropy_scaling_easy_axis(float(np.mean(Ea)), Kc=Ku)), "m^9.90": float(m ** 9.90)})
    out["cubic"] = {"Kc": Ku, "points": cub,
                    "exponent_T_le_0.4": analysis.power_law_exponent(np.array([p["m"] for p in cub[:4]]), np.array([p["k_eq4"] for p in cub[:4]]))[0]}
    out["paper"] = {"uniaxial_exponent": 2.95, "cubic_exponent": 9.90, "where": "P:52-59, P:105"}
    return out


def main(argv=None):
    """python -m paper_2103_03517_b200.configs [c1 ...]; under torchrun the point loops of c2 / c4 are dealt over the ranks
    (replicas), the single-lattice configs run on rank 0 only."""
    names = (argv or sys.argv[1:]) or ["c1", "c2", "c3", "c4", "c5"]
    table = {"c1": c1, "c2": c2, "c3": c3, "c4": c4, "c5": c5, "dw": dw, "f4": f4}
    dist = replicas.init_distributed()
    rank, local_rank, _ = replicas.world()
    dev = f"cuda:{local_rank}"
    for n in names:
        t0 = time.perf_counter()
        if n in ("c2", "c4"):
            res = table[n](device=dev, dist=dist)
        else:
            res = table[n](device=dev) if rank == 0 else None
        _sync()
        if res is not None:
            res["wall_s"] = round(time.perf_counter() - t0, 2)
            print(json.dumps(res), flush=True)
    if dist is not None:
        dist.barrier(); dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
