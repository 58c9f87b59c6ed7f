"""Seeded synthetic input generators (NumPy only).

This module holds NONE of the method's arithmetic: no Philox, no cone move, no energies.  It only
manufactures inputs -- initial spin states, bond masks, grain maps -- that are handed, unchanged, to both
the CUDA library (through the C ABI) and the CPU oracle (tests only).  It imports neither of them.

Recipes follow DESIGN.md section 6 (which restates BASELINE.json's configs as concrete inputs).
"""
from __future__ import annotations

import numpy as np

# bond-mask bit k: (+x, -x, +y, -y, +z, -z)   (include/mc.h)
_DIRS = ((0, +1), (0, -1), (1, +1), (1, -1), (2, +1), (2, -1))


def random_unit_spins(n_sites: int, seed: int, dtype=np.float32) -> np.ndarray:
    """Spins uniform on the sphere (config c3, P:9 ">10 million spins"): z = 2u-1, phi = 2 pi v.

    Computed in fp64, cast to fp32, renormalised in fp32 so that the stored state is unit to 1 ulp."""
    rng = np.random.default_rng(seed)
    z = 2.0 * rng.random(n_sites) - 1.0
    phi = 2.0 * np.pi * rng.random(n_sites)
    r = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    s = np.stack([r * np.cos(phi), r * np.sin(phi), z], axis=1)
    s = s.astype(dtype)
    s /= np.linalg.norm(s.astype(np.float64), axis=1, keepdims=True).astype(dtype)
    return np.ascontiguousarray(s)


def uniform_spins(n_sites: int, direction=(0.0, 0.0, 1.0), dtype=np.float32) -> np.ndarray:
    d = np.asarray(direction, dtype=np.float64)
    d = d / np.linalg.norm(d)
    return np.ascontiguousarray(np.broadcast_to(d.astype(dtype), (n_sites, 3)).copy())


def thermal_like_spins(n_sites: int, seed: int, spread: float, direction=(0.0, 0.0, 1.0), dtype=np.float32) -> np.ndarray:
    """Unit spins scattered about ``direction`` (Gaussian transverse kicks of width ``spread``): an ordered,
    low-temperature-looking state for parity tests at small T without running an equilibration."""
    rng = np.random.default_rng(seed)
    d = np.asarray(direction, dtype=np.float64)
    d = d / np.linalg.norm(d)
    s = d[None, :] + spread * rng.standard_normal((n_sites, 3))
    s /= np.linalg.norm(s, axis=1, keepdims=True)
    s = s.astype(dtype)
    s /= np.linalg.norm(s.astype(np.float64), axis=1, keepdims=True).astype(dtype)
    return np.ascontiguousarray(s)


def site_coords(nx: int, ny: int, nz: int):
    """Lexicographic site -> (x, y, z), x fastest."""
    s = np.arange(nx * ny * nz, dtype=np.int64)
    return s % nx, (s // nx) % ny, s // (nx * ny)


def boundary_mask(nx: int, ny: int, nz: int, periodic) -> np.ndarray:
    """6-bit bond mask that only encodes the boundary conditions (bit set = bond present)."""
    x, y, z = site_coords(nx, ny, nz)
    pos, dim = (x, y, z), (nx, ny, nz)
    mask = np.zeros(nx * ny * nz, dtype=np.uint8)
    for k, (axis, step) in enumerate(_DIRS):
        q = pos[axis] + step
        ok = np.ones_like(q, dtype=bool) if periodic[axis] else (q >= 0) & (q < dim[axis])
        mask |= (ok.astype(np.uint8) << k)
    return mask


def random_bond_mask(nx: int, ny: int, nz: int, periodic, seed: int, p_cut: float = 0.2) -> np.ndarray:
    """Symmetric random dilution of the bonds allowed by the boundary conditions (parity-test input)."""
    rng = np.random.default_rng(seed)
    x, y, z = site_coords(nx, ny, nz)
    pos, dim = [x, y, z], (nx, ny, nz)
    mask = boundary_mask(nx, ny, nz, periodic)
    for axis in range(3):
        cut = rng.random(nx * ny * nz) < p_cut            # decision attached to the bond's lower end, + direction
        kp, km = 2 * axis, 2 * axis + 1
        q = [p.copy() for p in pos]
        q[axis] = (q[axis] + 1) % dim[axis]
        nb = q[0] + nx * (q[1] + ny * q[2])
        has = ((mask >> kp) & 1).astype(bool)
        cut &= has
        if dim[axis] == 2 and periodic[axis]:
            # the +x and -x bonds of a site join the same pair of sites: cut them together to stay symmetric
            lower = pos[axis] == 0
            cut_pair = cut & lower
            for sites in (np.nonzero(cut_pair)[0], nb[cut_pair]):
                mask[sites] &= np.uint8(~((1 << kp) | (1 << km)) & 0xFF)
            continue
        mask[cut] &= np.uint8(~(1 << kp) & 0xFF)
        mask[nb[cut]] &= np.uint8(~(1 << km) & 0xFF)
    return mask


def voronoi_film(nx: int, ny: int, nz: int, mean_diameter: float, seed: int):
    """Granular thin film of config c5 (BASELINE.json configs[4]; reading C-21).

    Poisson-seeded 2-D Voronoi tessellation, in-plane periodic (minimum-image distance), columnar through
    the nz layers; open top and bottom.  Returns (bond_mask[N] uint8, region[N] uint16, region_axis[n,3] f64):
    bonds across a grain boundary or through an open face are cut (J = 0 across), and every grain gets an
    easy axis drawn uniformly on the sphere."""
    rng = np.random.default_rng(seed)
    n_seeds = max(1, int(round(nx * ny / (np.pi * mean_diameter ** 2 / 4.0))))
    if n_seeds > 65535:
        raise ValueError("more than 65535 grains do not fit the uint16 region id")
    px = rng.random(n_seeds) * nx
    py = rng.random(n_seeds) * ny
    zz = 2.0 * rng.random(n_seeds) - 1.0
    ph = 2.0 * np.pi * rng.random(n_seeds)
    rr = np.sqrt(1.0 - zz * zz)
    axes = np.stack([rr * np.cos(ph), rr * np.sin(ph), zz], axis=1)

    # nearest seed under the in-plane minimum-image metric: bucket the seeds on a coarse grid and search 3x3 cells
    cell = max(4.0, float(mean_diameter))
    gx, gy = max(1, int(nx // cell)), max(1, int(ny // cell))
    cw, ch = nx / gx, ny / gy
    buckets = [[[] for _ in range(gy)] for _ in range(gx)]
    for s in range(n_seeds):
        buckets[int(px[s] // cw) % gx][int(py[s] // ch) % gy].append(s)
    grain2d = np.empty((ny, nx), dtype=np.int64)
    reach = 1
    while True:
        ok = True
        for bx in range(gx):
            x0, x1 = int(np.ceil(bx * cw)), min(nx, int(np.ceil((bx + 1) * cw)))
            for by in range(gy):
                y0, y1 = int(np.ceil(by * ch)), min(ny, int(np.ceil((by + 1) * ch)))
                cand = []
                for dx in range(-reach, reach + 1):
                    for dy in range(-reach, reach + 1):
                        cand += buckets[(bx + dx) % gx][(by + dy) % gy]
                if not cand:
                    ok = False
                    break
                cand = np.unique(np.asarray(cand))
                X = np.arange(x0, x1)[None, :, None] + 0.5
                Y = np.arange(y0, y1)[:, None, None] + 0.5
                ddx = np.abs(X - px[cand][None, None, :]); ddx = np.minimum(ddx, nx - ddx)
                ddy = np.abs(Y - py[cand][None, None, :]); ddy = np.minimum(ddy, ny - ddy)
                d2 = ddx * ddx + ddy * ddy
                best = d2.argmin(axis=2)
                # the 3x3 (or wider) neighbourhood is exhaustive only if the winner is closer than its margin
                if np.sqrt(d2.min(axis=2)).max() > reach * min(cw, ch):
                    ok = False
                    break
                grain2d[y0:y1, x0:x1] = cand[best]
            if not ok:
                break
        if ok:
            break
        reach += 1
        if reach > max(gx, gy):
            raise RuntimeError("voronoi search did not converge")

    region = np.broadcast_to(grain2d[None, :, :], (nz, ny, nx)).reshape(-1).astype(np.uint16)
    periodic = (1, 1, 0)
    mask = boundary_mask(nx, ny, nz, periodic)
    x, y, z = site_coords(nx, ny, nz)
    pos, dim = [x, y, z], (nx, ny, nz)
    for k, (axis, step) in enumerate(_DIRS):
        q = [p.copy() for p in pos]
        q[axis] = (q[axis] + step) % dim[axis]
        nb = q[0] + nx * (q[1] + ny * q[2])
        same = region[nb] == region
        mask &= np.where(same, np.uint8(0xFF), np.uint8(~(1 << k) & 0xFF))
    return mask, np.ascontiguousarray(region), np.ascontiguousarray(axes)
