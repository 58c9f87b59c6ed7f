"""ctypes driver for the fp64 serial oracle (oracle/mc_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs.  The product package never imports this module and this
module never imports the product package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mc_oracle.c")
_HDR = os.path.join(_HERE, "mc_oracle.h")
_LIB = os.path.join(_HERE, "liboracle_mc.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (no fast-math).  Building the checker is not using it."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        tmp = f"{_LIB}.{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-Wall", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class OrcObs(C.Structure):
    _fields_ = [
        ("n_sites", C.c_uint64), ("sweep", C.c_uint64),
        ("cone_rad", C.c_double), ("last_acceptance", C.c_double),
        ("M", C.c_double * 3), ("m", C.c_double),
        ("E_total", C.c_double), ("E_exch", C.c_double), ("E_aniso", C.c_double), ("E_zeeman", C.c_double),
        ("torque", C.c_double * 3),
        ("n_samples", C.c_uint64),
        ("sum_m", C.c_double * 4), ("sum_m2", C.c_double * 4),
        ("sum_E", C.c_double), ("sum_E2", C.c_double),
        ("sum_torque", C.c_double * 3),
    ]


_lib = None


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(build())
    vp, i32, i64, u64, dbl = C.c_void_p, C.c_int, C.c_int64, C.c_uint64, C.c_double
    L.orc_philox4x32_10.argtypes = [vp, vp, vp]; L.orc_philox4x32_10.restype = None
    L.orc_uniform.argtypes = [C.c_uint32]; L.orc_uniform.restype = dbl
    L.orc_uniform_azimuth.argtypes = [C.c_uint32, C.c_uint32]; L.orc_uniform_azimuth.restype = dbl
    L.orc_site_uniforms.argtypes = [vp, i32, i32, i32, i32, u64, vp, vp, vp]; L.orc_site_uniforms.restype = None
    L.orc_pair_uniforms.argtypes = [vp, i32, i32, i32, i32, u64, vp, vp, vp]; L.orc_pair_uniforms.restype = None
    L.orc_cone_move.argtypes = [vp, dbl, dbl, dbl, vp]; L.orc_cone_move.restype = None
    L.orc_create.argtypes = [i32, i32, i32, vp, dbl, dbl, vp, dbl, vp, vp, vp, vp, i32, dbl, i32, u64]
    L.orc_create.restype = vp
    L.orc_create_bcc.argtypes = [i32, i32, i32, vp, dbl, dbl, vp, dbl, vp, dbl, i32, u64]
    L.orc_create_bcc.restype = vp
    L.orc_create_fcc.argtypes = [i32, i32, i32, vp, dbl, dbl, vp, dbl, vp, dbl, i32, u64]
    L.orc_create_fcc.restype = vp
    L.orc_create_basis.argtypes = [i32, i32, i32, i32, dbl, dbl, dbl, vp, dbl, vp, dbl, i32, u64]
    L.orc_create_basis.restype = vp
    L.orc_destroy.argtypes = [vp]; L.orc_destroy.restype = None
    for name in ("orc_set_spins", "orc_set_spins_f32", "orc_get_spins", "orc_init_uniform"):
        getattr(L, name).argtypes = [vp, vp]; getattr(L, name).restype = None
    L.orc_init_random.argtypes = [vp]; L.orc_init_random.restype = None
    L.orc_set_cone.argtypes = [vp, dbl]; L.orc_set_cone.restype = None
    L.orc_set_sweep.argtypes = [vp, u64]; L.orc_set_sweep.restype = None
    L.orc_set_adaptive.argtypes = [vp, i32]; L.orc_set_adaptive.restype = None
    L.orc_set_sampling.argtypes = [vp, i32]; L.orc_set_sampling.restype = None
    L.orc_half_sweep.argtypes = [vp, dbl, i32, vp, vp]; L.orc_half_sweep.restype = i64
    L.orc_end_sweep.argtypes = [vp, i64]; L.orc_end_sweep.restype = None
    L.orc_sweep.argtypes = [vp, dbl, i64]; L.orc_sweep.restype = None
    L.orc_sweep_random_order.argtypes = [vp, dbl, i64]; L.orc_sweep_random_order.restype = None
    L.orc_pairing.argtypes = [vp, u64, i32, vp, vp]; L.orc_pairing.restype = i32
    L.orc_site_of.argtypes = [vp, i32, i64]; L.orc_site_of.restype = i64
    L.orc_align_to.argtypes = [vp, vp]; L.orc_align_to.restype = i32
    L.orc_constrained_half_sweep.argtypes = [vp, dbl, vp, i32, vp, i32, i32, vp, vp]
    L.orc_constrained_half_sweep.restype = i64
    L.orc_constrained_sweep.argtypes = [vp, dbl, dbl, dbl, i64, i32, i32]; L.orc_constrained_sweep.restype = i32
    L.orc_observables.argtypes = [vp, vp]; L.orc_observables.restype = None
    L.orc_reset_accumulators.argtypes = [vp]; L.orc_reset_accumulators.restype = None
    L.orc_trace.argtypes = [vp, i64, vp]; L.orc_trace.restype = i64
    L.orc_site_energy.argtypes = [vp, i64, vp]; L.orc_site_energy.restype = dbl
    L.orc_total_energy.argtypes = [vp]; L.orc_total_energy.restype = dbl
    L.orc_profile_x.argtypes = [vp, vp]; L.orc_profile_x.restype = None
    _lib = L
    return L


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32); k = np.asarray(key, dtype=np.uint32); o = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(_p(c), _p(k), _p(o))
    return o


def uniform(r: int) -> float:
    return lib().orc_uniform(int(r) & 0xFFFFFFFF)


def uniform_azimuth(w0: int, w1: int) -> float:
    return lib().orc_uniform_azimuth(int(w0) & 0xFFFFFFFF, int(w1) & 0xFFFFFFFF)


def cone_move(S, theta, u0, u1):
    s = np.ascontiguousarray(S, dtype=np.float64); o = np.zeros(3)
    lib().orc_cone_move(_p(s), float(theta), float(u0), float(u1), _p(o))
    return o


class Oracle:
    """One lattice + Hamiltonian + RNG seed, state in fp64 (lexicographic [N,3])."""

    def __init__(self, nx, ny, nz, periodic=(1, 1, 1), J=1.0, Ku=0.0, eu=(0, 0, 1), Kc=0.0, B=(0, 0, 0),
                 bond_mask=None, region=None, region_axis=None, cone0=0.5, adaptive=True, seed=42, structure="sc", J2=0.0):
        self.L = lib()
        self.shape = (nx, ny, nz)
        self.structure = structure
        self.N = nx * ny * nz * {"sc": 1, "bcc": 2, "fcc": 4, "hcp": 8, "sc_nnn": 8}[structure]
        per = np.asarray(periodic, dtype=np.int32)
        eu_ = np.asarray(eu, dtype=np.float64); B_ = np.asarray(B, dtype=np.float64)
        if structure in ("bcc", "fcc"):   # sc sublattices = colours; site = sublattice*nx*ny*nz + cell (readings C-30, C-31)
            if bond_mask is not None or region is not None:
                raise ValueError("bcc / fcc mode has no bond mask / regions")
            self._mask = self._region = self._axis = None
            make = self.L.orc_create_bcc if structure == "bcc" else self.L.orc_create_fcc
            self.h = make(nx, ny, nz, _p(per), J, Ku, _p(eu_), Kc, _p(B_), float(cone0), int(bool(adaptive)), int(seed))
            if not self.h:
                raise ValueError("orc_create_bcc / orc_create_fcc rejected the lattice")
            return
        if structure in ("hcp", "sc_nnn"):   # eight non-interacting subsets (reading C-32): nx x ny x nz periodic cells of eight sites
            if bond_mask is not None or region is not None or tuple(int(v) for v in periodic) != (1, 1, 1):
                raise ValueError("hcp / sc_nnn mode: periodic boxes without bond mask / regions")
            self._mask = self._region = self._axis = None
            self.h = self.L.orc_create_basis(3 if structure == "hcp" else 4, nx, ny, nz, J, J2, Ku, _p(eu_), Kc, _p(B_),
                                             float(cone0), int(bool(adaptive)), int(seed))
            if not self.h:
                raise ValueError("orc_create_basis rejected the lattice")
            return
        if structure != "sc":
            raise ValueError("structure must be 'sc', 'bcc', 'fcc', 'hcp' or 'sc_nnn'")
        self._mask = None if bond_mask is None else np.ascontiguousarray(bond_mask, dtype=np.uint8).ravel()
        self._region = None if region is None else np.ascontiguousarray(region, dtype=np.uint16).ravel()
        self._axis = None if region_axis is None else np.ascontiguousarray(region_axis, dtype=np.float64)
        nreg = 0 if self._axis is None else self._axis.shape[0]
        self.h = self.L.orc_create(nx, ny, nz, _p(per), J, Ku, _p(eu_), Kc, _p(B_),
                                   _p(self._mask), _p(self._region), _p(self._axis), nreg,
                                   float(cone0), int(bool(adaptive)), int(seed))
        if not self.h:
            raise ValueError("orc_create rejected the lattice (periodic dims must be even)")

    def __del__(self):
        if getattr(self, "h", None):
            self.L.orc_destroy(self.h); self.h = None

    def site_uniforms(self, x, y, z, colour, sweep):
        """(u0, u1, u2) of the unconstrained update of site (x,y,z) in the given sweep (reading C-26)."""
        u = [C.c_double(), C.c_double(), C.c_double()]
        self.L.orc_site_uniforms(self.h, int(x), int(y), int(z), int(colour), int(sweep), C.byref(u[0]), C.byref(u[1]), C.byref(u[2]))
        return tuple(v.value for v in u)

    def init_random(self): self.L.orc_init_random(self.h)

    def profile_x(self):
        """[nx, 3] slice-averaged magnetisation along x (Fig. 2)."""
        out = np.zeros((self.shape[0], 3)); self.L.orc_profile_x(self.h, _p(out)); return out

    def pair_uniforms(self, x, y, z, colour, sweep):
        """(u0, u1, u2) of the constrained move of the pair led by site (x,y,z) (stream TAG_PAIR, reading C-26)."""
        u = [C.c_double(), C.c_double(), C.c_double()]
        self.L.orc_pair_uniforms(self.h, int(x), int(y), int(z), int(colour), int(sweep), C.byref(u[0]), C.byref(u[1]), C.byref(u[2]))
        return tuple(v.value for v in u)

    # ---- state
    def set_spins(self, xyz):
        a = np.ascontiguousarray(xyz)
        if a.dtype == np.float32:
            self.L.orc_set_spins_f32(self.h, _p(a.reshape(-1)))
        else:
            a = a.astype(np.float64, copy=False); self.L.orc_set_spins(self.h, _p(a.reshape(-1)))

    def get_spins(self):
        out = np.empty((self.N, 3)); self.L.orc_get_spins(self.h, _p(out)); return out

    def init_uniform(self, d):
        v = np.asarray(d, dtype=np.float64); self.L.orc_init_uniform(self.h, _p(v))

    def set_cone(self, c): self.L.orc_set_cone(self.h, float(c))
    def set_sweep(self, s): self.L.orc_set_sweep(self.h, int(s))
    def set_adaptive(self, a): self.L.orc_set_adaptive(self.h, int(bool(a)))
    def set_sampling(self, on): self.L.orc_set_sampling(self.h, int(bool(on)))

    # ---- Table A1
    def half_sweep(self, T, colour, want_detail=False):
        if want_detail:
            x = np.full(self.N, np.nan); acc = np.zeros(self.N, np.uint8)
            n = self.L.orc_half_sweep(self.h, float(T), int(colour), _p(x), _p(acc))
            return n, x, acc
        return self.L.orc_half_sweep(self.h, float(T), int(colour), None, None)

    def end_sweep(self, count): self.L.orc_end_sweep(self.h, int(count))
    def sweep(self, T, n=1): self.L.orc_sweep(self.h, float(T), int(n))
    def sweep_random_order(self, T, n=1): self.L.orc_sweep_random_order(self.h, float(T), int(n))

    # ---- Table A2
    def pairing(self, sweep, colour):
        Nc = self.N // 2
        partner = np.full(Nc, -1, np.int64); lead = np.zeros(Nc, np.uint8)
        rc = self.L.orc_pairing(self.h, int(sweep), int(colour), _p(partner), _p(lead))
        if rc:
            raise ValueError("pairing undefined (odd colour population)")
        return partner, lead

    def site_of(self, colour, a): return self.L.orc_site_of(self.h, int(colour), int(a))

    def align_to(self, eC):
        v = np.asarray(eC, dtype=np.float64); return self.L.orc_align_to(self.h, _p(v))

    def constrained_half_sweep(self, T, eC, colour, ML, ml_mode=0, pairing_mode=0, want_detail=False):
        v = np.asarray(eC, dtype=np.float64); ml = C.c_double(ML)
        x = acc = None
        if want_detail:
            x = np.full(self.N, np.nan); acc = np.zeros(self.N, np.uint8)
        n = self.L.orc_constrained_half_sweep(self.h, float(T), _p(v), int(colour), C.byref(ml),
                                              int(ml_mode), int(pairing_mode), _p(x), _p(acc))
        return (n, ml.value, x, acc) if want_detail else (n, ml.value)

    def constrained_sweep(self, T, theta, phi, n=1, ml_mode=0, pairing_mode=0):
        rc = self.L.orc_constrained_sweep(self.h, float(T), float(theta), float(phi), int(n), int(ml_mode), int(pairing_mode))
        if rc:
            raise ValueError("constrained sweep rejected (|M| too small, M.eC <= 0 or odd colour population)")

    # ---- read-out
    def observables(self):
        o = OrcObs(); self.L.orc_observables(self.h, C.byref(o)); return o

    def reset_accumulators(self): self.L.orc_reset_accumulators(self.h)

    def trace(self, max_rows=None):
        have = int(self.observables().sweep)
        max_rows = max(1, have if max_rows is None else min(int(max_rows), have))
        rows = np.empty((max_rows, 6)); k = self.L.orc_trace(self.h, int(max_rows), _p(rows)); return rows[:k].copy()

    def site_energy(self, site, S):
        v = np.ascontiguousarray(S, dtype=np.float64); return self.L.orc_site_energy(self.h, int(site), _p(v))

    def total_energy(self): return self.L.orc_total_energy(self.h)
