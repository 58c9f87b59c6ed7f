"""Thin ctypes binding over libmc_b200.so -- same names as include/mc.h, argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used for exactly two things: the device
workspace (a ``torch.empty(..., dtype=torch.uint8, device="cuda")``) and the CUDA stream.  If the shared library is
missing this module raises: there is no CPU fallback and the oracle is never imported from here.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmc_b200.so")

MC_OK, MC_EINVAL, MC_ECUDA, MC_ESTATE = 0, -1, -2, -3
MC_TRACE_CAPACITY = 16384
MC_PATH_AUTO, MC_PATH_GENERIC, MC_PATH_STAGED, MC_PATH_MARCH = 0, 1, 2, 3
MC_SC, MC_BCC, MC_FCC, MC_HCP, MC_SC_NNN = 0, 1, 2, 3, 4
STRUCTURES = {"sc": (MC_SC, 1), "bcc": (MC_BCC, 2), "fcc": (MC_FCC, 4), "hcp": (MC_HCP, 8), "sc_nnn": (MC_SC_NNN, 8)}   # id, spins per cell

# every symbol include/mc.h declares (tests/test_abi.py checks the header against this list and the .so)
SYMBOLS = [
    "mc_workspace_bytes", "mc_create", "mc_destroy", "mc_init_spins", "mc_set_spins", "mc_get_spins", "mc_set_cone",
    "mc_set_sweep", "mc_sweep", "mc_constrained_sweep", "mc_half_sweep", "mc_constrained_half_sweep", "mc_end_sweep",
    "mc_align_to", "mc_observables", "mc_reset_accumulators", "mc_trace", "mc_profile_x", "mc_profile_x_static", "mc_debug_set_path", "mc_debug_get_path", "mc_launch_count", "mc_last_error", "mc_version",
]


class McLattice(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("periodic", C.c_int32 * 3), ("structure", C.c_int32)]


class McHamiltonian(C.Structure):
    _fields_ = [
        ("J", C.c_double), ("Ku", C.c_double), ("eu", C.c_double * 3), ("Kc", C.c_double), ("B", C.c_double * 3),
        ("bond_mask", C.c_void_p), ("region", C.c_void_p), ("region_axis", C.c_void_p), ("n_regions", C.c_int32),
        ("cone0_rad", C.c_double), ("adaptive", C.c_int32), ("J2", C.c_double),
    ]


class McObs(C.Structure):
    _fields_ = [
        ("n_sites", C.c_uint64), ("sweep", C.c_uint64), ("cone_rad", C.c_double), ("last_acceptance", C.c_double),
        ("M", C.c_double * 3), ("m", C.c_double),
        ("E_total", C.c_double), ("E_exch", C.c_double), ("E_aniso", C.c_double), ("E_zeeman", C.c_double),
        ("torque", C.c_double * 3), ("n_samples", C.c_uint64),
        ("sum_m", C.c_double * 4), ("sum_m2", C.c_double * 4), ("sum_E", C.c_double), ("sum_E2", C.c_double),
        ("sum_torque", C.c_double * 3),
    ]


class McError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libmc_b200 error {code}: {msg}")
        self.code = code


_lib = None


def load():
    """Loads libmc_b200.so (built in-tree by paper_2103_03517_b200.build); fails loudly if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2103_03517_b200.build` (nvcc, sm_100a). "
                           "There is no CPU fallback.")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, u64, dbl, sz = C.c_void_p, C.c_int, C.c_int64, C.c_uint64, C.c_double, C.c_size_t
    L.mc_workspace_bytes.argtypes = [vp, vp]; L.mc_workspace_bytes.restype = sz
    L.mc_create.argtypes = [vp, vp, u64, vp, sz, vp, vp]; L.mc_create.restype = i32
    L.mc_destroy.argtypes = [vp]; L.mc_destroy.restype = i32
    L.mc_init_spins.argtypes = [vp, i32, vp]; L.mc_init_spins.restype = i32
    L.mc_set_spins.argtypes = [vp, vp]; L.mc_set_spins.restype = i32
    L.mc_get_spins.argtypes = [vp, vp]; L.mc_get_spins.restype = i32
    L.mc_set_cone.argtypes = [vp, dbl]; L.mc_set_cone.restype = i32
    L.mc_set_sweep.argtypes = [vp, u64]; L.mc_set_sweep.restype = i32
    L.mc_sweep.argtypes = [vp, dbl, i64]; L.mc_sweep.restype = i32
    L.mc_constrained_sweep.argtypes = [vp, dbl, dbl, dbl, i64]; L.mc_constrained_sweep.restype = i32
    L.mc_half_sweep.argtypes = [vp, dbl, i32, vp, vp]; L.mc_half_sweep.restype = i32
    L.mc_constrained_half_sweep.argtypes = [vp, dbl, dbl, dbl, i32, dbl, vp, vp]; L.mc_constrained_half_sweep.restype = i32
    L.mc_end_sweep.argtypes = [vp]; L.mc_end_sweep.restype = i32
    L.mc_align_to.argtypes = [vp, dbl, dbl]; L.mc_align_to.restype = i32
    L.mc_observables.argtypes = [vp, vp]; L.mc_observables.restype = i32
    L.mc_reset_accumulators.argtypes = [vp]; L.mc_reset_accumulators.restype = i32
    L.mc_trace.argtypes = [vp, i64, vp, vp]; L.mc_trace.restype = i32
    L.mc_profile_x.argtypes = [vp, vp]; L.mc_profile_x.restype = i32
    L.mc_profile_x_static.argtypes = [vp, vp]; L.mc_profile_x_static.restype = i32
    L.mc_debug_set_path.argtypes = [vp, i32]; L.mc_debug_set_path.restype = i32
    L.mc_debug_get_path.argtypes = [vp]; L.mc_debug_get_path.restype = i32
    L.mc_launch_count.argtypes = [vp]; L.mc_launch_count.restype = i64
    L.mc_last_error.argtypes = [vp]; L.mc_last_error.restype = C.c_char_p
    L.mc_version.argtypes = []; L.mc_version.restype = C.c_char_p
    _lib = L
    return L


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def make_structs(shape, periodic=(1, 1, 1), J=1.0, Ku=0.0, eu=(0, 0, 1), Kc=0.0, B=(0, 0, 0),
                 bond_mask=None, region=None, region_axis=None, cone0=0.5, adaptive=True, structure="sc", J2=0.0):
    """Fills mc_lattice / mc_hamiltonian; returns them plus the arrays that must stay alive during mc_create."""
    lat = McLattice(int(shape[0]), int(shape[1]), int(shape[2]), (C.c_int32 * 3)(*[int(p) for p in periodic]),   # 0 open, 1 periodic, 2 anti-periodic (x)
                    STRUCTURES[structure][0])
    keep = []
    def arr(a, dt):
        if a is None:
            return None
        v = np.ascontiguousarray(a, dtype=dt); keep.append(v); return v.ctypes.data
    ham = McHamiltonian()
    ham.J = float(J); ham.Ku = float(Ku); ham.eu = (C.c_double * 3)(*[float(v) for v in eu]); ham.Kc = float(Kc)
    ham.B = (C.c_double * 3)(*[float(v) for v in B])
    ham.bond_mask = arr(None if bond_mask is None else np.asarray(bond_mask).ravel(), np.uint8)
    ham.region = arr(None if region is None else np.asarray(region).ravel(), np.uint16)
    ham.region_axis = arr(region_axis, np.float64)
    ham.n_regions = 0 if region_axis is None else int(np.asarray(region_axis).shape[0])
    ham.cone0_rad = float(cone0); ham.adaptive = int(bool(adaptive)); ham.J2 = float(J2)
    return lat, ham, keep


class Lattice:
    """One handle = one lattice + Hamiltonian + seed on one CUDA stream.  Methods mirror include/mc.h one to one."""

    def __init__(self, nx, ny, nz, periodic=(1, 1, 1), J=1.0, Ku=0.0, eu=(0, 0, 1), Kc=0.0, B=(0, 0, 0),
                 bond_mask=None, region=None, region_axis=None, cone0=0.5, adaptive=True, seed=42,
                 device="cuda:0", stream=None, structure="sc", guard_bytes=0, J2=0.0):
        import torch  # device memory and streams only
        self.L = load()
        self.shape = (int(nx), int(ny), int(nz))
        self.N = int(nx) * int(ny) * int(nz) * STRUCTURES[structure][1]                        # spins per cell
        self.h = None
        lat, ham, keep = make_structs(self.shape, periodic, J, Ku, eu, Kc, B, bond_mask, region, region_axis, cone0, adaptive, structure, J2)
        nbytes = self.L.mc_workspace_bytes(C.byref(lat), C.byref(ham))
        if nbytes == 0:
            raise McError(MC_EINVAL, "mc_workspace_bytes rejected the lattice / Hamiltonian")
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            # guard_bytes > 0 (tests): the workspace sits between two canary zones that check_guards() verifies -- an
            # out-of-bounds write of any kernel shows up there (compute-sanitizer is not available on every pool)
            g = (int(guard_bytes) + 255) // 256 * 256
            self._alloc = torch.empty(nbytes + 2 * g, dtype=torch.uint8, device=self.device)
            if g:
                self._alloc[:g] = 0xA5; self._alloc[g + nbytes:] = 0xA5
            self._guard = g
            self.workspace = self._alloc[g: g + nbytes]
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            out = C.c_void_p()
            rc = self.L.mc_create(C.byref(lat), C.byref(ham), int(seed), self.workspace.data_ptr(), nbytes,
                                  self.stream.cuda_stream, C.byref(out))
        if rc != MC_OK:
            raise McError(rc, "mc_create failed (see stderr)")
        self.h = out
        self.workspace_bytes = nbytes

    def check_guards(self):
        """True if no byte of the canary zones around the workspace has been written (guard_bytes > 0)."""
        import torch
        torch.cuda.synchronize(self.device)
        g, n = self._guard, self.workspace_bytes
        return bool((self._alloc[:g] == 0xA5).all().item()) and bool((self._alloc[g + n:] == 0xA5).all().item())

    def _chk(self, rc):
        if rc != MC_OK:
            raise McError(rc, self.L.mc_last_error(self.h).decode())

    def close(self):
        if self.h:
            self.L.mc_destroy(self.h); self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- state
    def init_spins(self, mode=0, direction=(0, 0, 1)):
        d = np.asarray(direction, dtype=np.float64); self._chk(self.L.mc_init_spins(self.h, int(mode), _p(d)))

    def set_spins(self, xyz):
        a = np.ascontiguousarray(xyz, dtype=np.float32).reshape(-1)
        assert a.size == 3 * self.N
        self._chk(self.L.mc_set_spins(self.h, _p(a)))

    def get_spins(self):
        out = np.empty((self.N, 3), dtype=np.float32); self._chk(self.L.mc_get_spins(self.h, _p(out))); return out

    def set_cone(self, cone): self._chk(self.L.mc_set_cone(self.h, float(cone)))
    def set_sweep(self, sweep): self._chk(self.L.mc_set_sweep(self.h, int(sweep)))

    # ---- the hot path
    def sweep(self, T, n=1): self._chk(self.L.mc_sweep(self.h, float(T), int(n)))

    def constrained_sweep(self, T, theta, phi, n=1):
        self._chk(self.L.mc_constrained_sweep(self.h, float(T), float(theta), float(phi), int(n)))

    # ---- test hooks
    def half_sweep(self, T, colour, want_detail=False):
        if not want_detail:
            self._chk(self.L.mc_half_sweep(self.h, float(T), int(colour), None, None)); return None
        x = np.full(self.N, np.nan, dtype=np.float32); acc = np.zeros(self.N, dtype=np.uint8)
        self._chk(self.L.mc_half_sweep(self.h, float(T), int(colour), _p(x), _p(acc)))
        return x, acc

    def constrained_half_sweep(self, T, theta, phi, colour, ML, want_detail=False):
        x = acc = None
        if want_detail:
            x = np.full(self.N, np.nan, dtype=np.float32); acc = np.zeros(self.N, dtype=np.uint8)
        self._chk(self.L.mc_constrained_half_sweep(self.h, float(T), float(theta), float(phi), int(colour), float(ML), _p(x), _p(acc)))
        return (x, acc) if want_detail else None

    def end_sweep(self): self._chk(self.L.mc_end_sweep(self.h))
    def align_to(self, theta, phi): self._chk(self.L.mc_align_to(self.h, float(theta), float(phi)))

    # ---- read-out
    def observables(self):
        o = McObs(); self._chk(self.L.mc_observables(self.h, C.byref(o))); return o

    def reset_accumulators(self): self._chk(self.L.mc_reset_accumulators(self.h))

    def profile_x(self):
        """[nx, 3] slice-averaged magnetisation along x (mc_profile_x; Fig. 2)."""
        out = np.empty((self.shape[0], 3)); self._chk(self.L.mc_profile_x(self.h, _p(out))); return out

    def profile_x_static(self, out=None):
        """mc_profile_x_static: the same profile with its scratch in a fixed array of the library (no allocation; nx <= 8192).
        ``out``: a caller-owned C-contiguous float64 [nx, 3] array to fill (a new one if None)."""
        if out is None: out = np.empty((self.shape[0], 3))
        assert out.dtype == np.float64 and out.flags.c_contiguous and out.size == 3 * self.shape[0]
        self._chk(self.L.mc_profile_x_static(self.h, _p(out))); return out

    def trace(self, max_rows=MC_TRACE_CAPACITY):
        rows = np.empty((int(max_rows), 6)); k = C.c_int64(0)
        self._chk(self.L.mc_trace(self.h, int(max_rows), _p(rows), C.byref(k)))
        return rows[: k.value].copy()

    def debug_set_path(self, path): self._chk(self.L.mc_debug_set_path(self.h, int(path)))
    def debug_get_path(self): return int(self.L.mc_debug_get_path(self.h))
    def launch_count(self): return int(self.L.mc_launch_count(self.h))
