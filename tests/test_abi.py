"""The C-ABI library loads on a CPU-only box and exports every symbol include/mc.h declares (no compute calls)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2103_03517_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "mc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mc_[a-z_]+)\s*\(", text)))


def test_header_and_binding_list_the_same_symbols():
    assert _declared_symbols() == sorted(binding.SYMBOLS)


def test_library_exports_every_declared_symbol(lib):
    for name in _declared_symbols():
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.mc_version()


def test_struct_sizes_match_the_header_layout():
    assert C.sizeof(binding.McLattice) == 28
    assert C.sizeof(binding.McHamiltonian) == 8 + 8 + 24 + 8 + 24 + 8 + 8 + 8 + 8 + 8 + 8 + 8
    assert C.sizeof(binding.McObs) == 8 * (2 + 2 + 3 + 1 + 4 + 3 + 1 + 4 + 4 + 2 + 3)


def test_workspace_sizing_and_argument_validation_run_on_the_host(lib):
    lat, ham, _ = binding.make_structs((224, 224, 224), Kc=0.01)
    n = lib.mc_workspace_bytes(C.byref(lat), C.byref(ham))
    assert 224 ** 3 * 24 <= n <= 224 ** 3 * 24 + (8 << 20)          # 12 B/spin of state + 12 B/spin of staging + small fixed overhead
    mask = np.zeros(16 * 16 * 4, np.uint8); region = np.zeros(16 * 16 * 4, np.uint16)
    lat2, ham2, _k = binding.make_structs((16, 16, 4), periodic=(1, 1, 0), Ku=0.02, bond_mask=mask, region=region, region_axis=np.eye(3))
    n2 = lib.mc_workspace_bytes(C.byref(lat2), C.byref(ham2))
    assert n2 > 16 * 16 * 4 * 15
    for shape, per in (((7, 4, 4), (1, 1, 1)), ((8, 3, 4), (1, 1, 1)), ((0, 4, 4), (1, 1, 1)), ((8, 4, 5), (1, 1, 1))):
        l, h, _ = binding.make_structs(shape, periodic=per)
        assert lib.mc_workspace_bytes(C.byref(l), C.byref(h)) == 0  # odd nx / odd periodic dimension / empty
    l, h, _ = binding.make_structs((8, 3, 5), periodic=(1, 0, 0))
    assert lib.mc_workspace_bytes(C.byref(l), C.byref(h)) > 0        # odd OPEN dimensions are fine
    out = C.c_void_p()
    assert lib.mc_create(C.byref(lat), C.byref(ham), 42, None, 0, None, C.byref(out)) == binding.MC_EINVAL
    assert lib.mc_sweep(None, 1.0, 1) == binding.MC_EINVAL
    assert lib.mc_last_error(None) == b"null handle"
