"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a without a GPU, loads, and
exports every symbol include/amr_godunov.h declares; host-only argument validation works without a
device (no compute calls here)."""
import ctypes as C
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "amr_godunov.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(amr_[a-z_0-9]+)\s*\(", src)))


def test_library_builds_loads_and_exports_the_header():
    from paper_1412_0934_b200 import build, binding
    path = build.build()
    assert os.path.exists(path)
    L = binding.lib()
    declared = _declared_symbols()
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(L, name), name
    assert sorted(binding.EXPORTS) == declared
    assert b"sm_100a" in L.amr_version()


def test_descriptor_validation_needs_no_device():
    from paper_1412_0934_b200 import binding
    L = binding.lib()
    d = binding._Desc()
    d.npatch, d.n, d.nghost, d.nfields, d.dtype, d.level, d.dx = 4096, 16, 3, 9, binding.AMR_F32, 0, 1.0 / 256
    d.self_periodic = 1
    nbytes = L.amr_patch_batch_bytes(C.byref(d))
    state = 2 * 9 * 4096 * 16 ** 3 * 4
    assert state <= nbytes <= state + (1 << 20)          # interiors only, two buffers, small tables
    d.n = 12
    assert L.amr_patch_batch_bytes(C.byref(d)) == 0 and b"multiple of 8" in L.amr_last_error()
    d.n, d.nfields = 16, 6
    assert L.amr_patch_batch_bytes(C.byref(d)) == 0
    d.nfields, d.level = 9, 1                            # level > 0 reserves the prolongation halo
    assert L.amr_patch_batch_bytes(C.byref(d)) >= state + 9 * 4096 * 22 ** 3 * 4
    h = C.c_void_p()
    assert L.amr_patch_batch_create(C.byref(d), None, 0, None, C.byref(h)) == -1
    assert L.amr_hydro_step(None, 1.0, 1.4, 1, 1) == -1
