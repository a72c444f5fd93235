"""CPU checks of the boundary: libts.so builds, loads and exports every symbol include/ts.h declares;
the host-only memory estimate behaves like the paper's scaler."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libts():
    from paper_2508_06628_b200 import build
    path = build.build()
    return C.CDLL(path)


def _declared():
    src = open(os.path.join(ROOT, "include", "ts.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = set(re.findall(r"\b(ts_[a-z_]+)\s*\(", src))
    return sorted(names)


def test_every_declared_symbol_is_exported(libts):
    names = _declared()
    assert len(names) >= 19 and "ts_state_create" in names and "ts_fire_step" in names
    for n in names:
        assert hasattr(libts, n), n


def test_binding_lists_the_same_symbols():
    import paper_2508_06628_b200 as ts
    assert sorted(ts.EXPORTS) == _declared()
    ts.lib()


def test_status_strings(libts):
    libts.ts_status_string.restype = C.c_char_p
    seen = {libts.ts_status_string(k) for k in range(9)}
    assert len(seen) == 9 and b"ok" in seen


def test_invalid_arguments_return_without_a_device(libts):
    assert libts.ts_state_destroy(None) == 1
    assert libts.ts_build_neighbors(None, None) == 1
    assert libts.ts_md_step(None, None, 1, 0, None) == 1
    out = C.c_size_t()
    libts.ts_estimate_system_bytes.argtypes = [C.c_int64, C.c_double, C.c_double, C.c_double, C.c_int32, C.POINTER(C.c_size_t)]
    assert libts.ts_estimate_system_bytes(0, 1.0, 1.0, 1.25, 0, C.byref(out)) == 1
    assert libts.ts_estimate_system_bytes(10, -1.0, 1.0, 1.25, 0, C.byref(out)) == 1


def test_estimate_scales_with_atoms_times_density():
    """bytes(system) = a N + b N rho r_list^3: the paper's n_atoms_x_density scaler."""
    import paper_2508_06628_b200 as ts
    r = 9.5
    b1 = ts.ts_estimate_system_bytes(864, 31.56 ** 3, r, 1.25, ts.TS_F32)
    b2 = ts.ts_estimate_system_bytes(2 * 864, 2 * 31.56 ** 3, r, 1.25, ts.TS_F32)     # same density, twice the atoms
    b3 = ts.ts_estimate_system_bytes(864, 0.5 * 31.56 ** 3, r, 1.25, ts.TS_F32)       # twice the density
    assert abs(b2 - 2 * b1) < 0.01 * b1
    assert b3 > 1.5 * b1
    # pair storage dominates: 4 bytes x N x nbar x slack
    nbar = 864 / 31.56 ** 3 * 4.0 / 3.0 * 3.141592653589793 * r ** 3
    assert b1 > 4 * 864 * nbar * 1.25
    assert ts.ts_estimate_system_bytes(864, 31.56 ** 3, r, 1.25, ts.TS_F64) > b1
