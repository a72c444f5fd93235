"""paper_2508_06628_b200 -- thin Python binding of libts (include/ts.h).

Argument marshalling only: every step of the hot path (binning, counting sort, neighbour CSR,
pair potentials, integrators, FIRE, reductions) runs in the CUDA kernels of csrc/.  PyTorch is
used for device memory and streams.  There is no CPU fallback: importing works without a GPU (so
the symbol table can be checked), but every compute call needs the CUDA library and a device and
fails loudly otherwise.  Nothing here imports oracle/.

The ts_* functions mirror the C entry points one to one; SimState bundles the caller-owned device
arrays (the paper's SimState: atom-wise attributes concatenated, system-wise stacked).
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libts.so")

TS_F32, TS_F64 = 0, 1
TS_LJ, TS_MORSE, TS_SOFT_SPHERE = 0, 1, 2
TS_WANT_ENERGY, TS_WANT_VIRIAL = 1, 2
TS_NVE, TS_BAOAB = 0, 1
TS_FIRE_FRESH, TS_FIRE_RUNNING, TS_FIRE_CONVERGED, TS_FIRE_FAILED = 0, 1, 2, 3
TS_FLAG_NBR_OVERFLOW, TS_FLAG_SHIFT_RANGE, TS_FLAG_NONFINITE, TS_FLAG_BAD_CELL = 1, 2, 4, 8
KINDS = {"lj": TS_LJ, "morse": TS_MORSE, "soft_sphere": TS_SOFT_SPHERE}

EXPORTS = ["ts_workspace_bytes", "ts_estimate_system_bytes", "ts_state_create", "ts_state_destroy",
           "ts_build_neighbors", "ts_compute_forces", "ts_md_step", "ts_fire_step", "ts_poll",
           "ts_converged_mask", "ts_swap_systems", "ts_get_neighbors", "ts_set_system_steps",
           "ts_get_system_steps", "ts_set_engine", "ts_invalidate", "ts_launch_count", "ts_clear_error",
           "ts_status_string", "ts_last_error", "ts_sched_fill", "ts_sched_max_scaler",
           "ts_sched_binpack", "ts_sched_partition", "ts_repack_systems", "ts_get_capacity",
           "ts_estimate_system_pairs", "ts_export_edges", "ts_md_step_external", "ts_fire_step_external",
           "ts_measure_fma_tflops", "ts_get_resident_neighbors", "ts_export_edges_static", "ts_static_scratch_setup",
           "ts_fire_status_async"]

TS_PHASE_INIT, TS_PHASE_PRE, TS_PHASE_POST, TS_PHASE_CHECK0 = 0, 1, 2, 3
(TS_OK, TS_ERR_INVALID_ARG, TS_ERR_CUDA, TS_ERR_WORKSPACE_TOO_SMALL, TS_ERR_NBR_OVERFLOW, TS_ERR_STALE_NBR,
 TS_ERR_NONFINITE, TS_ERR_UNSUPPORTED, TS_ERR_STICKY) = range(9)


class ts_units(C.Structure):
    _fields_ = [("mass_conv", C.c_double), ("kB", C.c_double)]


class ts_potential(C.Structure):
    _fields_ = [("kind", C.c_int32), ("n_types", C.c_int32), ("p0", C.c_void_p), ("p1", C.c_void_p),
                ("p2", C.c_void_p), ("rc", C.c_void_p), ("shift_energy", C.c_int32)]


class ts_state_desc(C.Structure):
    _fields_ = [("n_atoms", C.c_int64), ("n_systems", C.c_int32), ("dtype", C.c_int32), ("units", ts_units),
                ("pos", C.c_void_p), ("vel", C.c_void_p), ("force", C.c_void_p), ("mass", C.c_void_p),
                ("type", C.c_void_p), ("system_idx", C.c_void_p), ("cell", C.c_void_p),
                ("energy", C.c_void_p), ("virial", C.c_void_p), ("kinetic", C.c_void_p), ("sys_uid", C.c_void_p)]


class ts_nbr_params(C.Structure):
    _fields_ = [("skin", C.c_double), ("slack", C.c_double)]


class ts_md_params(C.Structure):
    _fields_ = [("integrator", C.c_int32), ("dt", C.c_double), ("temperature", C.c_double),
                ("friction", C.c_double), ("seed", C.c_uint64)]


class ts_fire_params(C.Structure):
    _fields_ = [("dt_start", C.c_double), ("dt_max", C.c_double), ("f_inc", C.c_double), ("f_dec", C.c_double),
                ("alpha_start", C.c_double), ("f_alpha", C.c_double), ("f_max", C.c_double),
                ("n_min", C.c_int32), ("max_steps", C.c_int32)]


class ts_report(C.Structure):
    _fields_ = [("flags", C.c_uint32), ("n_rebuilds", C.c_int32), ("nnz", C.c_int64), ("nnz_capacity", C.c_int64),
                ("steps_done", C.c_int64), ("n_converged", C.c_int32), ("n_failed", C.c_int32),
                ("max_neighbors", C.c_int32), ("list_valid", C.c_int32), ("resident_rebuilds", C.c_int64),
                ("engine", C.c_int32), ("reserved", C.c_int32)]


_lib = None


def lib():
    """The C-ABI library; raises if it has not been built (python -m paper_2508_06628_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2508_06628_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        for name in EXPORTS:
            getattr(L, name)          # AttributeError if a declared symbol is not exported
        L.ts_status_string.restype = C.c_char_p
        L.ts_last_error.restype = C.c_char_p
        L.ts_last_error.argtypes = [C.c_void_p]
        L.ts_launch_count.restype = C.c_int64
        L.ts_launch_count.argtypes = [C.c_void_p]
        L.ts_estimate_system_bytes.argtypes = [C.c_int64, C.c_double, C.c_double, C.c_double, C.c_int32,
                                               C.POINTER(C.c_size_t)]
        _lib = L
    return _lib


class TsError(RuntimeError):
    def __init__(self, code, what, detail=""):
        self.code = code
        msg = lib().ts_status_string(code).decode()
        super().__init__(f"{what}: {msg} ({code}) {detail}".strip())


def _check(code, what, handle=None):
    if code != 0:
        detail = lib().ts_last_error(handle).decode() if handle else ""
        raise TsError(code, what, detail)


_raw_stream = None


def _stream():
    """torch's current CUDA stream as a raw handle.  torch.cuda.current_stream() builds a Stream object (~20 us); the
    raw getter behind it costs about a microsecond, which matters for callers that step once per call."""
    global _raw_stream
    import torch
    if _raw_stream is None:
        fast = getattr(torch._C, "_cuda_getCurrentRawStream", None)
        _raw_stream = (lambda: fast(torch.cuda.current_device())) if fast is not None else \
                      (lambda: torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(_raw_stream())


# ------------------------------------------------------------------------------- 1:1 entry points
def ts_estimate_system_bytes(n_atoms, volume, r_list, slack=1.25, dtype=TS_F32):
    out = C.c_size_t()
    _check(lib().ts_estimate_system_bytes(int(n_atoms), float(volume), float(r_list), float(slack), int(dtype),
                                          C.byref(out)), "ts_estimate_system_bytes")
    return out.value


def ts_workspace_bytes(desc, pot, nbr):
    out = C.c_size_t()
    _check(lib().ts_workspace_bytes(C.byref(desc), C.byref(pot), C.byref(nbr), C.byref(out)), "ts_workspace_bytes")
    return out.value


def ts_state_create(desc, pot, nbr, workspace_ptr, workspace_bytes):
    h = C.c_void_p()
    _check(lib().ts_state_create(C.byref(desc), C.byref(pot), C.byref(nbr), C.c_void_p(workspace_ptr),
                                 C.c_size_t(workspace_bytes), C.byref(h)), "ts_state_create")
    return h


def ts_state_destroy(h):
    _check(lib().ts_state_destroy(h), "ts_state_destroy")


def ts_build_neighbors(h):
    _check(lib().ts_build_neighbors(h, _stream()), "ts_build_neighbors", h)


def ts_compute_forces(h, want=TS_WANT_ENERGY | TS_WANT_VIRIAL):
    _check(lib().ts_compute_forces(h, C.c_uint32(want), _stream()), "ts_compute_forces", h)


def ts_md_step(h, params, n_steps, want=TS_WANT_ENERGY):
    _check(lib().ts_md_step(h, C.byref(params), C.c_int32(n_steps), C.c_uint32(want), _stream()), "ts_md_step", h)


def ts_fire_step(h, params, n_steps):
    _check(lib().ts_fire_step(h, C.byref(params), C.c_int32(n_steps), _stream()), "ts_fire_step", h)


def ts_poll(h):
    r = ts_report()
    _check(lib().ts_poll(h, C.byref(r), _stream()), "ts_poll", h)
    return r


def ts_clear_error(h):
    _check(lib().ts_clear_error(h, _stream()), "ts_clear_error", h)


def ts_converged_mask(h, n_systems):
    mask = np.zeros(n_systems, np.uint8)
    status = np.zeros(n_systems, np.int32)
    steps = np.zeros(n_systems, np.int32)
    _check(lib().ts_converged_mask(h, mask.ctypes.data_as(C.c_void_p), status.ctypes.data_as(C.c_void_p),
                                   steps.ctypes.data_as(C.c_void_p), _stream()), "ts_converged_mask", h)
    return mask.astype(bool), status, steps


def ts_fire_status_async(h, status_ptr, steps_ptr):
    """status_ptr / steps_ptr: addresses of page-locked HOST int32 arrays of S entries (0 = skip)."""
    _check(lib().ts_fire_status_async(h, C.c_void_p(status_ptr), C.c_void_p(steps_ptr), _stream()), "ts_fire_status_async", h)


def ts_swap_systems(h, slots, fresh_desc):
    slots = np.ascontiguousarray(np.asarray(slots, dtype=np.int32))
    _check(lib().ts_swap_systems(h, slots.ctypes.data_as(C.c_void_p), C.c_int32(slots.size), C.byref(fresh_desc),
                                 _stream()), "ts_swap_systems", h)


def ts_repack_systems(h, keep, fresh_desc, fresh_n_atoms):
    keep = np.ascontiguousarray(np.asarray(keep, dtype=np.int32))
    fn = np.ascontiguousarray(np.asarray(fresh_n_atoms, dtype=np.int32))
    _check(lib().ts_repack_systems(h, keep.ctypes.data_as(C.c_void_p), C.c_int32(keep.size),
                                   C.byref(fresh_desc) if fresh_desc is not None else None,
                                   fn.ctypes.data_as(C.c_void_p), _stream()), "ts_repack_systems", h)


def ts_get_capacity(h):
    n, s, p = C.c_int64(), C.c_int32(), C.c_int64()
    _check(lib().ts_get_capacity(h, C.byref(n), C.byref(s), C.byref(p)), "ts_get_capacity", h)
    return n.value, s.value, p.value


def ts_estimate_system_pairs(n_atoms, volume, r_list, slack=1.25):
    out = C.c_int64()
    _check(lib().ts_estimate_system_pairs(C.c_int64(int(n_atoms)), C.c_double(volume), C.c_double(r_list),
                                          C.c_double(slack), C.byref(out)), "ts_estimate_system_pairs")
    return out.value


def ts_export_edges(h, edge_i_ptr, edge_j_ptr, edge_shift_ptr, cap, n_edges_ptr):
    _check(lib().ts_export_edges(h, C.c_void_p(edge_i_ptr), C.c_void_p(edge_j_ptr), C.c_void_p(edge_shift_ptr),
                                 C.c_int64(cap), C.c_void_p(n_edges_ptr), _stream()), "ts_export_edges", h)


def ts_export_edges_static(h, edge_i_ptr, edge_j_ptr, edge_shift_ptr, cap, n_edges_ptr):
    _check(lib().ts_export_edges_static(h, C.c_void_p(edge_i_ptr), C.c_void_p(edge_j_ptr), C.c_void_p(edge_shift_ptr),
                                        C.c_int64(cap), C.c_void_p(n_edges_ptr), _stream()), "ts_export_edges_static", h)


def ts_static_scratch_setup():
    """Looks up the library's static scratch array on the current device; returns its limit in systems."""
    n = C.c_int64(0)
    _check(lib().ts_static_scratch_setup(C.byref(n)), "ts_static_scratch_setup")
    return int(n.value)


def ts_md_step_external(h, params, phase):
    _check(lib().ts_md_step_external(h, C.byref(params), C.c_int32(phase), _stream()), "ts_md_step_external", h)


def ts_fire_step_external(h, params, phase):
    _check(lib().ts_fire_step_external(h, C.byref(params), C.c_int32(phase), _stream()), "ts_fire_step_external", h)


def ts_get_resident_neighbors(h, system, n_atoms_of_system):
    off = np.zeros(n_atoms_of_system + 1, np.int64)
    nnz = C.c_int64()
    _check(lib().ts_get_resident_neighbors(h, C.c_int32(system), off.ctypes.data_as(C.c_void_p), None, None, C.c_int64(0),
                                           C.byref(nnz), _stream()), "ts_get_resident_neighbors", h)
    j = np.zeros(nnz.value, np.int32)
    shift = np.zeros((nnz.value, 3), np.int8)
    _check(lib().ts_get_resident_neighbors(h, C.c_int32(system), off.ctypes.data_as(C.c_void_p), j.ctypes.data_as(C.c_void_p),
                                           shift.ctypes.data_as(C.c_void_p), C.c_int64(nnz.value), C.byref(nnz), _stream()),
           "ts_get_resident_neighbors", h)
    return off, j, shift


def ts_measure_fma_tflops(kind, scratch_ptr):
    out = C.c_double()
    _check(lib().ts_measure_fma_tflops(C.c_int32(kind), C.c_void_p(scratch_ptr), C.byref(out), _stream()),
           "ts_measure_fma_tflops")
    return out.value


def ts_get_neighbors(h, n_atoms):
    off = np.zeros(n_atoms + 1, np.int64)
    _check(lib().ts_get_neighbors(h, off.ctypes.data_as(C.c_void_p), None, None, C.c_int64(0), _stream()),
           "ts_get_neighbors", h)
    nnz = int(off[-1])
    j = np.zeros(nnz, np.int32)
    shift = np.zeros((nnz, 3), np.int8)
    _check(lib().ts_get_neighbors(h, off.ctypes.data_as(C.c_void_p), j.ctypes.data_as(C.c_void_p),
                                  shift.ctypes.data_as(C.c_void_p), C.c_int64(nnz), _stream()), "ts_get_neighbors", h)
    return off, j, shift


def ts_set_system_steps(h, steps):
    steps = np.ascontiguousarray(np.asarray(steps, dtype=np.uint64))
    _check(lib().ts_set_system_steps(h, steps.ctypes.data_as(C.c_void_p), _stream()), "ts_set_system_steps", h)


def ts_get_system_steps(h, n_systems):
    steps = np.zeros(n_systems, np.uint64)
    _check(lib().ts_get_system_steps(h, steps.ctypes.data_as(C.c_void_p), _stream()), "ts_get_system_steps", h)
    return steps


def ts_set_engine(h, engine):
    _check(lib().ts_set_engine(h, C.c_int32(engine)), "ts_set_engine", h)


def ts_invalidate(h):
    _check(lib().ts_invalidate(h), "ts_invalidate", h)


def ts_launch_count(h):
    return int(lib().ts_launch_count(h))


# ------------------------------------------------------------------------------- host scheduling
def _dptr(a):
    return a.ctypes.data_as(C.c_void_p)


def ts_sched_fill(cost, budget):
    cost = np.ascontiguousarray(np.asarray(cost, dtype=np.float64))
    n, used = C.c_int64(), C.c_double()
    _check(lib().ts_sched_fill(_dptr(cost), C.c_int64(cost.size), C.c_double(budget), C.byref(n), C.byref(used)),
           "ts_sched_fill")
    return n.value, used.value


def ts_sched_max_scaler(n_systems, scaler):
    ns = np.ascontiguousarray(np.asarray(n_systems, dtype=np.int64))
    sc = np.ascontiguousarray(np.asarray(scaler, dtype=np.float64))
    out = C.c_double()
    _check(lib().ts_sched_max_scaler(_dptr(ns), _dptr(sc), C.c_int32(ns.size), C.byref(out)), "ts_sched_max_scaler")
    return out.value


def ts_sched_binpack(cost, capacity):
    cost = np.ascontiguousarray(np.asarray(cost, dtype=np.float64))
    bins = np.zeros(cost.size, np.int32)
    nb = C.c_int32()
    _check(lib().ts_sched_binpack(_dptr(cost), C.c_int64(cost.size), C.c_double(capacity), _dptr(bins), C.byref(nb)),
           "ts_sched_binpack")
    return bins, nb.value


def ts_sched_partition(cost, n_ranks):
    cost = np.ascontiguousarray(np.asarray(cost, dtype=np.float64))
    rank = np.zeros(cost.size, np.int32)
    load = np.zeros(n_ranks, np.float64)
    _check(lib().ts_sched_partition(_dptr(cost), C.c_int64(cost.size), C.c_int32(n_ranks), _dptr(rank), _dptr(load)),
           "ts_sched_partition")
    return rank, load


def md_params(integrator="nve", dt=1.0, temperature=0.0, friction=0.0, seed=0, **_):
    integ = {"nve": TS_NVE, "baoab": TS_BAOAB}.get(integrator, integrator)
    return ts_md_params(int(integ), float(dt), float(temperature), float(friction), int(seed))


def fire_params(dt_start, dt_max, f_inc=1.1, f_dec=0.5, alpha_start=0.1, f_alpha=0.99, f_max=1e-4, n_min=5,
                max_steps=50000, **_):
    return ts_fire_params(dt_start, dt_max, f_inc, f_dec, alpha_start, f_alpha, f_max, int(n_min), int(max_steps))


from .state import SimState  # noqa: E402,F401
