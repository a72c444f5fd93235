"""ctypes wrapper around oracle/ts_oracle.c -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package (it is the fp64 O(N^2) all-images oracle of SURVEY.md section 8(c)).  It imports
nothing from paper_2508_06628_b200 and the CUDA path imports nothing from here.

Batches are duck-typed: any object with attributes pos, vel, mass, type, sys_offset, cell,
potential (kind, n_types, p0, p1, p2, rc, shift_energy), mass_conv, kB.  Inputs are never
modified; results come back as fresh numpy arrays.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_KINDS = {"lj": 0, "morse": 1, "soft_sphere": 2}
_lib = None


class _Batch(C.Structure):
    _fields_ = [("n_atoms", C.c_int64), ("n_systems", C.c_int32), ("sys_off", C.c_void_p),
                ("pos", C.c_void_p), ("vel", C.c_void_p), ("force", C.c_void_p),
                ("mass", C.c_void_p), ("type", C.c_void_p), ("cell", C.c_void_p),
                ("kind", C.c_int32), ("n_types", C.c_int32), ("shift_energy", C.c_int32),
                ("p0", C.c_void_p), ("p1", C.c_void_p), ("p2", C.c_void_p), ("rc", C.c_void_p),
                ("mass_conv", C.c_double), ("kB", C.c_double)]


class _Fire(C.Structure):
    _fields_ = [("dt_start", C.c_double), ("dt_max", C.c_double), ("f_inc", C.c_double),
                ("f_dec", C.c_double), ("alpha_start", C.c_double), ("f_alpha", C.c_double),
                ("f_max", C.c_double), ("n_min", C.c_int32), ("max_steps", C.c_int32)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
    return _lib


def default_threads():
    return max(1, os.cpu_count() or 1)


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a, shape=None):
    a = np.ascontiguousarray(np.array(a, dtype=np.float64, copy=True))
    if shape is not None:
        a = a.reshape(shape)
    return a


class _Held:
    """A C batch plus the numpy arrays that keep its memory alive."""

    def __init__(self, b):
        pot = b.potential
        self.sys_off = np.ascontiguousarray(np.asarray(b.sys_offset, dtype=np.int64))
        S = self.sys_off.size - 1
        N = int(self.sys_off[-1])
        self.pos = _f64(b.pos, (N, 3))
        self.vel = _f64(b.vel, (N, 3)) if getattr(b, "vel", None) is not None else np.zeros((N, 3))
        self.force = np.zeros((N, 3))
        self.mass = _f64(b.mass, (N,))
        self.type = np.ascontiguousarray(np.asarray(b.type, dtype=np.int32))
        self.cell = _f64(b.cell, (S, 3, 3))
        nt = int(pot.n_types)
        self.p0, self.p1, self.p2, self.rc = (_f64(getattr(pot, k), (nt * nt,)) for k in ("p0", "p1", "p2", "rc"))
        kind = pot.kind if isinstance(pot.kind, int) else _KINDS[pot.kind]
        self.S, self.N = S, N
        self.c = _Batch(N, S, _p(self.sys_off), _p(self.pos), _p(self.vel), _p(self.force),
                        _p(self.mass), _p(self.type), _p(self.cell), kind, nt,
                        int(bool(pot.shift_energy)), _p(self.p0), _p(self.p1), _p(self.p2), _p(self.rc),
                        float(b.mass_conv), float(b.kB))


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


# ------------------------------------------------------------------------------- O1
def cell_geometry(h):
    h = _f64(h, (9,))
    hinv, hperp, vol = np.zeros(9), np.zeros(3), C.c_double()
    _check(lib().orc_cell_geometry(_p(h), _p(hinv), _p(hperp), C.byref(vol)), "cell_geometry")
    return hinv.reshape(3, 3), hperp, vol.value


def pairs(pos, cell, R):
    """Directed pair set P(R) of ONE system: arrays i, j (int32), S [n,3] (int32), r2."""
    pos = _f64(pos).reshape(-1, 3)
    h = _f64(cell, (9,))
    n = pos.shape[0]
    cnt = C.c_int64()
    rc = lib().orc_pairs(_p(pos), C.c_int64(n), _p(h), C.c_double(R), C.c_int64(0), None, None, None, None, C.byref(cnt))
    if rc not in (0, 2):
        _check(rc, "pairs")
    m = cnt.value
    oi, oj, oS, r2 = np.zeros(m, np.int32), np.zeros(m, np.int32), np.zeros((m, 3), np.int32), np.zeros(m)
    _check(lib().orc_pairs(_p(pos), C.c_int64(n), _p(h), C.c_double(R), C.c_int64(m), _p(oi), _p(oj), _p(oS), _p(r2), C.byref(cnt)), "pairs")
    return oi, oj, oS, r2


# ------------------------------------------------------------------------------- O2
def pair_potential(kind, p0, p1, p2, rc, shift_energy, r):
    V, dV = C.c_double(), C.c_double()
    k = kind if isinstance(kind, int) else _KINDS[kind]
    _check(lib().orc_pair_potential(k, C.c_double(p0), C.c_double(p1), C.c_double(p2), C.c_double(rc),
                                    int(bool(shift_energy)), C.c_double(r), C.byref(V), C.byref(dV)), "pair_potential")
    return V.value, dV.value


def energy_forces(batch, nthreads=None):
    h = _Held(batch)
    E, W, Eabs = np.zeros(h.S), np.zeros((h.S, 3, 3)), np.zeros(h.S)
    _check(lib().orc_energy_forces(C.byref(h.c), _p(E), _p(W), _p(Eabs), nthreads or default_threads()), "energy_forces")
    return {"E": E, "F": h.force, "W": W, "Eabs": Eabs}


def kinetic(batch):
    h = _Held(batch)
    KE = np.zeros(h.S)
    _check(lib().orc_kinetic(C.byref(h.c), _p(KE)), "kinetic")
    return KE


# ------------------------------------------------------------------------------- O5
def philox4x32_10(ctr, key):
    ctr = np.ascontiguousarray(np.asarray(ctr, dtype=np.uint32))
    key = np.ascontiguousarray(np.asarray(key, dtype=np.uint32))
    out = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(_p(ctr), _p(key), _p(out))
    return out


def normals_from_words(w):
    w = np.ascontiguousarray(np.asarray(w, dtype=np.uint32))
    xi = np.zeros(3)
    lib().orc_normals_from_words(_p(w), _p(xi))
    return xi


def langevin_xi(seed, sys_uid, local_idx, step):
    xi = np.zeros(3)
    lib().orc_langevin_xi(C.c_uint64(seed), C.c_uint32(sys_uid), C.c_uint32(local_idx), C.c_uint64(step), _p(xi))
    return xi


# ------------------------------------------------------------------------------- O3 / O4
def md_run(batch, integrator, dt, n_steps, temperature=0.0, friction=0.0, seed=0, sys_uid=None,
           step=None, history=False, nthreads=None):
    """integrator: 'nve' (O3) or 'baoab' (O4).  Returns the state after n_steps."""
    h = _Held(batch)
    integ = {"nve": 0, "baoab": 1}[integrator]
    E, W, KE = np.zeros(h.S), np.zeros((h.S, 3, 3)), np.zeros(h.S)
    uid = None if sys_uid is None else np.ascontiguousarray(np.asarray(sys_uid, dtype=np.uint32))
    stp = np.zeros(h.S, np.uint64) if step is None else np.ascontiguousarray(np.array(step, dtype=np.uint64))
    eh = np.zeros((n_steps + 1, h.S)) if history else None
    kh = np.zeros((n_steps + 1, h.S)) if history else None
    _check(lib().orc_md_run(C.byref(h.c), integ, C.c_double(dt), C.c_double(temperature), C.c_double(friction),
                            C.c_uint64(seed), _p(uid), _p(stp), int(n_steps), _p(E), _p(W), _p(KE), _p(eh), _p(kh),
                            nthreads or default_threads()), "md_run")
    return {"pos": h.pos, "vel": h.vel, "F": h.force, "E": E, "W": W, "KE": KE, "step": stp,
            "epot_hist": eh, "ke_hist": kh}


# ------------------------------------------------------------------------------- O6
FIRE_FRESH, FIRE_RUNNING, FIRE_CONVERGED, FIRE_FAILED = 0, 1, 2, 3


def fire_run(batch, params, n_steps, state=None, nthreads=None):
    """params: object/dict with dt_start, dt_max, f_inc, f_dec, alpha_start, f_alpha, f_max,
    n_min, max_steps.  state: dict from a previous call (continues) or None (fresh)."""
    h = _Held(batch)
    g = (lambda k: params[k]) if isinstance(params, dict) else (lambda k: getattr(params, k))
    fp = _Fire(g("dt_start"), g("dt_max"), g("f_inc"), g("f_dec"), g("alpha_start"), g("f_alpha"),
               g("f_max"), int(g("n_min")), int(g("max_steps")))
    if state is None:
        state = {"dt": np.zeros(h.S), "alpha": np.zeros(h.S), "npos": np.zeros(h.S, np.int32),
                 "nsteps": np.zeros(h.S, np.int32), "status": np.zeros(h.S, np.int32),
                 "E": np.zeros(h.S), "fmax": np.zeros(h.S)}
    st = {k: np.ascontiguousarray(np.array(v, copy=True)) for k, v in state.items()}
    E, fmax = st["E"], st["fmax"]
    _check(lib().orc_fire_run(C.byref(h.c), C.byref(fp), int(n_steps), _p(st["dt"]), _p(st["alpha"]), _p(st["npos"]),
                              _p(st["nsteps"]), _p(st["status"]), _p(E), _p(fmax), nthreads or default_threads()), "fire_run")
    return {"pos": h.pos, "vel": h.vel, "F": h.force, "E": E, "fmax": fmax, "state": st}
