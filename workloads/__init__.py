"""Seeded synthetic inputs for the five BASELINE.json configs (SURVEY.md section 8(d), R13/R14/R20/
R28/R32/R33).  This module serves BOTH the oracle and the CUDA path and therefore holds none of
the method's arithmetic: no potential, no integrator, no neighbour list.  It only lays out
lattices, draws random numbers and rejects inputs that sit within `w` of a cutoff (R28) with a
KD-tree distance query of its own (scipy), so neither side's pair search decides the inputs.

Stand-in statement: the paper benchmarks FCC copper supercells of 16..864 atoms under Langevin MD
(section 4); no dataset is involved.  These generators keep those shapes (FCC
supercells up to 864 atoms, batched near capacity) and add the ragged/triclinic/FIRE cases that
BASELINE.json:configs names.  Random streams: numpy Generator(PCG64(SeedSequence([cfg, system,..]))).
"""
from dataclasses import dataclass, field, replace

import numpy as np
from scipy.spatial import cKDTree

MASS_CONV_METAL = 103.64269652680505     # eV fs^2 / (amu A^2)   (R1)
KB_METAL = 8.617333262145179e-5          # eV / K                (R1)


@dataclass
class Potential:
    kind: str                  # "lj" | "morse" | "soft_sphere"
    n_types: int
    p0: np.ndarray             # [nt, nt]  LJ eps   | Morse D     | soft eps
    p1: np.ndarray             # [nt, nt]  LJ sigma | Morse alpha | soft sigma
    p2: np.ndarray             # [nt, nt]  -        | Morse r0    | soft exponent
    rc: np.ndarray             # [nt, nt]  cutoff
    shift_energy: bool = True  # R10

    @property
    def rc_max(self):
        return float(np.max(self.rc))


@dataclass
class Batch:
    name: str
    pos: np.ndarray            # [N,3] float64 (values representable in `dtype`)
    vel: np.ndarray            # [N,3]
    mass: np.ndarray           # [N]
    type: np.ndarray           # [N] int32
    system_idx: np.ndarray     # [N] int32, non-decreasing
    sys_offset: np.ndarray     # [S+1] int64
    cell: np.ndarray           # [S,3,3], rows = lattice vectors (R4)
    potential: Potential
    mass_conv: float
    kB: float
    skin: float
    dtype: str = "f64"         # precision the run is specified in ("f32" | "f64")
    sys_uid: np.ndarray = None # [S] uint32 persistent ids (R18)
    md: dict = field(default_factory=dict)     # integrator, dt, temperature, friction, seed, n_steps
    fire: dict = field(default_factory=dict)

    @property
    def n_atoms(self):
        return int(self.sys_offset[-1])

    @property
    def n_systems(self):
        return int(self.sys_offset.size - 1)

    @property
    def r_list(self):
        return self.potential.rc_max + self.skin

    def system(self, s):
        """A one-system Batch view (copies)."""
        return take(self, [s])


def _finish(name, parts, potential, mass_conv, kB, skin, dtype, uids, md=None, fire=None):
    n = np.array([p[0].shape[0] for p in parts], dtype=np.int64)
    off = np.concatenate([[0], np.cumsum(n)]).astype(np.int64)
    b = Batch(name=name,
              pos=np.concatenate([p[0] for p in parts]), vel=np.concatenate([p[1] for p in parts]),
              mass=np.concatenate([p[2] for p in parts]), type=np.concatenate([p[3] for p in parts]).astype(np.int32),
              system_idx=np.repeat(np.arange(len(parts), dtype=np.int32), n), sys_offset=off,
              cell=np.stack([p[4] for p in parts]), potential=potential, mass_conv=mass_conv, kB=kB, skin=skin,
              dtype=dtype, sys_uid=np.asarray(uids, dtype=np.uint32), md=md or {}, fire=fire or {})
    return b


def take(b, systems):
    """Batch made of the listed systems of b, in that order."""
    systems = list(systems)
    parts = []
    for s in systems:
        a0, a1 = int(b.sys_offset[s]), int(b.sys_offset[s + 1])
        parts.append((b.pos[a0:a1].copy(), b.vel[a0:a1].copy(), b.mass[a0:a1].copy(), b.type[a0:a1].copy(), b.cell[s].copy()))
    return _finish(b.name, parts, b.potential, b.mass_conv, b.kB, b.skin, b.dtype, b.sys_uid[systems], dict(b.md), dict(b.fire))


def concat(batches):
    b0 = batches[0]
    parts, uids = [], []
    for b in batches:
        for s in range(b.n_systems):
            a0, a1 = int(b.sys_offset[s]), int(b.sys_offset[s + 1])
            parts.append((b.pos[a0:a1], b.vel[a0:a1], b.mass[a0:a1], b.type[a0:a1], b.cell[s]))
            uids.append(b.sys_uid[s])
    return _finish(b0.name, parts, b0.potential, b0.mass_conv, b0.kB, b0.skin, b0.dtype, uids, dict(b0.md), dict(b0.fire))


def _round(a, dtype):
    """Round to the run's storage precision and promote back (R27): both sides see these values."""
    return a.astype(np.float32).astype(np.float64) if dtype == "f32" else np.asarray(a, dtype=np.float64)


def _rng(*key):
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([int(k) for k in key])))


# ------------------------------------------------------------------------------- lattices
_FCC = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]], dtype=np.float64)
_BCC = np.array([[0, 0, 0], [.5, .5, .5]], dtype=np.float64)


def lattice(basis, a, reps):
    """Fractional basis x conventional cubic cell a, replicated reps=(n1,n2,n3).  Returns pos, cell."""
    n1, n2, n3 = reps
    g = np.stack(np.meshgrid(np.arange(n1), np.arange(n2), np.arange(n3), indexing="ij"), -1).reshape(-1, 3)
    pos = (g[:, None, :] + basis[None, :, :]).reshape(-1, 3) * a
    return pos, np.diag([n1 * a, n2 * a, n3 * a]).astype(np.float64)


def maxwell_boltzmann(rng, mass, T, kB, mass_conv):
    """v ~ N(0, kB T / (m mass_conv)) per component, then COM velocity removed (R20)."""
    sig = np.sqrt(kB * T / (mass * mass_conv))
    v = rng.standard_normal((mass.size, 3)) * sig[:, None]
    v -= (mass[:, None] * v).sum(0) / mass.sum()
    return v


# ------------------------------------------------------------------------------- R28 rejection
def near_cutoff_atoms(pos, cell, radii, w):
    """Indices of atoms in a pair (any periodic image) whose distance is within w of a radius.
    Own KD-tree query over explicit ghost images; shares nothing with either pair search."""
    hinv = np.linalg.inv(cell)
    f = pos @ hinv
    fw = f - np.floor(f)
    xw = fw @ cell
    Rm = max(radii) + w
    hperp = 1.0 / np.linalg.norm(hinv, axis=0)
    m = Rm / hperp
    nimg = np.ceil(m).astype(int)
    pts, parent = [], []
    idx = np.arange(pos.shape[0])
    for s0 in range(-nimg[0], nimg[0] + 1):
        for s1 in range(-nimg[1], nimg[1] + 1):
            for s2 in range(-nimg[2], nimg[2] + 1):
                fg = fw + np.array([s0, s1, s2], dtype=np.float64)
                keep = np.all((fg > -m) & (fg < 1.0 + m), axis=1)
                if keep.any():
                    pts.append(fg[keep] @ cell)
                    parent.append(idx[keep])
    pts, parent = np.concatenate(pts), np.concatenate(parent)
    tc, ta = cKDTree(xw), cKDTree(pts)
    sd = tc.sparse_distance_matrix(ta, Rm, output_type="ndarray")
    d = sd["v"]
    bad = np.zeros(d.size, dtype=bool)
    for R in radii:
        bad |= np.abs(d - R) < w
    bad &= d > 0.0
    return np.unique(np.concatenate([sd["i"][bad], parent[sd["j"][bad]]]))


def _clean(base, draw, cell, radii, w, dtype, key, max_attempts=50):
    """R28: re-draw the displacement of every atom in a near-cutoff pair from sub-seed
    (key..., atom, attempt) until clean.  `draw(rng, n)` -> [n,3] displacements."""
    disp = draw(_rng(*key, 0), base.shape[0])
    pos = _round(base + disp, dtype)
    for attempt in range(1, max_attempts + 1):
        bad = near_cutoff_atoms(pos, cell, radii, w)
        if bad.size == 0:
            return pos
        for i in bad:
            disp[i] = draw(_rng(*key, 1 + int(i), attempt), 1)[0]
        pos = _round(base + disp, dtype)
    raise RuntimeError("R28 rejection did not converge")


def reject_width(dtype, length_scale=1.0):
    """w = 1e-6 A for fp64 runs, 1e-4 A for fp32 runs, scaled by sigma in reduced units (R28)."""
    return (1e-4 if dtype == "f32" else 1e-6) * length_scale


def _single_type(kind, p0, p1, p2, rc, shift=True):
    a = lambda v: np.array([[v]], dtype=np.float64)
    return Potential(kind, 1, a(p0), a(p1), a(p2), a(rc), shift)


# ------------------------------------------------------------------------------- cfg1, cfg2
LJ_AR = dict(eps=0.0104, sigma=3.40, rc=8.5, mass=39.948, a=5.26)


def fcc_argon(cfg_id, n_systems, reps, disp, skin, T, dtype, md, name, system_ids=None, clean=True, w=None):
    pot = _single_type("lj", LJ_AR["eps"], LJ_AR["sigma"], 0.0, LJ_AR["rc"])
    base, cell = lattice(_FCC, LJ_AR["a"], (reps,) * 3)
    cell = _round(cell, dtype)
    parts, ids = [], list(range(n_systems)) if system_ids is None else list(system_ids)
    radii = [pot.rc_max, pot.rc_max + skin]
    for sid in ids:
        if clean:
            pos = _clean(base, disp, cell, radii, w or reject_width(dtype), dtype, (cfg_id, sid))
        else:
            pos = _round(base + disp(_rng(cfg_id, sid, 0), base.shape[0]), dtype)
        mass = np.full(base.shape[0], LJ_AR["mass"])
        vel = _round(maxwell_boltzmann(_rng(cfg_id, sid, 10**6), mass, T, KB_METAL, MASS_CONV_METAL), dtype)
        parts.append((pos, vel, _round(mass, dtype), np.zeros(base.shape[0], np.int32), cell))
    return _finish(name, parts, pot, MASS_CONV_METAL, KB_METAL, skin, dtype, ids, md=md)


def cfg1(n_systems=4, reps=4, dtype="f64", clean=True, system_ids=None, w=None):
    """BASELINE.json:configs[0]: 4 x 256-atom FCC Ar, U(-0.02,0.02) A displacements, MB 50 K, NVE."""
    disp = lambda rng, n: rng.uniform(-0.02, 0.02, size=(n, 3))
    md = dict(integrator="nve", dt=2.0, temperature=50.0, friction=0.0, seed=0, n_steps=100)
    return fcc_argon(1, n_systems, reps, disp, 0.5, 50.0, dtype, md, "cfg1", system_ids, clean, w)


def cfg2(n_systems=64, reps=6, dtype="f32", clean=True, system_ids=None, w=None):
    """BASELINE.json:configs[1]: 64 x 864-atom FCC Ar, N(0,0.05 A), skin 1.0, BAOAB 80 K (graded)."""
    disp = lambda rng, n: rng.normal(0.0, 0.05, size=(n, 3))
    md = dict(integrator="baoab", dt=2.0, temperature=80.0, friction=0.01, seed=42, n_steps=1000)
    return fcc_argon(2, n_systems, reps, disp, 1.0, 80.0, dtype, md, "cfg2", system_ids, clean, w)


# ------------------------------------------------------------------------------- cfg3 (R32)
CU_MORSE = dict(D=0.3429, alpha=1.3588, r0=2.866, rc=6.0, mass=63.546, a_fcc=3.615, a_bcc=3.615 / 2.0 ** (1.0 / 3.0))


def _closest_supercell(b, n_star, lo=32, hi=2048):
    best = None
    for n1 in range(1, 17):
        for n2 in range(n1, 33):
            for n3 in range(n2, 2 * n1 + 1):
                n = b * n1 * n2 * n3
                if lo <= n <= hi:
                    k = (abs(n - n_star), n, n1, n2, n3)
                    if best is None or k < best:
                        best = k
    return best[2:], best[1]


def cfg3(n_systems=512, dtype="f32", clean=True, system_ids=None, n_range=(32, 2048), w=None):
    """BASELINE.json:configs[2]: ragged Cu FCC/BCC supercells, sheared triclinic cells, Morse."""
    pot = _single_type("morse", CU_MORSE["D"], CU_MORSE["alpha"], CU_MORSE["r0"], CU_MORSE["rc"])
    skin = 0.5
    radii = [pot.rc_max, pot.rc_max + skin]
    ids = list(range(n_systems)) if system_ids is None else list(system_ids)
    parts = []
    for sid in ids:
        rng = _rng(3, sid, 10**6 + 1)
        n_star = int(rng.integers(n_range[0], n_range[1] + 1))
        fcc = bool(rng.integers(0, 2))
        basis, a = (_FCC, CU_MORSE["a_fcc"]) if fcc else (_BCC, CU_MORSE["a_bcc"])
        reps, _ = _closest_supercell(basis.shape[0], n_star, n_range[0], n_range[1])
        base, cell = lattice(basis, a, reps)
        eps = np.zeros((3, 3))
        e = rng.uniform(-0.1, 0.1, size=3)
        eps[0, 1] = eps[1, 0] = e[0]; eps[0, 2] = eps[2, 0] = e[1]; eps[1, 2] = eps[2, 1] = e[2]
        strain = np.eye(3) + eps
        cell = _round(cell @ strain, dtype)
        base = base @ strain
        noise = lambda r, n: r.normal(0.0, 0.1, size=(n, 3))
        if clean:
            pos = _clean(base, noise, cell, radii, w or reject_width(dtype), dtype, (3, sid))
        else:
            pos = _round(base + noise(_rng(3, sid, 0), base.shape[0]), dtype)
        mass = np.full(base.shape[0], CU_MORSE["mass"])
        vel = _round(maxwell_boltzmann(_rng(3, sid, 10**6), mass, 300.0, KB_METAL, MASS_CONV_METAL), dtype)
        parts.append((pos, vel, _round(mass, dtype), np.zeros(base.shape[0], np.int32), cell))
    md = dict(integrator="nve", dt=1.0, temperature=300.0, friction=0.0, seed=0, n_steps=500)
    return _finish("cfg3", parts, pot, MASS_CONV_METAL, KB_METAL, skin, dtype, ids, md=md)


# ------------------------------------------------------------------------------- cfg4 (R13, R14, R24)
FIRE_DEFAULTS = dict(dt_start=0.02, dt_max=0.2, f_inc=1.1, f_dec=0.5, alpha_start=0.1, f_alpha=0.99,
                     f_max=1e-4, n_min=5, max_steps=50000)


def soft_sphere_binary():
    sig = np.array([1.0, 1.4])
    sij = 0.5 * (sig[:, None] + sig[None, :])
    one = np.ones((2, 2))
    return Potential("soft_sphere", 2, one.copy(), sij, 2.0 * one, sij.copy(), True)


def cfg4(system_ids, n_atoms=256, dtype="f64", clean=True, phi=0.9, w=None):
    """BASELINE.json:configs[3]: 50:50 soft-sphere mixture at packing fraction 0.9, stream ids."""
    pot = soft_sphere_binary()
    skin = 0.3
    nh = n_atoms // 2
    typ = np.concatenate([np.zeros(nh, np.int32), np.ones(n_atoms - nh, np.int32)])
    sig = np.where(typ == 0, 1.0, 1.4)
    L = (np.sum(np.pi / 6.0 * sig ** 3) / phi) ** (1.0 / 3.0)
    cell = _round(np.eye(3) * L, dtype)
    radii = sorted(set(np.unique(pot.rc).tolist() + [pot.rc_max + skin]))
    parts = []
    for sid in system_ids:
        draw = lambda r, n: r.uniform(0.0, L, size=(n, 3))
        if clean:
            pos = _clean(np.zeros((n_atoms, 3)), draw, cell, radii, w or reject_width(dtype), dtype, (4, sid))
        else:
            pos = _round(draw(_rng(4, sid, 0), n_atoms), dtype)
        parts.append((pos, np.zeros((n_atoms, 3)), np.ones(n_atoms), typ, cell))
    return _finish("cfg4", parts, pot, 1.0, 1.0, skin, dtype, list(system_ids), fire=dict(FIRE_DEFAULTS))


# ------------------------------------------------------------------------------- cfg5 (R33)
def cfg5_start(system_ids, n_atoms=1000, rho=0.8442, dtype="f32"):
    """Uniform random starting positions for the LJ liquid (before the 200-step soft-sphere FIRE
    pre-relaxation that R33 runs with the library itself); soft-sphere eps=sigma=1, exponent 2."""
    L = (n_atoms / rho) ** (1.0 / 3.0)
    cell = _round(np.eye(3) * L, dtype)
    pot = _single_type("soft_sphere", 1.0, 1.0, 2.0, 1.0)
    parts = []
    for sid in system_ids:
        pos = _round(_rng(5, sid, 0).uniform(0.0, L, size=(n_atoms, 3)), dtype)
        parts.append((pos, np.zeros((n_atoms, 3)), np.ones(n_atoms), np.zeros(n_atoms, np.int32), cell))
    fire = dict(FIRE_DEFAULTS, dt_start=0.01, dt_max=0.1)
    return _finish("cfg5_start", parts, pot, 1.0, 1.0, 0.3, dtype, list(system_ids), fire=fire)


def cfg5_md(relaxed, dtype="f32", T=0.722):
    """LJ-liquid MD batch from pre-relaxed positions: eps=sigma=1, rc=2.5, skin 0.3, MB at T*."""
    pot = _single_type("lj", 1.0, 1.0, 0.0, 2.5)
    parts = []
    for s in range(relaxed.n_systems):
        a0, a1 = int(relaxed.sys_offset[s]), int(relaxed.sys_offset[s + 1])
        mass = np.ones(a1 - a0)
        vel = _round(maxwell_boltzmann(_rng(5, int(relaxed.sys_uid[s]), 10**6), mass, T, 1.0, 1.0), dtype)
        parts.append((_round(relaxed.pos[a0:a1], dtype), vel, mass, np.zeros(a1 - a0, np.int32), relaxed.cell[s]))
    md = dict(integrator="nve", dt=0.005, temperature=T, friction=0.0, seed=0, n_steps=200)
    return _finish("cfg5", parts, pot, 1.0, 1.0, 0.3, dtype, relaxed.sys_uid, md=md)


def with_(b, **kw):
    return replace(b, **kw)
