"""GPU parity: the CUDA path (through the C ABI) against the fp64 CPU oracle, element by element, on
the same seeded inputs.  Tolerances are BASELINE.json:north_star's: pair sets bit-exact; fp64 E rel
1e-12, F abs 1e-10, x after 100 steps 1e-8; fp32 F within 1e-4 of the system's max |F|, E rel 1e-5
(R31: relative to max(|E|, sum 1/2 |V|))."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ts():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2508_06628_b200 as m
    m.lib()
    return m


ENGINES = [0, 1]


def _cases():
    """Small batches shaped like the five configs: several tiles, ragged tails, tiny sheared boxes."""
    c = {}
    c["cfg1_f64"] = lambda: wl.cfg1(n_systems=4)
    c["cfg2_f32"] = lambda: wl.cfg2(n_systems=3, dtype="f32")
    c["cfg2_f64"] = lambda: wl.cfg2(n_systems=2, dtype="f64")
    c["cfg3_f32"] = lambda: wl.cfg3(n_systems=12, dtype="f32", n_range=(32, 700))
    c["cfg3_f64"] = lambda: wl.cfg3(n_systems=8, dtype="f64", n_range=(32, 400))
    c["cfg4_f64"] = lambda: wl.cfg4(range(6))
    c["tiny_f64"] = lambda: wl.cfg1(n_systems=2, reps=1)       # 4 atoms, box 5.26 A << r_c: self images
    c["small_f64"] = lambda: wl.cfg1(n_systems=3, reps=2)      # 32 atoms, box 10.52 A < 2 r_list
    return c


CASES = _cases()


def _pair_sets(orc, b, R):
    out = []
    for s in range(b.n_systems):
        a0, a1 = int(b.sys_offset[s]), int(b.sys_offset[s + 1])
        i, j, S, _ = orc.pairs(b.pos[a0:a1], b.cell[s], R)
        out.append(set(zip((i + a0).tolist(), (j + a0).tolist(), S[:, 0].tolist(), S[:, 1].tolist(), S[:, 2].tolist())))
    return out


@pytest.mark.parametrize("name", list(CASES))
def test_neighbour_pair_sets_bit_exact(ts, orc, name):
    b = CASES[name]()
    st = ts.SimState(b, engine=0)
    st.build_neighbors()
    off, j, shift = st.get_neighbors()
    rep = st.poll()
    assert rep.flags == 0 and rep.list_valid == 1
    i = np.repeat(np.arange(b.n_atoms), np.diff(off))
    got = set(zip(i.tolist(), j.tolist(), shift[:, 0].tolist(), shift[:, 1].tolist(), shift[:, 2].tolist()))
    assert len(got) == j.size                                  # no duplicate (i, j, S)
    want = set().union(*_pair_sets(orc, b, b.r_list))
    assert got == want
    assert rep.nnz == len(want) and rep.nnz <= rep.nnz_capacity
    assert rep.max_neighbors == int(np.diff(off).max())
    st.close()


def _check_efw(b, st, o, fp32):
    E, F, W = st.numpy("energy"), st.numpy("force").astype(np.float64), st.numpy("virial")
    scale = np.maximum(np.abs(o["E"]), o["Eabs"])
    if fp32:
        assert np.all(np.abs(E - o["E"]) <= 1e-5 * scale)
        for s in range(b.n_systems):
            a0, a1 = int(b.sys_offset[s]), int(b.sys_offset[s + 1])
            fmax = np.linalg.norm(o["F"][a0:a1], axis=1).max()
            assert np.abs(F[a0:a1] - o["F"][a0:a1]).max() <= 1e-4 * fmax
        wscale = np.abs(o["W"]).reshape(b.n_systems, -1).max(1) + o["Eabs"]
        assert np.all(np.abs(W - o["W"]).reshape(b.n_systems, -1).max(1) <= 1e-4 * wscale)
    else:
        assert np.all(np.abs(E - o["E"]) <= 1e-12 * scale)
        assert np.abs(F - o["F"]).max() <= 1e-10
        wscale = np.abs(o["W"]).reshape(b.n_systems, -1).max(1) + o["Eabs"]
        assert np.all(np.abs(W - o["W"]).reshape(b.n_systems, -1).max(1) <= 1e-11 * wscale)


@pytest.mark.parametrize("name", list(CASES))
def test_energy_forces_virial(ts, orc, name):
    b = CASES[name]()
    o = orc.energy_forces(b)
    st = ts.SimState(b, engine=0)
    st.compute_forces(ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
    assert st.poll().flags == 0
    _check_efw(b, st, o, b.dtype == "f32")
    KE = st.numpy("kinetic")
    assert np.allclose(KE, orc.kinetic(b), rtol=1e-6 if b.dtype == "f32" else 1e-13, atol=1e-300)
    st.close()


def test_results_do_not_depend_on_skin(ts, orc):
    b = CASES["cfg1_f64"]()
    o = orc.energy_forces(b)
    for skin in (0.0, 0.3, 1.2):
        st = ts.SimState(b, skin=skin, engine=0)
        st.compute_forces()
        _check_efw(b, st, o, False)
        st.close()


@pytest.mark.parametrize("engine", ENGINES)
def test_nve_100_steps_fp64_cfg1(ts, orc, engine):
    b = wl.cfg1(n_systems=4)
    o = orc.md_run(b, "nve", 2.0, 100)
    st = ts.SimState(b, engine=engine)
    st.md_step(b.md, 100)
    rep = st.poll()
    assert rep.flags == 0
    assert np.abs(st.numpy("pos") - o["pos"]).max() <= 1e-8
    assert np.abs(st.numpy("vel") - o["vel"]).max() <= 1e-10
    assert np.abs(st.numpy("force") - o["F"]).max() <= 1e-9
    assert np.allclose(st.numpy("energy"), o["E"], rtol=1e-10)
    assert np.allclose(st.numpy("kinetic"), o["KE"], rtol=1e-10)
    assert np.array_equal(st.get_system_steps(), np.full(4, 100, np.uint64))
    st.close()


@pytest.mark.parametrize("engine", ENGINES)
def test_baoab_100_steps_fp64_cfg2(ts, orc, engine):
    b = wl.cfg2(n_systems=2, dtype="f64")
    md = dict(b.md)
    o = orc.md_run(b, "baoab", md["dt"], 100, temperature=md["temperature"], friction=md["friction"],
                   seed=md["seed"], sys_uid=b.sys_uid)
    st = ts.SimState(b, engine=engine)
    st.md_step(md, 60)
    st.md_step(md, 40)                                         # split call: per-system step counter carries on (R18)
    assert st.poll().flags == 0
    assert np.abs(st.numpy("pos") - o["pos"]).max() <= 1e-8
    assert np.abs(st.numpy("vel") - o["vel"]).max() <= 1e-10
    assert np.allclose(st.numpy("energy"), o["E"], rtol=1e-9)
    st.close()


@pytest.mark.parametrize("engine", ENGINES)
def test_nve_morse_triclinic_fp64(ts, orc, engine):
    b = wl.cfg3(n_systems=6, dtype="f64", n_range=(32, 300))
    o = orc.md_run(b, "nve", 1.0, 100)
    st = ts.SimState(b, engine=engine)
    st.md_step(dict(b.md), 100, ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
    rep = st.poll()
    assert rep.flags == 0 and rep.n_rebuilds >= 1
    assert np.abs(st.numpy("pos") - o["pos"]).max() <= 1e-8
    assert np.allclose(st.numpy("energy"), o["E"], rtol=1e-9)
    assert np.abs(st.numpy("virial") - o["W"]).max() <= 1e-8 * np.abs(o["W"]).max()
    st.close()


@pytest.mark.parametrize("engine", ENGINES)
def test_fp32_replay_parity_after_md(ts, orc, engine):
    """R29: after k fp32 steps the GPU's own positions are fed to the oracle; forces must agree to
    1e-4 of max|F| except for atoms in a pair within 1e-5 A of r_c (counted, not compared)."""
    b = wl.cfg2(n_systems=2, dtype="f32")
    st = ts.SimState(b, engine=engine)
    st.md_step(dict(b.md), 50)
    assert st.poll().flags == 0
    bb = wl.with_(b, pos=st.numpy("pos").astype(np.float64), vel=st.numpy("vel").astype(np.float64))
    o = orc.energy_forces(bb)
    F = st.numpy("force").astype(np.float64)
    rc = b.potential.rc_max
    dont_care = np.zeros(b.n_atoms, bool)
    for s in range(b.n_systems):
        a0, a1 = int(b.sys_offset[s]), int(b.sys_offset[s + 1])
        i, j, S, r2 = orc.pairs(bb.pos[a0:a1], bb.cell[s], rc + 1e-3)
        near = np.abs(np.sqrt(r2) - rc) < 1e-5
        dont_care[a0 + i[near]] = True
    assert dont_care.mean() < 0.01
    for s in range(b.n_systems):
        a0, a1 = int(b.sys_offset[s]), int(b.sys_offset[s + 1])
        ok = ~dont_care[a0:a1]
        fmax = np.linalg.norm(o["F"][a0:a1], axis=1).max()
        assert np.abs(F[a0:a1] - o["F"][a0:a1])[ok].max() <= 1e-4 * fmax
    scale = np.maximum(np.abs(o["E"]), o["Eabs"])
    assert np.all(np.abs(st.numpy("energy") - o["E"]) <= 1e-5 * scale)
    st.close()


@pytest.mark.parametrize("engine", ENGINES)
def test_fp32_baoab_noise_follows_the_oracle_stream(ts, orc, engine):
    """fp32 runs evaluate log / sin / cos with the hardware approximations (R19).  After ONE BAOAB
    step the fp32 velocities must still be the oracle's to fp32 accuracy: same Philox counters, same
    Box-Muller pairing of the words, same signs.  The kick from the noise is c2 sqrt(kT/m) xi
    (~2.5e-4 A/fs per unit normal), so 2e-7 A/fs absolute resolves a 1e-3 error on xi."""
    b = wl.cfg2(n_systems=2, dtype="f32")
    md = dict(b.md)
    o = orc.md_run(b, "baoab", md["dt"], 1, temperature=md["temperature"], friction=md["friction"],
                   seed=md["seed"], sys_uid=b.sys_uid)
    st = ts.SimState(b, engine=engine)
    st.md_step(md, 1)
    assert st.poll().flags == 0
    dv = np.abs(st.numpy("vel").astype(np.float64) - o["vel"])
    assert dv.max() <= 2e-7
    assert np.abs(st.numpy("pos").astype(np.float64) - o["pos"]).max() <= 2e-5
    st.close()


@pytest.mark.parametrize("engine", ENGINES)
def test_nve_binary_soft_sphere_fp64(ts, orc, engine):
    """Two atom types (per-pair parameter table) under MD: the resident engine's generic, multi-type pair path and the
    general engine against the oracle (the cfg4 mixture, here with velocities and velocity Verlet instead of FIRE)."""
    b = wl.cfg4(range(5), n_atoms=200)
    rng = np.random.Generator(np.random.PCG64(12345))
    b = wl.with_(b, vel=rng.normal(0.0, 0.3, size=b.vel.shape))
    md = dict(integrator="nve", dt=0.004, temperature=0.0, friction=0.0, seed=0)
    o = orc.md_run(b, "nve", md["dt"], 60)
    st = ts.SimState(b, engine=engine)
    st.md_step(md, 60, ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
    rep = st.poll()
    assert rep.flags == 0 and rep.engine == engine
    assert np.abs(st.numpy("pos") - o["pos"]).max() <= 1e-8
    assert np.abs(st.numpy("force") - o["F"]).max() <= 1e-8
    assert np.allclose(st.numpy("energy"), o["E"], rtol=1e-9)
    assert np.abs(st.numpy("virial") - o["W"]).max() <= 1e-8 * np.abs(o["W"]).max()
    st.close()


def test_resident_engine_is_deterministic(ts):
    """Fixed reduction orders, no atomics on the physics: two runs of the same batch agree bit for bit (positions,
    velocities, forces, energies, virials), for MD and for FIRE."""
    b = wl.cfg2(n_systems=3, dtype="f32")
    outs = []
    for _ in range(2):
        st = ts.SimState(b, engine=1)
        st.md_step(dict(b.md), 120, ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
        assert st.poll().flags == 0 and st.poll().engine == 1
        outs.append([st.numpy(k).copy() for k in ("pos", "vel", "force", "energy", "virial", "kinetic")])
        st.close()
    for a, c in zip(*outs):
        assert np.array_equal(a, c)
    f = wl.cfg4(range(4), n_atoms=128)
    outs = []
    for _ in range(2):
        st = ts.SimState(f, engine=1)
        st.fire_step(f.fire, 150)
        assert st.poll().flags == 0 and st.poll().engine == 1
        outs.append([st.numpy(k).copy() for k in ("pos", "vel", "force", "energy")])
        st.close()
    for a, c in zip(*outs):
        assert np.array_equal(a, c)


def test_rows_longer_than_the_build_buffer(ts, orc):
    """General engine: a list radius with more than 256 neighbours per atom (the shared-memory row buffer of the
    one-pass neighbour search): the long rows take the second walk; pair sets stay bit-exact, E / F / W in tolerance."""
    b = wl.cfg1(n_systems=2, reps=4)
    st = ts.SimState(b, skin=6.0, engine=0)                    # r_list = 14.5 A: ~350 neighbours per atom
    st.compute_forces(ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
    off, j, shift = st.get_neighbors()
    rep = st.poll()
    assert rep.flags == 0 and rep.list_valid == 1 and rep.max_neighbors > 256
    i = np.repeat(np.arange(b.n_atoms), np.diff(off))
    got = set(zip(i.tolist(), j.tolist(), shift[:, 0].tolist(), shift[:, 1].tolist(), shift[:, 2].tolist()))
    want = set().union(*_pair_sets(orc, b, b.potential.rc_max + 6.0))
    assert got == want and len(got) == j.size
    _check_efw(b, st, orc.energy_forces(b), False)
    st.close()


RESIDENT_STATIC = {
    "cfg1_f64": lambda: wl.cfg1(n_systems=4),
    "cfg2_f32": lambda: wl.cfg2(n_systems=3, dtype="f32"),
    "cfg2_f64": lambda: wl.cfg2(n_systems=2, dtype="f64"),
    "cfg3_f32": lambda: wl.cfg3(n_systems=6, dtype="f32", n_range=(500, 900)),
    "cfg3_f64": lambda: wl.cfg3(n_systems=4, dtype="f64", n_range=(500, 700)),
    "cfg4_f64": lambda: wl.cfg4(range(6)),
    "cfg4_f32": lambda: wl.cfg4(range(4), dtype="f32"),
}


@pytest.mark.parametrize("name", list(RESIDENT_STATIC))
def test_resident_engine_static_energy_forces_virial(ts, orc, name):
    """The pair phase of the system-resident engine at step 0 (no integration): E, F and the 3x3 virial of LJ, Morse
    and the two-type soft-sphere table against the oracle, fp32 and fp64, element by element."""
    b = RESIDENT_STATIC[name]()
    o = orc.energy_forces(b)
    st = ts.SimState(b, engine=1)
    st.md_step(dict(b.md) if b.md else dict(integrator="nve", dt=1.0), 0, ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
    rep = st.poll()
    assert rep.flags == 0 and rep.engine == 1, (rep.flags, rep.engine)
    _check_efw(b, st, o, b.dtype == "f32")
    st.close()


@pytest.mark.parametrize("name", ["cfg2_f32", "cfg2_f64", "cfg5_f32", "cfg4_f64"])
def test_resident_list_is_a_tight_superset_of_the_oracle_pair_set(ts, orc, name):
    """The list of the benched (system-resident) engine, exported and decoded: it contains every oracle pair within
    r_list and nothing beyond r_list plus the documented inflation (a few 1e-6 of the longest cell edge), on cfg2- and
    cfg5-shaped systems and on the two-type mixture; also after the atoms have moved (a list built mid-trajectory)."""
    if name.startswith("cfg2"):
        b = wl.cfg2(n_systems=2, dtype=name[-3:])
    elif name == "cfg5_f32":
        start = wl.cfg5_start(range(2))                        # R33: random positions pre-relaxed by the library itself
        sf = ts.SimState(start)
        sf.fire_step(dict(start.fire, f_max=1e-12, max_steps=10 ** 6), 200)
        b = wl.cfg5_md(wl.with_(start, pos=sf.numpy("pos").astype(np.float64)))
        sf.close()
    else:
        b = wl.cfg4(range(3))
    st = ts.SimState(b, engine=1, slack=2.0 if name == "cfg5_f32" else 1.25)
    lmax = max(np.linalg.norm(b.cell[s], axis=1).max() for s in range(b.n_systems))
    for moved in (False, True):
        if moved and b.md:
            st.md_step(dict(b.md), 7)
        pos = st.numpy("pos").astype(np.float64)
        for s in range(b.n_systems):
            a0, a1 = int(b.sys_offset[s]), int(b.sys_offset[s + 1])
            off, j, shift = st.get_resident_neighbors(s)
            i = np.repeat(np.arange(a0, a1), np.diff(off))
            got = set(zip(i.tolist(), j.tolist(), shift[:, 0].tolist(), shift[:, 1].tolist(), shift[:, 2].tolist()))
            assert len(got) == j.size                                              # no duplicate (i, j, S)
            lo = orc.pairs(pos[a0:a1], b.cell[s], b.r_list)
            hi = orc.pairs(pos[a0:a1], b.cell[s], b.r_list + 16e-6 * lmax)
            as_set = lambda p: set(zip((p[0] + a0).tolist(), (p[1] + a0).tolist(), p[2][:, 0].tolist(), p[2][:, 1].tolist(), p[2][:, 2].tolist()))
            assert as_set(lo) <= got <= as_set(hi), (name, s, len(as_set(lo)), len(got), len(as_set(hi)))
    assert st.poll().flags == 0
    st.close()


def test_mixed_engine_dispatch_of_a_ragged_batch(ts, orc):
    """A ragged Morse batch (cfg3-shaped, 32..900 atoms): the systems whose cells are at least 2 r_list high run in the
    system-resident engine, size class by size class, the small ones next to them in the general engine; every system
    follows the oracle (fp64: positions to 1e-8 after 60 steps, E / KE / W), and a later whole-batch call still works."""
    b = wl.cfg3(n_systems=24, dtype="f64", n_range=(32, 900))
    o = orc.md_run(b, "nve", b.md["dt"], 60)
    st = ts.SimState(b, engine=1)
    st.md_step(dict(b.md), 25, ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
    st.md_step(dict(b.md), 35, ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
    rep = st.poll()
    assert rep.flags == 0 and rep.engine == 2, (rep.flags, rep.engine)           # both engines stepped systems
    assert np.abs(st.numpy("pos") - o["pos"]).max() <= 1e-8
    assert np.abs(st.numpy("vel") - o["vel"]).max() <= 1e-10
    assert np.allclose(st.numpy("energy"), o["E"], rtol=1e-10) and np.allclose(st.numpy("kinetic"), o["KE"], rtol=1e-10)
    wscale = np.abs(o["W"]).reshape(b.n_systems, -1).max(1)
    assert np.all(np.abs(st.numpy("virial") - o["W"]).reshape(b.n_systems, -1).max(1) <= 1e-9 * wscale)
    assert np.array_equal(st.get_system_steps(), np.full(b.n_systems, 60, np.uint64))
    st.compute_forces(ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)                     # whole batch through the general engine
    assert st.poll().flags == 0
    assert np.abs(st.numpy("force") - o["F"]).max() <= 1e-9
    st.set_engine(0)
    st.md_step(dict(b.md), 5)
    o2 = orc.md_run(b, "nve", b.md["dt"], 65)
    assert st.poll().engine == 0 and np.abs(st.numpy("pos") - o2["pos"]).max() <= 1e-8
    st.set_engine(1)                                 # back: the lists the resident engine had saved are stale and are rebuilt
    st.md_step(dict(b.md), 5)
    o3 = orc.md_run(b, "nve", b.md["dt"], 70)
    assert st.poll().engine == 2 and np.abs(st.numpy("pos") - o3["pos"]).max() <= 1e-8
    st.close()
