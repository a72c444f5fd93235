"""Pins for oracle O3 (velocity Verlet), O4 (BAOAB) and O5 (Philox + Box-Muller)."""
import copy
import os

import numpy as np
import pytest

import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------------------- O5
def test_philox_known_answers(orc):
    n = 0
    for line in open(os.path.join(GOLD, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        assert orc.philox4x32_10(w[0:4], w[4:6]).tolist() == w[6:10]
        n += 1
    assert n == 3


def test_philox_counter_layout_and_box_muller(orc):
    seed, uid, local, step = 0x1234567890ABCDEF, 77, 5, (3 << 32) | 9
    words = orc.philox4x32_10([local, uid, step & 0xffffffff, step >> 32], [seed & 0xffffffff, seed >> 32])
    xi = orc.langevin_xi(seed, uid, local, step)
    assert np.array_equal(xi, orc.normals_from_words(words))
    u = (words.astype(np.float64) + 0.5) / 2.0 ** 32
    exp = [np.sqrt(-2 * np.log(u[0])) * np.cos(2 * np.pi * u[1]), np.sqrt(-2 * np.log(u[0])) * np.sin(2 * np.pi * u[1]),
           np.sqrt(-2 * np.log(u[2])) * np.cos(2 * np.pi * u[3])]
    assert np.allclose(xi, exp, rtol=1e-13, atol=1e-15)
    # extreme words: never NaN/Inf; tails truncate at sqrt(2*33*ln2) = 6.764 sigma (R19)
    x0 = orc.normals_from_words([0, 0, 0, 0])
    assert np.all(np.isfinite(x0)) and x0[0] == pytest.approx(np.sqrt(66 * np.log(2.0)), rel=1e-9)
    x1 = orc.normals_from_words([0xffffffff] * 4)
    assert np.all(np.isfinite(x1)) and np.abs(x1).max() < 1e-4
    # distinct (atom, system, step) give distinct streams
    assert not np.array_equal(orc.langevin_xi(42, 0, 1, 0), orc.langevin_xi(42, 1, 0, 0))
    assert not np.array_equal(orc.langevin_xi(42, 0, 0, 1), orc.langevin_xi(42, 0, 0, 0))


def test_normal_moments(orc):
    xs = np.array([orc.langevin_xi(42, s, i, t) for s in range(4) for i in range(500) for t in range(5)]).ravel()
    n = xs.size
    assert abs(xs.mean()) < 4 / np.sqrt(n)
    assert abs(xs.var() - 1) < 4 * np.sqrt(2 / n)
    assert abs(np.mean(xs ** 4) - 3) < 4 * np.sqrt(96 / n)


# ------------------------------------------------------------------------------- O3
def test_nve_time_reversibility(orc):
    b = wl.cfg1(n_systems=1, reps=3, clean=False)
    r = orc.md_run(b, "nve", 2.0, 40)
    bb = copy.deepcopy(b)
    bb.pos, bb.vel = r["pos"], -r["vel"]
    r2 = orc.md_run(bb, "nve", 2.0, 40)
    assert np.abs(r2["pos"] - b.pos).max() < 1e-9
    assert np.abs(r2["vel"] + b.vel).max() < 1e-12


def test_nve_second_order_and_cfg1_drift_bound(orc):
    b = wl.cfg1()
    n = b.n_atoms / b.n_systems
    r = orc.md_run(b, "nve", 2.0, 100, history=True)
    etot = r["epot_hist"] + r["ke_hist"]
    drift = np.abs(etot - etot[0]).max() / n
    assert drift <= 2e-6                                     # stated bound, SURVEY 8(c) NVE pin (eV/atom)
    r_half = orc.md_run(b, "nve", 1.0, 200, history=True)
    e2 = r_half["epot_hist"] + r_half["ke_hist"]
    ratio = np.abs(etot - etot[0]).max() / np.abs(e2 - e2[0]).max()
    assert 3.0 <= ratio <= 5.0                               # second-order integrator
    # R16: what a step leaves behind -- E, KE returned are those of the final state
    assert np.array_equal(r["E"], r["epot_hist"][-1]) and np.array_equal(r["KE"], r["ke_hist"][-1])
    fin = copy.deepcopy(b); fin.pos, fin.vel = r["pos"], r["vel"]
    assert np.allclose(orc.energy_forces(fin)["F"], r["F"], atol=0) and np.allclose(orc.kinetic(fin), r["KE"], rtol=1e-15)


def test_kinetic_energy_definition(orc):
    b = wl.cfg1(n_systems=2, clean=False)
    ke = orc.kinetic(b)
    exp = [0.5 * np.sum(b.mass[a0:a1, None] * b.mass_conv * b.vel[a0:a1] ** 2) for a0, a1 in zip(b.sys_offset[:-1], b.sys_offset[1:])]
    assert np.allclose(ke, exp, rtol=1e-13)
    # MB at 50 K: T_kin = 2 KE / (3 N kB) within 5 sigma of 50 K
    T = 2 * ke / (3 * 256 * b.kB)
    assert np.all(np.abs(T - 50) < 5 * 50 * np.sqrt(2 / (3 * 256)))


# ------------------------------------------------------------------------------- O4
def test_baoab_gamma_zero_is_velocity_verlet_bitwise(orc):
    b = wl.cfg1(n_systems=2, reps=2, clean=False)
    a = orc.md_run(b, "nve", 2.0, 5)
    c = orc.md_run(b, "baoab", 2.0, 5, temperature=80.0, friction=0.0, seed=42)
    # with gamma = 0: c1 = 1, c2 = 0, and x + dt/2 v + dt/2 v vs x + dt v differ only by rounding order
    assert np.abs(a["pos"] - c["pos"]).max() < 1e-12 and np.abs(a["vel"] - c["vel"]).max() < 1e-15


def _free_particles(n=2000, m=39.948):
    pot = wl._single_type("lj", 0.0, 1.0, 0.0, 1.5)          # eps = 0: no forces
    rng = np.random.default_rng(3)
    per = 50                                                 # many small systems: threads split systems
    parts = [(rng.uniform(0, 50, size=(per, 3)), rng.normal(0, 1e-3, size=(per, 3)), np.full(per, m),
              np.zeros(per, np.int32), np.eye(3) * 50.0) for _ in range(n // per)]
    return wl._finish("free", parts, pot, wl.MASS_CONV_METAL, wl.KB_METAL, 0.0, "f64", list(range(n // per)))


def test_baoab_zero_temperature_is_pure_damping(orc):
    b = _free_particles(50)
    dt, g, n = 2.0, 0.01, 7
    r = orc.md_run(b, "baoab", dt, n, temperature=0.0, friction=g, seed=1)
    c1 = np.exp(-g * dt)
    assert c1 == pytest.approx(0.98019867330675530, rel=1e-15)            # cfg2 constant
    assert np.sqrt(1 - c1 * c1) == pytest.approx(0.19801656710406, rel=1e-12)
    assert np.allclose(r["vel"], b.vel * c1 ** n, rtol=1e-13)
    # drift: x_n = x_0 + dt/2 * sum_k (v_k + v_{k+1})
    vs = b.vel[None] * (c1 ** np.arange(n + 1))[:, None, None]
    assert np.allclose(r["pos"], b.pos + 0.5 * dt * (vs[:-1] + vs[1:]).sum(0), rtol=1e-13)


def test_baoab_free_particle_velocity_variance(orc):
    b = _free_particles(3000)
    T = 80.0
    r = orc.md_run(b, "baoab", 2.0, 400, temperature=T, friction=0.05, seed=42)     # 40 relaxation times
    var = r["vel"].var()
    exp = b.kB * T / (39.948 * b.mass_conv)
    assert abs(var / exp - 1) < 5 * np.sqrt(2 / r["vel"].size)
    assert orc.kinetic(wl.with_(b, vel=r["vel"])).sum() == pytest.approx(1.5 * 3000 * b.kB * T, rel=5 * np.sqrt(2 / 9000))


def test_baoab_restart_is_bit_reproducible(orc):
    """Counter-based RNG keyed on the system's own step (R18): 6 steps = 3 + save/restore + 3."""
    b = wl.cfg1(n_systems=2, reps=2, clean=False)
    kw = dict(temperature=80.0, friction=0.01, seed=42, sys_uid=b.sys_uid)
    full = orc.md_run(b, "baoab", 2.0, 6, **kw)
    h1 = orc.md_run(b, "baoab", 2.0, 3, **kw)
    h2 = orc.md_run(wl.with_(b, pos=h1["pos"], vel=h1["vel"]), "baoab", 2.0, 3, step=h1["step"], **kw)
    assert np.array_equal(full["pos"], h2["pos"]) and np.array_equal(full["vel"], h2["vel"])
    # a system's noise does not depend on its batch slot (uid travels with it)
    solo = orc.md_run(wl.take(b, [1]), "baoab", 2.0, 6, **dict(kw, sys_uid=b.sys_uid[[1]]))
    a0 = b.sys_offset[1]
    assert np.array_equal(solo["pos"], full["pos"][a0:])
