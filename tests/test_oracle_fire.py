"""Pins for oracle O6 (FIRE, Bitzek et al. PRL 97, 170201) -- SURVEY.md 8(c) FIRE pin row."""
import numpy as np
import pytest

import workloads as wl


def _morse_dimer(r):
    pot = wl._single_type("morse", 0.3429, 1.3588, 2.866, 6.0)
    pos = np.array([[5.0, 5.0, 5.0], [5.0 + r, 5.0, 5.0]])
    return wl._finish("dimer", [(pos, np.zeros((2, 3)), np.full(2, 63.546), np.zeros(2, np.int32), np.eye(3) * 30.0)], pot,
                      wl.MASS_CONV_METAL, wl.KB_METAL, 0.0, "f64", [0])


P = dict(dt_start=1.0, dt_max=10.0, f_inc=1.1, f_dec=0.5, alpha_start=0.1, f_alpha=0.99, f_max=1e-8, n_min=5, max_steps=5000)


def test_fire_dimer_converges_to_r0(orc):
    b = _morse_dimer(3.3)
    r = orc.fire_run(b, P, 5000)
    st = r["state"]
    assert st["status"][0] == orc.FIRE_CONVERGED and 0 < st["nsteps"][0] < 2000
    assert np.linalg.norm(r["pos"][1] - r["pos"][0]) == pytest.approx(2.866, abs=1e-7)
    assert r["fmax"][0] < P["f_max"]
    V, _ = orc.pair_potential("morse", 0.3429, 1.3588, 2.866, 6.0, True, 2.866)
    assert r["E"][0] == pytest.approx(V, rel=1e-10)


def test_fire_step_rules(orc):
    """Step one at a time: dt <= dt_max always; P <= 0 => v = 0, dt halves, alpha resets, N_pos = 0;
    after more than n_min downhill steps dt grows by f_inc and alpha shrinks by f_alpha."""
    b = _morse_dimer(3.6)
    st, cur = None, b
    saw_uphill = saw_growth = False
    for _ in range(300):
        prev = st
        r = orc.fire_run(cur, P, 1, state=st)
        st = r["state"]
        if st["status"][0] == orc.FIRE_CONVERGED:
            break
        assert st["dt"][0] <= P["dt_max"] * (1 + 1e-15)
        if prev is not None and prev["status"][0] == orc.FIRE_RUNNING:
            if st["dt"][0] < prev["dt"][0]:
                saw_uphill = True
                assert st["dt"][0] == prev["dt"][0] * P["f_dec"] and st["alpha"][0] == P["alpha_start"]
                assert st["npos"][0] == 0 and not r["vel"].any()
            else:
                assert st["npos"][0] == prev["npos"][0] + 1
                if st["npos"][0] > P["n_min"]:
                    saw_growth = True
                    assert st["dt"][0] == min(prev["dt"][0] * P["f_inc"], P["dt_max"])
                    assert st["alpha"][0] == prev["alpha"][0] * P["f_alpha"]
                else:
                    assert st["dt"][0] == prev["dt"][0] and st["alpha"][0] == prev["alpha"][0]
        cur = wl.with_(cur, pos=r["pos"], vel=r["vel"])
    assert saw_uphill and saw_growth and st["status"][0] == orc.FIRE_CONVERGED


def test_fire_batch_chunk_independence_and_freeze(orc):
    ids = [0, 1, 2]
    p = dict(wl.FIRE_DEFAULTS, f_max=1e-3)
    b = wl.cfg4(ids, n_atoms=32, clean=False)
    whole = orc.fire_run(b, p, 400)
    # one system alone gives bit-identical results (R22, O7)
    for k, sid in enumerate(ids):
        solo = orc.fire_run(wl.cfg4([sid], n_atoms=32, clean=False), p, 400)
        a0, a1 = b.sys_offset[k], b.sys_offset[k + 1]
        assert np.array_equal(solo["pos"], whole["pos"][a0:a1])
        assert solo["state"]["nsteps"][0] == whole["state"]["nsteps"][k]
    # chunked stepping (K_check cadence) cannot change the result; frozen systems stay bitwise unchanged
    cur, st = b, None
    for _ in range(40):
        r = orc.fire_run(cur, p, 10, state=st)
        st = r["state"]
        cur = wl.with_(cur, pos=r["pos"], vel=r["vel"])
    assert np.array_equal(r["pos"], whole["pos"]) and np.array_equal(st["nsteps"], whole["state"]["nsteps"])
    assert np.all(st["status"] == orc.FIRE_CONVERGED)
    # final state passes the criterion when re-evaluated from scratch (R30 ii)
    F = orc.energy_forces(cur)["F"]
    for k in range(3):
        a0, a1 = b.sys_offset[k], b.sys_offset[k + 1]
        assert np.linalg.norm(F[a0:a1], axis=1).max() < p["f_max"]


def test_fire_already_converged_and_max_steps(orc):
    base, cell = wl.lattice(wl._FCC, 5.26, (2, 2, 2))
    b = wl.cfg1(n_systems=1, reps=2, clean=False)
    b.pos = base                                                    # perfect lattice: F = 0
    r = orc.fire_run(b, dict(P, f_max=1e-6), 10)
    assert r["state"]["status"][0] == orc.FIRE_CONVERGED and r["state"]["nsteps"][0] == 0
    assert np.array_equal(r["pos"], base)
    r = orc.fire_run(_morse_dimer(3.3), dict(P, max_steps=3), 10)
    assert r["state"]["status"][0] == orc.FIRE_FAILED and r["state"]["nsteps"][0] == 3
