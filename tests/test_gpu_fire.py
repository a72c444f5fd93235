"""GPU parity for FIRE and the in-flight swap (a10) through the C ABI."""
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


@pytest.mark.parametrize("engine", [0, 1])
def test_fire_first_100_steps_match_oracle(ts, orc, engine):
    """R30(i): state after the first 100 FIRE steps to 1e-8, including the per-system scalars."""
    b = wl.cfg4(range(5))
    o = orc.fire_run(b, b.fire, 100)
    st = ts.SimState(b, engine=engine)
    st.fire_step(b.fire, 100)
    assert st.poll().flags == 0
    mask, status, steps = st.converged_mask()
    assert np.array_equal(status, o["state"]["status"])
    assert np.array_equal(steps, o["state"]["nsteps"])
    assert np.abs(st.numpy("pos") - o["pos"]).max() <= 1e-8
    assert np.abs(st.numpy("vel") - o["vel"]).max() <= 1e-8
    assert np.allclose(st.numpy("energy"), o["E"], rtol=1e-9)
    st.close()


@pytest.mark.parametrize("engine", [0, 1])
def test_fire_split_calls_equal_one_call(ts, engine):
    """R22: results are independent of the host's check cadence."""
    b = wl.cfg4(range(3))
    a = ts.SimState(b, engine=engine)
    a.fire_step(b.fire, 60)
    c = ts.SimState(b, engine=engine)
    for _ in range(6):
        c.fire_step(b.fire, 10)
    assert np.abs(a.numpy("pos") - c.numpy("pos")).max() <= 1e-10
    assert np.array_equal(a.converged_mask()[2], c.converged_mask()[2])
    a.close(); c.close()


@pytest.mark.parametrize("engine", [0, 1])
def test_fire_converges_and_freezes(ts, orc, engine):
    """R30(ii): the GPU's final positions, re-evaluated by the oracle, satisfy the criterion and the
    energies agree to 1e-12; frozen systems stay bitwise unchanged under further calls (R22)."""
    b = wl.cfg4(range(4), n_atoms=64)
    fire = dict(b.fire, f_max=1e-4, max_steps=20000)
    st = ts.SimState(b, engine=engine)
    for _ in range(400):
        st.fire_step(fire, 50)
        mask, status, steps = st.converged_mask()
        if mask.all():
            break
    assert mask.all(), (status, steps)
    pos = st.numpy("pos").copy()
    vel = st.numpy("vel").copy()
    E = st.numpy("energy").copy()
    bb = wl.with_(b, pos=pos)
    o = orc.energy_forces(bb)
    fmax = np.array([np.linalg.norm(o["F"][64 * s:64 * (s + 1)], axis=1).max() for s in range(4)])
    assert np.all(fmax < 1e-4 * (1 + 1e-6))
    assert np.all(np.abs(E - o["E"]) <= 1e-12 * np.maximum(np.abs(o["E"]), o["Eabs"]))
    st.fire_step(fire, 25)                                     # all frozen: nothing may change
    assert np.array_equal(st.numpy("pos"), pos) and np.array_equal(st.numpy("vel"), vel)
    assert np.array_equal(st.converged_mask()[2], steps)
    # oracle's own step counts, reported (R30(iii)): chaotic dynamics may differ late, so compare loosely
    oo = orc.fire_run(b, fire, 20000)
    assert np.all(oo["state"]["status"] == 2)
    print("fire steps gpu", steps, "oracle", oo["state"]["nsteps"])
    st.close()


@pytest.mark.parametrize("engine", [0, 1])
def test_fire_max_steps_marks_failed(ts, engine):
    b = wl.cfg4(range(2), n_atoms=64)
    fire = dict(b.fire, f_max=1e-12, max_steps=7)
    st = ts.SimState(b, engine=engine)
    st.fire_step(fire, 20)
    mask, status, steps = st.converged_mask()
    assert list(status) == [ts.TS_FIRE_FAILED] * 2 and list(steps) == [7, 7]
    rep = st.poll()
    assert rep.n_failed == 2 and rep.n_converged == 0
    st.close()


@pytest.mark.parametrize("engine", [0, 1])
def test_swap_gives_batch_independent_results(ts, orc, engine):
    """O7 / R18: a system's trajectory does not depend on the slot or batch it travels in."""
    b = wl.cfg4(range(4), n_atoms=64)
    st = ts.SimState(b, engine=engine)
    st.fire_step(b.fire, 30)
    fresh = wl.cfg4([10, 11], n_atoms=64)
    st.swap_systems([2, 0], fresh)                             # id 10 -> slot 2, id 11 -> slot 0
    mask, status, steps = st.converged_mask()
    assert status[2] == ts.TS_FIRE_FRESH and status[0] == ts.TS_FIRE_FRESH and steps[2] == 0
    st.fire_step(b.fire, 40)
    assert st.poll().flags == 0
    pos = st.numpy("pos")
    o_new = orc.fire_run(fresh, b.fire, 40)
    o_old = orc.fire_run(wl.take(b, [1, 3]), b.fire, 70)
    assert np.abs(pos[128:192] - o_new["pos"][0:64]).max() <= 1e-8
    assert np.abs(pos[0:64] - o_new["pos"][64:128]).max() <= 1e-8
    assert np.abs(pos[64:128] - o_old["pos"][0:64]).max() <= 1e-8
    assert np.abs(pos[192:256] - o_old["pos"][64:128]).max() <= 1e-8
    st.close()


def test_swap_baoab_noise_follows_sys_uid(ts, orc):
    """R18: the Philox counter uses (sys_uid, local index, the system's own step)."""
    b = wl.cfg2(n_systems=2, reps=3, dtype="f64")
    md = dict(b.md)
    st = ts.SimState(b, engine=0)
    st.md_step(md, 10)
    fresh = wl.cfg2(n_systems=1, reps=3, dtype="f64", system_ids=[7])
    st.swap_systems([0], fresh)
    st.md_step(md, 15)
    o = orc.md_run(fresh, "baoab", md["dt"], 15, temperature=md["temperature"], friction=md["friction"],
                   seed=md["seed"], sys_uid=fresh.sys_uid)
    n = fresh.n_atoms
    assert np.abs(st.numpy("pos")[:n] - o["pos"]).max() <= 1e-9
    o2 = orc.md_run(wl.take(b, [1]), "baoab", md["dt"], 25, temperature=md["temperature"], friction=md["friction"],
                    seed=md["seed"], sys_uid=[b.sys_uid[1]])
    assert np.abs(st.numpy("pos")[n:] - o2["pos"]).max() <= 1e-9
    assert list(st.get_system_steps()) == [15, 25]
    st.close()


def test_overflow_is_detected_and_nothing_is_written_past_capacity(ts):
    """A workspace sized for a dilute batch must flag overflow when the same slots receive a dense one."""
    b = wl.cfg4(range(2), n_atoms=64, phi=0.3)
    st = ts.SimState(b, slack=1.0, engine=0)
    dense = wl.cfg4([5, 6], n_atoms=64, phi=0.9)
    dense = wl.with_(dense, cell=dense.cell * 0.55, pos=dense.pos * 0.55)   # ~6x the density
    st.swap_systems([0, 1], dense)
    st.build_neighbors()
    rep = st.poll()
    assert rep.flags & ts.TS_FLAG_NBR_OVERFLOW and rep.list_valid == 0
    with pytest.raises(ts.TsError) as e:
        st.compute_forces()
    assert e.value.code == 8                                   # TS_ERR_STICKY until cleared
    st.close()
