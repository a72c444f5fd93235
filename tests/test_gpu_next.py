"""GPU tests of the rows SURVEY.md 8(f) calls "next" and of the ragged in-flight path of row a10:
ts_repack_systems / RaggedInFlightRelaxer (K12), BinRunner (NEXT-1),
ts_export_edges + external-model stepping (NEXT-2).  Every comparison is with the fp64 CPU
oracle of the system run alone (O7: systems are independent, so batch composition must not matter)."""
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


SIZES = [48, 96, 64, 160, 80, 128, 56, 112, 72, 144, 40, 104]     # atoms of stream id k: SIZES[k % 12]


def _mixed(sid):
    """Stream id -> one soft-sphere system whose size depends on the id (Fig. 3: structures of different sizes)."""
    return wl.cfg4([sid], n_atoms=SIZES[sid % len(SIZES)])


@pytest.mark.parametrize("engine", [0, 1])
def test_repack_keeps_running_systems_and_admits_fresh_ones(ts, orc, engine):
    """ts_repack_systems in the middle of a FIRE run: the kept systems continue exactly as if nothing had happened
    (state after 60 steps equals the oracle's solo run to 1e-8), the fresh ones start at step 0."""
    ids = [0, 1, 2, 3]
    b = wl.concat([_mixed(i) for i in ids])
    fire = dict(b.fire, f_max=1e-30, max_steps=10 ** 6)       # nobody converges: compare raw trajectories
    st = ts.SimState(b, engine=engine)
    st.fire_step(fire, 25)
    fresh = wl.concat([_mixed(7), _mixed(10)])                # 112 + 40 atoms into the room of systems 1 (96) and 3 (160)
    st.repack([2, 0], fresh)                                  # kept in a NEW order: old 2, old 0, then 7, 10
    assert (st.N, st.S) == (64 + 48 + 112 + 40, 4)
    st.fire_step(fire, 35)
    rep = st.poll()
    assert rep.flags == 0 and rep.engine == engine
    pos, steps = st.numpy("pos"), st.converged_mask()[2]
    assert list(steps) == [60, 60, 35, 35]
    off = st.sys_offset
    for k, (sid, n) in enumerate([(2, 60), (0, 60), (7, 35), (10, 35)]):
        one = _mixed(sid)
        o = orc.fire_run(one, dict(one.fire, f_max=1e-30, max_steps=10 ** 6), n)
        assert np.abs(pos[off[k]:off[k + 1]] - o["pos"]).max() <= 1e-8, (sid, n)
    # capacity: a batch that does not fit is refused and nothing changes
    with pytest.raises(ts.TsError) as err:
        st.repack([0, 1, 2, 3], wl.concat([_mixed(3), _mixed(9)]))
    assert err.value.code == ts.TS_ERR_WORKSPACE_TOO_SMALL and (st.N, st.S) == (264, 4)
    st.fire_step(fire, 5)
    assert st.poll().flags == 0 and list(st.converged_mask()[2]) == [65, 65, 40, 40]
    st.close()


def test_ragged_inflight_relaxer_mixed_sizes(ts, orc):
    """A stream of systems of different sizes through one state with a byte budget: every id is relaxed exactly once,
    the capacity is never exceeded, every final state passes the oracle's own convergence check, and the results do
    not depend on the budget or the check cadence (R22)."""
    from paper_2508_06628_b200 import scheduler as sch
    n_total = 14
    fire = dict(_mixed(0).fire, f_max=1e-4, max_steps=20000)
    per = [sch.batch_system_bytes(_mixed(i))[0] for i in range(n_total)]
    r = sch.RaggedInFlightRelaxer(_mixed, n_total, fire, budget_bytes=sum(per[:4]) + 1.0, k_check=10)
    res = r.run()
    assert sorted(res) == list(range(n_total)) and r.unfinished == [] and r.failed == []
    assert r.n_repacks >= 3 and r.peak_systems <= 4 and r.peak_atoms <= sum(SIZES[:4])
    for sid, rec in res.items():
        assert rec["status"] == ts.TS_FIRE_CONVERGED and rec["pos"].shape[0] == SIZES[sid % len(SIZES)]
        o = orc.energy_forces(wl.with_(_mixed(sid), pos=rec["pos"]))
        assert np.sqrt((o["F"] ** 2).sum(1)).max() < fire["f_max"]             # R30(ii)
        assert abs(rec["energy"] - o["E"][0]) <= 1e-12 * max(abs(o["E"][0]), o["Eabs"][0])
    r2 = sch.RaggedInFlightRelaxer(_mixed, n_total, fire, budget_bytes=sum(per[:6]) + 1.0, k_check=7)
    res2 = r2.run()
    for sid in res:
        assert res2[sid]["fire_steps"] == res[sid]["fire_steps"]
        assert np.abs(res2[sid]["pos"] - res[sid]["pos"]).max() <= 1e-6


def test_bin_runner_matches_solo_runs(ts, orc):
    """BinningAutobatcher as a runner: a ragged Morse batch packed into bins by the byte scaler and stepped bin by bin
    on two streams; every system's trajectory equals the oracle run of that system alone."""
    from paper_2508_06628_b200 import scheduler as sch
    b = wl.cfg3(n_systems=9, dtype="f64", n_range=(32, 300))
    costs = sch.batch_system_bytes(b)
    runner = sch.BinRunner(b, budget_bytes=1.05 * max(costs.max(), costs.sum() / 4))
    assert len(runner.bins) >= 3 and sorted(np.concatenate(runner.bins).tolist()) == list(range(9))
    for systems in runner.bins:
        assert costs[systems].sum() <= runner_budget(runner, costs)
    out = runner.run_md(40, ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
    o = orc.md_run(b, "nve", b.md["dt"], 40)
    assert np.abs(out["pos"] - o["pos"]).max() <= 1e-8
    assert np.allclose(out["energy"], o["E"], rtol=1e-10) and np.allclose(out["kinetic"], o["KE"], rtol=1e-10)


def runner_budget(runner, costs):
    return 1.05 * max(costs.max(), costs.sum() / 4)


def _torch_lj_forces(torch, pos, cell, system_idx, edge_index, shift, eps, sigma, rc):
    """The stand-in external model: Lennard-Jones forces from the exported edge list in plain torch ops."""
    i, j = edge_index[0], edge_index[1]
    h = cell[system_idx[i].long()]                                           # [E,3,3], rows = lattice vectors
    rij = pos[j] - pos[i] + torch.einsum("ek,ekc->ec", shift, h)
    r2 = (rij * rij).sum(1)
    inside = r2 < rc * rc
    s6 = (sigma * sigma / r2) ** 3
    g = torch.where(inside, -24.0 * eps * (2.0 * s6 * s6 - s6) / r2, torch.zeros_like(r2))   # V'(r) / r
    F = torch.zeros_like(pos)
    F.index_add_(0, i, g[:, None] * rij)                                     # F_i = sum V'(r) r_ij / r
    return F


def test_edge_export_and_external_model_md(ts, orc):
    """NEXT-2: the list exported on the device is the oracle's pair set at r_list; an external force provider (plain
    torch on the GPU) driven through ts_md_step_external reproduces the oracle's NVE trajectory."""
    import torch
    b = wl.cfg1(n_systems=3, reps=3)                           # 3 x 108 atoms, box 15.78 A < 2 r_list: image shifts matter
    st = ts.SimState(b, engine=0)
    md = ts.md_params(**b.md)
    st.md_step_external(md, ts.TS_PHASE_INIT)
    ei, es = st.export_edges()
    got = set(zip(ei[0].tolist(), ei[1].tolist(), *[es[:, k].to(torch.int64).tolist() for k in range(3)]))
    want = set()
    for s in range(b.n_systems):
        a0, a1 = int(b.sys_offset[s]), int(b.sys_offset[s + 1])
        i, j, S, _ = orc.pairs(b.pos[a0:a1], b.cell[s], b.r_list)
        want |= set(zip((i + a0).tolist(), (j + a0).tolist(), S[:, 0].tolist(), S[:, 1].tolist(), S[:, 2].tolist()))
    assert got == want and len(got) == ei.shape[1]
    pot = b.potential
    eps, sigma, rc = float(pot.p0[0, 0]), float(pot.p1[0, 0]), float(pot.rc[0, 0])
    model = lambda: _torch_lj_forces(torch, st.pos, st.cell, st.system_idx, *st.export_edges(), eps, sigma, rc)
    st.force.copy_(model())
    n = 25
    for _ in range(n):
        st.md_step_external(md, ts.TS_PHASE_PRE)
        st.force.copy_(model())
        st.md_step_external(md, ts.TS_PHASE_POST)
    rep = st.poll()
    assert rep.flags == 0 and rep.steps_done == n
    o = orc.md_run(b, "nve", b.md["dt"], n)
    assert np.abs(st.numpy("pos") - o["pos"]).max() <= 1e-8
    assert np.abs(st.numpy("vel") - o["vel"]).max() <= 1e-10
    assert np.allclose(st.numpy("kinetic"), o["KE"], rtol=1e-10)
    assert np.array_equal(st.get_system_steps(), np.full(3, n, np.uint64))
    st.close()


def test_external_model_fire_matches_library_fire(ts, orc):
    """FIRE driven through ts_fire_step_external with the library's own pair kernel as the "external" provider gives the
    state of ts_fire_step (to rounding: the energy-only and the full pair kernel sum in different orders), and both
    follow the oracle for the first 60 steps."""
    b = wl.cfg4(range(3), n_atoms=64)
    fire = dict(b.fire, f_max=1e-30, max_steps=10 ** 6)
    ref = ts.SimState(b, engine=0)
    ref.fire_step(fire, 60)
    st = ts.SimState(b, engine=0)
    fp = ts.fire_params(**fire)
    st.fire_step_external(fp, ts.TS_PHASE_INIT)
    st.compute_forces(ts.TS_WANT_ENERGY)
    st.fire_step_external(fp, ts.TS_PHASE_CHECK0)
    for _ in range(60):
        st.fire_step_external(fp, ts.TS_PHASE_PRE)
        st.compute_forces(ts.TS_WANT_ENERGY)
        st.fire_step_external(fp, ts.TS_PHASE_POST)
    assert st.poll().flags == 0
    assert np.abs(st.numpy("pos") - ref.numpy("pos")).max() <= 1e-10 and np.abs(st.numpy("vel") - ref.numpy("vel")).max() <= 1e-10
    o = orc.fire_run(b, fire, 60)
    assert np.abs(st.numpy("pos") - o["pos"]).max() <= 1e-8
    assert list(st.converged_mask()[2]) == [60, 60, 60]
    st.close(); ref.close()


# ------------------------------------------------------------------ the resident engine's list across calls
def _chunked_vs_single(ts, b, n, chunk, mode, params):
    """The same run as one call of n steps and as calls of `chunk` steps; returns the two states and rebuild counts."""
    out = []
    for step in (n, chunk):
        st = ts.SimState(b, engine=1)
        r0 = st.poll().resident_rebuilds
        for _ in range(n // step):
            if mode == "md":
                st.md_step(params, step)
            else:
                st.fire_step(params, step)
        rep = st.poll()
        assert rep.flags == 0 and rep.engine == 1
        out.append((st.numpy("pos").copy(), st.numpy("vel").copy(), st.numpy("energy").copy(), rep.resident_rebuilds - r0))
        st.close()
    return out


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_resident_list_survives_calls_md(ts, orc, dtype):
    """Calls of one step continue with the list the last call saved (no build per call): the trajectory is that of one
    long call, the number of list builds is the same (one forced build per system in the first call only), and it
    follows the oracle."""
    b = wl.cfg2(n_systems=3, reps=4, dtype=dtype)                    # 3 x 256 atoms, LJ, BAOAB, clusters of one CTA
    md = ts.md_params(**b.md)
    (p1, v1, e1, rb1), (p2, v2, e2, rb2) = _chunked_vs_single(ts, b, 60, 1, "md", md)
    # not bitwise: the last step of a call computes its forces together with E (another summation order than the
    # forces-only pass of the steps before it), and one-step calls take that pass every step
    tol = 1e-4 if dtype == "f32" else 1e-9
    assert np.abs(p1 - p2).max() <= tol and np.abs(v1 - v2).max() <= tol
    assert abs(rb1 - rb2) <= 3 and rb2 < 3 * 20                      # 60 one-step calls did not build 180 lists
    if dtype == "f64":
        o = orc.md_run(b, "baoab", b.md["dt"], 60, friction=b.md["friction"], temperature=b.md["temperature"], seed=b.md["seed"])
        assert np.abs(p2 - o["pos"]).max() <= 1e-8


def test_resident_list_survives_calls_cluster_of_two(ts):
    """The same with systems large enough for a cluster of two CTAs (every CTA saves its own part)."""
    b = wl.cfg2(n_systems=2, reps=6, dtype="f32")                    # 2 x 864 atoms
    md = ts.md_params(**b.md)
    (p1, v1, e1, rb1), (p2, v2, e2, rb2) = _chunked_vs_single(ts, b, 120, 5, "md", md)
    assert np.abs(p1 - p2).max() <= 1e-4 and np.abs(v1 - v2).max() <= 1e-4 and abs(rb1 - rb2) <= 2 and rb2 < 2 * 24


def test_resident_list_survives_calls_fire_and_swap(ts, orc):
    """FIRE in calls of 5 steps equals FIRE in one call; a swapped-in system gets a fresh build (its slot's saved list
    belonged to the system that left), an invalidated state rebuilds everything."""
    b = wl.cfg4(range(4), n_atoms=64)
    fire = dict(b.fire, f_max=1e-30, max_steps=10 ** 6)
    (p1, v1, e1, rb1), (p2, v2, e2, rb2) = _chunked_vs_single(ts, b, 60, 5, "fire", fire)
    assert np.abs(p1 - p2).max() <= 1e-9 and np.abs(v1 - v2).max() <= 1e-9 and abs(rb1 - rb2) <= 2
    st = ts.SimState(b, engine=1)
    st.fire_step(fire, 20)
    st.swap_systems([2], wl.cfg4([9], n_atoms=64))
    st.fire_step(fire, 20)
    st.fire_step(fire, 20)
    pos, off = st.numpy("pos"), st.sys_offset
    for k, (sid, n) in enumerate([(0, 60), (1, 60), (9, 40), (3, 60)]):
        one = wl.cfg4([sid], n_atoms=64)
        o = orc.fire_run(one, dict(one.fire, f_max=1e-30, max_steps=10 ** 6), n)
        assert np.abs(pos[off[k]:off[k + 1]] - o["pos"]).max() <= 1e-8, sid
    # positions written from outside + ts_invalidate: the saved lists are dropped, the result is that of a fresh state
    new_pos = st.pos.clone()
    new_pos[: int(off[1])] += 0.05
    st.pos.copy_(new_pos)
    st.invalidate()
    st.md_step(ts.md_params(integrator="nve", dt=1e-3), 0, ts.TS_WANT_ENERGY)
    f1, e1 = st.numpy("force").copy(), st.numpy("energy").copy()
    o = orc.energy_forces(wl.with_(b, pos=new_pos.cpu().numpy()))      # cfg4 systems share cell, types and masses
    assert np.abs(f1 - o["F"]).max() <= 1e-9 * max(1.0, np.abs(o["F"]).max())
    st.close()



# ------------------------------------------------------------------ general engine: reproducible reductions
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_general_engine_is_bitwise_reproducible(ts, dtype):
    """E, W, KE and the FIRE sums of the general engine are added in a fixed order (ts_sys_store: per-warp partials in
    slots, added in slot order by a one-warp-per-system kernel), not with floating-point atomics: two runs of the same ragged batch -- systems
    that share warps, systems that span many blocks -- agree bit for bit, trajectories included (FIRE steers by its sums)."""
    b = wl.cfg3(n_systems=12, dtype=dtype, n_range=(32, 1500))
    out = []
    for _ in range(2):
        st = ts.SimState(b, engine=0)
        st.md_step(dict(b.md), 30, ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
        rec = [st.numpy(k).copy() for k in ("pos", "vel", "force", "energy", "virial", "kinetic")]
        st.close()
        out.append(rec)
    for x, y in zip(*out):
        assert np.array_equal(x, y)
    # the same batch in mixed dispatch (resident engine for the systems it holds, general engine next to it)
    out = []
    for _ in range(2):
        st = ts.SimState(b, engine=1)
        st.md_step(dict(b.md), 12, ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
        st.md_step(dict(b.md), 18, ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
        assert st.poll().engine == 2
        out.append([st.numpy(k).copy() for k in ("pos", "vel", "force", "energy", "virial", "kinetic")])
        st.close()
    for x, y in zip(*out):
        assert np.array_equal(x, y)
    c = wl.cfg4(range(9), n_atoms=96, dtype=dtype if dtype == "f64" else "f32")
    fire = dict(c.fire, f_max=1e-30, max_steps=10 ** 6)
    out = []
    for _ in range(2):
        st = ts.SimState(c, engine=0)
        st.fire_step(fire, 80)
        out.append([st.numpy(k).copy() for k in ("pos", "vel", "energy")])
        st.close()
    for x, y in zip(*out):
        assert np.array_equal(x, y)


# ------------------------------------------------------------------ degenerate systems
def _degenerate_batch(dtype="f64"):
    """One atom alone in a big box, two atoms out of each other's reach, a dilute gas whose rows are mostly empty, a
    crystal, and a single atom in a box so small that it sees its own images: the empty and the self-image corners of
    the list code, ragged in one batch (argon Lennard-Jones, r_c 8.5, skin 1.0)."""
    rng = np.random.default_rng(20260511)
    pot = wl._single_type("lj", wl.LJ_AR["eps"], wl.LJ_AR["sigma"], 0.0, wl.LJ_AR["rc"])
    m = wl.LJ_AR["mass"]

    def part(pos, L, v_scale=1e-3):
        pos = np.asarray(pos, dtype=np.float64)
        vel = rng.normal(0.0, v_scale, size=pos.shape)
        return (pos, vel, np.full(pos.shape[0], m), np.zeros(pos.shape[0], np.int32), np.eye(3) * L)

    crystal = wl.cfg1(n_systems=1, reps=4, dtype=dtype)                      # 256 atoms, 21 A box
    parts = [part([[3.0, 4.0, 5.0]], 40.0),
             part([[1.0, 1.0, 1.0], [21.0, 20.0, 19.0]], 40.0),
             part(rng.uniform(0.0, 60.0, size=(40, 3)), 60.0),
             (crystal.pos, crystal.vel, crystal.mass, crystal.type, crystal.cell[0]),
             part([[0.5, 0.25, 0.125]], 7.0)]                                 # images at 7 A < r_c on every axis
    md = dict(integrator="nve", dt=2.0, temperature=0.0, friction=0.0, seed=1)
    return wl._finish("degenerate", parts, pot, wl.MASS_CONV_METAL, wl.KB_METAL, 1.0, dtype, list(range(5)), md=md)


@pytest.mark.parametrize("engine", [0, 1])
def test_degenerate_systems_empty_rows_and_self_images(ts, orc, engine):
    b = _degenerate_batch()
    o0 = orc.energy_forces(b)
    assert o0["E"][0] == 0.0 and o0["E"][1] == 0.0 and o0["E"][4] != 0.0     # nothing in reach / only its own images
    st = ts.SimState(b, engine=engine)
    st.md_step(dict(b.md), 0, ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
    rep = st.poll()
    assert rep.flags == 0 and rep.engine == (0 if engine == 0 else 2)        # the 7 A box cannot be resident: mixed dispatch
    scale = np.maximum(np.abs(o0["E"]), o0["Eabs"]) + 1e-300
    assert np.all(np.abs(st.numpy("energy") - o0["E"]) <= 1e-12 * scale + 1e-18)
    assert np.abs(st.numpy("force") - o0["F"]).max() <= 1e-10
    assert np.abs(st.numpy("virial") - o0["W"]).max() <= 1e-9 * max(1.0, np.abs(o0["W"]).max())
    for _ in range(3):                                                        # three calls: the lists (also the empty ones) carry over
        st.md_step(dict(b.md), 10)
    o = orc.md_run(b, "nve", b.md["dt"], 30)
    assert st.poll().flags == 0
    assert np.abs(st.numpy("pos") - o["pos"]).max() <= 1e-8 and np.abs(st.numpy("vel") - o["vel"]).max() <= 1e-10
    assert np.allclose(st.numpy("kinetic"), o["KE"], rtol=1e-10, atol=1e-18)
    st.close()


@pytest.mark.parametrize("engine", [0, 1])
def test_degenerate_systems_fire_and_edges(ts, orc, engine):
    """FIRE on the degenerate batch: the systems without forces converge with 0 steps and stay bit-unchanged, the others
    follow the oracle; the edge export counts no edge for the empty systems (both export entry points)."""
    import torch
    b = _degenerate_batch()
    fire = dict(dt_start=1.0, dt_max=10.0, f_inc=1.1, f_dec=0.5, alpha_start=0.1, f_alpha=0.99, f_max=1e-6, n_min=5, max_steps=10 ** 6)
    st = ts.SimState(b, engine=engine)
    st.fire_step(fire, 40)
    assert st.poll().flags == 0
    mask, status, steps = st.converged_mask()
    assert list(status[:2]) == [ts.TS_FIRE_CONVERGED] * 2 and list(steps[:2]) == [0, 0]        # F = 0 from the start
    assert status[4] == ts.TS_FIRE_CONVERGED and steps[4] == 0                                # the images' forces cancel
    off = b.sys_offset
    assert np.array_equal(st.numpy("pos")[: off[2]], b.pos[: off[2]])
    o = orc.fire_run(b, fire, 40)
    assert np.abs(st.numpy("pos") - o["pos"]).max() <= 1e-8
    assert list(steps) == list(o["state"]["nsteps"]) and list(status) == list(o["state"]["status"])
    st.close()
    st = ts.SimState(b, engine=0)
    st.md_step_external(ts.md_params(**b.md), ts.TS_PHASE_INIT)
    ei, es = st.export_edges()
    ei, es = ei.clone(), es.clone()
    cap = st.capacity()[2]
    oi = torch.full((2, cap), -7, dtype=torch.int64, device=st.device)
    os_ = torch.full((cap, 3), -7.0, dtype=st.tdtype, device=st.device)
    on = torch.full((1,), -7, dtype=torch.int64, device=st.device)
    st.export_edges_static(oi, os_, on)
    n = int(on.item())
    assert n == ei.shape[1] and torch.equal(oi[:, :n], ei) and torch.equal(os_[:n], es)
    i_sys = st.system_idx[ei[0]].cpu().numpy()
    counts = np.bincount(i_sys, minlength=5)
    want = [len(orc.pairs(b.pos[off[s]:off[s + 1]], b.cell[s], b.r_list)[0]) for s in range(5)]
    assert list(counts) == want and counts[0] == 0 and counts[1] == 0 and counts[4] > 0
    st.close()


def test_largest_resident_system_and_one_beyond(ts, orc):
    """2048 atoms is the most the resident engine holds (fp32: eight CTAs per system; in fp64 the slots of such a system
    do not fit shared memory and it goes to the general engine); 2916 atoms always go to the general engine.  fp32 replay
    parity (R29) after 12 NVE steps in two calls, and the plan says which engine took which."""
    a = wl.cfg1(n_systems=1, reps=8, dtype="f32", system_ids=[3])            # 8^3 x 4 = 2048 atoms
    c = wl.cfg1(n_systems=1, reps=9, dtype="f32", system_ids=[4])            # 9^3 x 4 = 2916 atoms
    b = wl.concat([a, c])
    st = ts.SimState(b, engine=1)
    st.md_step(dict(b.md), 5, ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
    st.md_step(dict(b.md), 7, ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL)
    rep = st.poll()
    assert rep.flags == 0 and rep.engine == 2
    bb = wl.with_(b, pos=st.numpy("pos").astype(np.float64), vel=st.numpy("vel").astype(np.float64))
    o = orc.energy_forces(bb)
    F = st.numpy("force").astype(np.float64)
    for s in range(2):
        a0, a1 = int(b.sys_offset[s]), int(b.sys_offset[s + 1])
        fmax = np.linalg.norm(o["F"][a0:a1], axis=1).max()
        bad = np.abs(F[a0:a1] - o["F"][a0:a1]).max(1) > 1e-4 * fmax
        assert bad.mean() < 0.01                                              # atoms with a pair within rounding of r_c (R29)
    scale = np.maximum(np.abs(o["E"]), o["Eabs"])
    assert np.all(np.abs(st.numpy("energy") - o["E"]) <= 1e-5 * scale)
    off, j, sh = st.get_resident_neighbors(0)                                 # the 2048-atom system is the resident one
    assert off.shape[0] == 2049 and off[-1] > 0
    with pytest.raises(ts.TsError):
        st.get_resident_neighbors(1)                                          # the 2916-atom system is not
    st.close()
    d64 = ts.SimState(wl.cfg1(n_systems=1, reps=8, system_ids=[3]), engine=1)   # the same 2048 atoms in fp64
    d64.md_step(dict(b.md), 2)
    assert d64.poll().engine == 0
    d64.close()
