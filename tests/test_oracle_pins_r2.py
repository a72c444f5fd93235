"""Round-2 pins for the parts of the oracle that had none:

  * O6 step (4), reading R21: the FIRE velocity mixing v <- (1 - a) v + a |v|/|F| F with the alpha
    from BEFORE its update, on a non-collinear system where v has a component perpendicular to F
    (on a 1-D dimer v || F whenever P > 0 and the mix is the identity, so the dimer pins of
    test_oracle_fire.py cannot see it); the P == 0 boundary (strict P > 0 of O6 step 4/5).
  * `Eabs` = sum 1/2 |V| returned by energy_forces (R31): every GPU energy tolerance is scaled by
    it, so it is pinned against a dimer and against an independent numpy lattice sum with V of
    both signs.
  * BAOAB in a (nearly) harmonic well: <(r - <r>)^2> of a Morse dimer against the Boltzmann
    average evaluated by quadrature (harmonic limit kB T / k, k = 2 D alpha^2) -- SURVEY 8(c) BAOAB pin.
  * cfg3-shaped NVE drift bound (Morse truncated with a force jump at r_c): <= 1e-3 eV/atom over 500 steps.

Expected values are computed here in numpy from the textbook formulas (Bitzek et al., PRL 97, 170201
(2006) eq. for the velocity mixing; Boltzmann statistics), never by re-calling the routine under test.
"""
import numpy as np
import pytest

import workloads as wl

D, AL, R0, RCM, MCU = 0.3429, 1.3588, 2.866, 6.0, 63.546


def _morse(r):
    e = np.exp(-AL * (r - R0))
    return D * ((1 - e) ** 2 - 1), 2 * D * AL * (1 - e) * e


def _batch(pos, vel, mass, cell=40.0, pot=None, mass_conv=wl.MASS_CONV_METAL, kB=wl.KB_METAL):
    pos = np.asarray(pos, float)
    pot = pot or wl._single_type("morse", D, AL, R0, RCM)
    n = len(pos)
    return wl._finish("pin", [(pos, np.asarray(vel, float), np.full(n, float(mass)), np.zeros(n, np.int32), np.eye(3) * cell)],
                      pot, mass_conv, kB, 0.0, "f64", [0])


def _numpy_forces(pos):
    """Open-boundary Morse forces of a small cluster (all distances < r_c, box >> cluster): plain numpy."""
    n = len(pos)
    F = np.zeros((n, 3))
    for i in range(n):
        for j in range(n):
            if i != j:
                rv = pos[j] - pos[i]
                r = np.linalg.norm(rv)
                assert r < RCM
                F[i] += _morse(r)[1] * rv / r
    return F


FP = dict(dt_start=1.0, dt_max=10.0, f_inc=1.1, f_dec=0.5, alpha_start=0.1, f_alpha=0.99, f_max=1e-8, n_min=5, max_steps=5000)


def _running_state(dt, alpha, npos, nsteps=17):
    return {"dt": np.array([dt]), "alpha": np.array([alpha]), "npos": np.array([npos], np.int32),
            "nsteps": np.array([nsteps], np.int32), "status": np.array([1], np.int32), "E": np.zeros(1), "fmax": np.zeros(1)}


def test_fire_mixing_noncollinear_uses_alpha_before_its_update(orc):
    """One FIRE step of a 4-atom non-planar cluster entered RUNNING with N_pos = N_min (so this very
    step also updates alpha and dt).  Bitzek's rule with the pre-update alpha, evaluated in numpy."""
    pos = np.array([[10.0, 10.0, 10.0], [12.9, 10.2, 9.9], [11.3, 12.6, 10.4], [11.5, 11.0, 12.5]])
    rng = np.random.Generator(np.random.PCG64(7))
    vel = rng.normal(0.0, 2e-3, size=(4, 3))
    dt, a_old, npos = 1.7, 0.0731, FP["n_min"]
    b = _batch(pos, vel, MCU)
    # the oracle's forces on this cluster are the plain numpy double loop (separately pinned potentials)
    F0 = _numpy_forces(pos)
    assert np.allclose(orc.energy_forces(b)["F"], F0, rtol=0, atol=1e-14)
    im = 1.0 / (MCU * wl.MASS_CONV_METAL)
    v1 = vel + 0.5 * dt * F0 * im
    x1 = pos + dt * v1
    F1 = _numpy_forces(x1)
    v2 = v1 + 0.5 * dt * F1 * im
    P = np.sum(F1 * v2)
    assert P > 0.0                                            # downhill: the mixing branch
    fn, vn = np.sqrt(np.sum(F1 * F1)), np.sqrt(np.sum(v2 * v2))
    want = (1.0 - a_old) * v2 + a_old * (vn / fn) * F1        # alpha BEFORE the update (R21)
    wrong_after = (1.0 - a_old * FP["f_alpha"]) * v2 + a_old * FP["f_alpha"] * (vn / fn) * F1
    r = orc.fire_run(b, FP, 1, state=_running_state(dt, a_old, npos))
    st = r["state"]
    assert st["status"][0] == orc.FIRE_RUNNING and st["nsteps"][0] == 18
    assert np.allclose(r["pos"], x1, rtol=0, atol=1e-13)
    scale = np.abs(want).max()
    assert np.abs(r["vel"] - want).max() <= 1e-12 * scale
    assert np.abs(r["vel"] - wrong_after).max() > 1e-5 * scale          # the excluded reading is resolvable
    # the component of the 3N-dim velocity perpendicular to the 3N-dim force shrinks by exactly (1 - alpha_old)
    fh = (F1 / fn).ravel()
    perp_in = v2.ravel() - np.dot(v2.ravel(), fh) * fh
    perp_out = r["vel"].ravel() - np.dot(r["vel"].ravel(), fh) * fh
    assert np.linalg.norm(perp_in) > 0.2 * vn                 # the case really has a perpendicular part
    assert np.allclose(perp_out, (1.0 - a_old) * perp_in, rtol=0, atol=1e-13 * vn)
    # |v| is preserved to first order only along F: the parallel part becomes (1 - a) v_par + a |v|
    par_out = np.dot(r["vel"].ravel(), fh)
    assert par_out == pytest.approx((1.0 - a_old) * np.dot(v2.ravel(), fh) + a_old * vn, rel=1e-12)
    # N_pos = N_min + 1 > N_min: dt grows, alpha shrinks -- after the mixing used the old alpha
    assert st["npos"][0] == npos + 1
    assert st["dt"][0] == min(dt * FP["f_inc"], FP["dt_max"]) and st["alpha"][0] == a_old * FP["f_alpha"]


def test_fire_mixing_below_n_min_keeps_dt_and_alpha(orc):
    pos = np.array([[10.0, 10.0, 10.0], [12.9, 10.2, 9.9], [11.3, 12.6, 10.4]])
    b = _batch(pos, np.zeros((3, 3)), MCU)
    r = orc.fire_run(b, FP, 1, state=_running_state(1.3, 0.1, 2))
    st = r["state"]
    assert st["npos"][0] == 3 and st["dt"][0] == 1.3 and st["alpha"][0] == 0.1     # from rest P > 0 after one step


def test_fire_p_exactly_zero_takes_the_uphill_branch(orc):
    """O6 steps 4/5: the mixing needs P > 0 strictly.  A dimer along x with both velocities along y
    and dt = 0 (the step is the identity, so v stays exactly perpendicular to F): P == 0 exactly while
    max |F| > f_max.  Expected: v <- 0, N_pos <- 0, alpha <- alpha_start, dt <- dt f_dec."""
    pos = np.array([[5.0, 5.0, 5.0], [8.3, 5.0, 5.0]])
    vel = np.array([[0.0, 1e-3, 0.0], [0.0, 1e-3, 0.0]])
    b = _batch(pos, vel, MCU, cell=30.0)
    F = orc.energy_forces(b)["F"]
    assert np.all(F[:, 1:] == 0.0) and abs(F[0, 0]) > 1e-3    # F exactly along x
    r = orc.fire_run(b, FP, 1, state=_running_state(0.0, 0.0731, 4))
    st = r["state"]
    assert st["status"][0] == orc.FIRE_RUNNING and st["nsteps"][0] == 18
    assert not r["vel"].any()                                 # P <= 0: stop
    assert st["npos"][0] == 0 and st["alpha"][0] == FP["alpha_start"] and st["dt"][0] == 0.0
    # and the same geometry with a slightly downhill velocity mixes instead
    vel2 = vel + np.array([[1e-6, 0, 0], [-1e-6, 0, 0]]) * np.sign(F[0, 0])
    r2 = orc.fire_run(_batch(pos, vel2, MCU, cell=30.0), FP, 1, state=_running_state(0.0, 0.0731, 4))
    assert r2["state"]["npos"][0] == 5 and r2["vel"].any()


# ------------------------------------------------------------------------------- Eabs (R31)
def test_eabs_dimer(orc):
    for r in (2.4, 2.866, 4.7):                               # V_shifted > 0, < 0, < 0
        b = _batch([[5, 5, 5], [5 + r, 5, 5]], np.zeros((2, 3)), MCU, cell=30.0)
        o = orc.energy_forces(b)
        V = _morse(r)[0] - _morse(RCM)[0]
        assert o["E"][0] == pytest.approx(V, rel=1e-13)
        assert o["Eabs"][0] == pytest.approx(abs(V), rel=1e-13)      # two directed pairs x 1/2 |V|


def test_eabs_fcc_lattice_sum_with_both_signs(orc):
    """Compressed perfect FCC (a = 4.6 A: the first shell sits inside sigma, V > 0; the outer shells
    have V < 0), LJ cfg1 parameters.  E/atom and Eabs/atom from an independent numpy enumeration of
    the lattice vectors within r_c."""
    eps, sig, rc, a = 0.0104, 3.40, 8.5, 4.6
    lj = lambda r: 4 * eps * ((sig / r) ** 12 - (sig / r) ** 6)
    pot = wl._single_type("lj", eps, sig, 0.0, rc)
    base, cell = wl.lattice(wl._FCC, a, (2, 2, 2))            # 32 atoms, box 9.2 A: multiple images
    b = wl._finish("fcc", [(base, np.zeros_like(base), np.ones(32), np.zeros(32, np.int32), cell)], pot, 1.0, 1.0, 0.0, "f64", [0])
    o = orc.energy_forces(b)
    g = np.arange(-4, 5)
    R = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 1, 3) + wl._FCC[None, :, :]
    d = np.linalg.norm(R.reshape(-1, 3) * a, axis=1)
    d = d[(d > 1e-9) & (d < rc)]
    V = lj(d) - lj(rc)
    assert (V > 0).any() and (V < 0).any()
    assert o["E"][0] / 32 == pytest.approx(0.5 * V.sum(), rel=1e-12)
    assert o["Eabs"][0] / 32 == pytest.approx(0.5 * np.abs(V).sum(), rel=1e-12)
    assert o["Eabs"][0] > 1.05 * abs(o["E"][0])               # the two differ: an |E| in place of sum |V| would fail


def test_eabs_of_cfg_shapes_is_at_least_abs_e(orc):
    for b in (wl.cfg1(n_systems=1, reps=2, clean=False), wl.cfg4(range(2), n_atoms=32, clean=False)):
        o = orc.energy_forces(b)
        assert np.all(o["Eabs"] >= np.abs(o["E"]) * (1 - 1e-14))


# ------------------------------------------------------------------------------- BAOAB in a well
def test_baoab_morse_dimer_bond_fluctuation(orc):
    """Langevin BAOAB samples the Boltzmann distribution: for a Morse dimer the bond length r has
    density ~ r^2 exp(-V(r)/kT).  Var(r) over many dimers and times against the quadrature value
    (harmonic limit kT / (2 D alpha^2))."""
    T, dt, gamma = 40.0, 2.0, 0.02
    kT = wl.KB_METAL * T
    rr = np.linspace(2.0, 4.5, 200001)
    w = rr ** 2 * np.exp(-(_morse(rr)[0] + D) / kT)
    m1 = np.trapezoid(w * rr, rr) / np.trapezoid(w, rr)
    var_exact = np.trapezoid(w * (rr - m1) ** 2, rr) / np.trapezoid(w, rr)
    k = 2 * D * AL ** 2
    assert var_exact == pytest.approx(kT / k, rel=0.05)       # nearly harmonic at 40 K
    n_dim = 384
    rng = np.random.Generator(np.random.PCG64(11))
    parts = []
    for _ in range(n_dim):
        u = rng.normal(size=3); u /= np.linalg.norm(u)
        p = np.array([15.0, 15.0, 15.0]) + np.outer([-0.5, 0.5], u * R0)
        parts.append((p, np.zeros((2, 3)), np.full(2, MCU), np.zeros(2, np.int32), np.eye(3) * 30.0))
    b = wl._finish("dimers", parts, wl._single_type("morse", D, AL, R0, RCM), wl.MASS_CONV_METAL, wl.KB_METAL, 0.0, "f64",
                   list(range(n_dim)))
    samples, cur, step = [], b, None
    r = orc.md_run(cur, "baoab", dt, 1500, temperature=T, friction=gamma, seed=5, sys_uid=b.sys_uid)     # equilibrate
    for _ in range(12):                                       # 12 samples 400 fs apart (>> 1 / gamma = 50 fs)
        cur = wl.with_(cur, pos=r["pos"], vel=r["vel"])
        r = orc.md_run(cur, "baoab", dt, 200, temperature=T, friction=gamma, seed=5, sys_uid=b.sys_uid, step=r["step"])
        p = r["pos"].reshape(n_dim, 2, 3)
        samples.append(np.linalg.norm(p[:, 1] - p[:, 0], axis=1))
    s = np.concatenate(samples)
    n_eff = s.size
    assert s.mean() == pytest.approx(m1, abs=5 * np.sqrt(var_exact / n_eff))
    assert s.var() == pytest.approx(var_exact, rel=5 * np.sqrt(2.0 / n_eff) + 0.01)    # + O(dt^2) discretisation


# ------------------------------------------------------------------------------- cfg3 drift (reported bound)
def test_cfg3_nve_drift_bound_500_steps(orc):
    b = wl.cfg3(n_systems=3, dtype="f64", n_range=(32, 120))
    r = orc.md_run(b, "nve", 1.0, 500, history=True)
    etot = r["epot_hist"] + r["ke_hist"]
    n = np.diff(b.sys_offset)
    drift = np.abs(etot - etot[0]).max(0) / n
    assert np.all(drift <= 1e-3), drift                       # SURVEY 8(c) NVE pin, eV/atom (force jump 0.013 eV/A at r_c)
