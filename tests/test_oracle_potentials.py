"""Pins for oracle O2 (potentials, energy/force/virial) against closed forms.
SURVEY.md section 8(c) "What pins each part": dimer closed forms, FCC shell sums."""
import numpy as np
import pytest

import workloads as wl

EPS, SIG, RC = 0.0104, 3.40, 8.5


def lj(r, eps=EPS, sig=SIG):
    return 4 * eps * ((sig / r) ** 12 - (sig / r) ** 6)


def dlj(r, eps=EPS, sig=SIG):
    return -24 * eps * (2 * (sig / r) ** 12 - (sig / r) ** 6) / r


def test_lj_dimer_closed_forms(orc):
    rmin = 2 ** (1 / 6) * SIG
    assert rmin == pytest.approx(3.816370964, abs=1e-9)
    Vc = lj(RC)
    assert Vc == pytest.approx(-1.6969566781e-4, rel=1e-9)
    V, dV = orc.pair_potential("lj", EPS, SIG, 0.0, RC, True, rmin)
    assert V == pytest.approx(-EPS - Vc, rel=1e-13)
    assert V == pytest.approx(-0.0102303043322, rel=1e-10)
    assert abs(dV) < 1e-15
    V, dV = orc.pair_potential("lj", EPS, SIG, 0.0, RC, True, SIG)
    assert dV == pytest.approx(-24 * EPS / SIG, rel=1e-13)
    assert V == pytest.approx(-Vc, rel=1e-12)
    assert orc.pair_potential("lj", EPS, SIG, 0.0, RC, True, RC) == (0.0, 0.0)      # strict cutoff
    V, _ = orc.pair_potential("lj", EPS, SIG, 0.0, RC, False, 5.0)
    assert V == pytest.approx(lj(5.0), rel=1e-14)


def test_morse_dimer_closed_forms(orc):
    D, a, r0, rc = 0.3429, 1.3588, 2.866, 6.0
    e = np.exp(-a * (rc - r0))
    Vc = D * ((1 - e) ** 2 - 1)
    assert Vc == pytest.approx(-9.631219157e-3, rel=1e-9)
    V, dV = orc.pair_potential("morse", D, a, r0, rc, True, r0)
    assert V == pytest.approx(-D - Vc, rel=1e-13) and abs(dV) < 1e-15
    # V'(6.0) evaluated just inside the cutoff
    _, dV = orc.pair_potential("morse", D, a, r0, rc, True, rc * (1 - 1e-15))
    assert dV == pytest.approx(1.299369220e-2, rel=1e-8)
    V, _ = orc.pair_potential("morse", D, a, r0, rc, False, 1e9 if False else 5.9)
    assert V == pytest.approx(D * ((1 - np.exp(-a * (5.9 - r0))) ** 2 - 1), rel=1e-13)


def test_soft_sphere_closed_forms(orc):
    eps, sig = 1.7, 1.3
    V, dV = orc.pair_potential("soft_sphere", eps, sig, 2.0, sig, True, sig / 2)
    assert V == pytest.approx(eps / 8, rel=1e-14)
    assert abs(dV) == pytest.approx(eps / (2 * sig), rel=1e-14) and dV < 0
    assert orc.pair_potential("soft_sphere", eps, sig, 2.0, sig, True, sig) == (0.0, 0.0)
    V, dV = orc.pair_potential("soft_sphere", eps, sig, 2.5, sig, True, 0.4 * sig)       # non-integer exponent
    assert V == pytest.approx(eps / 2.5 * 0.6 ** 2.5, rel=1e-13)
    assert dV == pytest.approx(-eps / sig * 0.6 ** 1.5, rel=1e-13)


def _dimer_batch(pos, cell, pot):
    pos = np.asarray(pos, float)
    return wl._finish("dimer", [(pos, np.zeros_like(pos), np.ones(len(pos)), np.zeros(len(pos), np.int32), np.asarray(cell, float))],
                      pot, 1.0, 1.0, 0.0, "f64", [0])


@pytest.mark.parametrize("r", [3.3, 3.816370964, 5.1, 8.4999])
def test_dimer_in_periodic_boxes(orc, r):
    pot = wl._single_type("lj", EPS, SIG, 0.0, RC)
    L = 40.0
    cubic = np.eye(3) * L
    shear = np.array([[L, 0, 0], [0.3 * L, L, 0], [0.1 * L, -0.2 * L, L]])
    u = np.array([1.0, 2.0, -0.5]); u /= np.linalg.norm(u)
    cases = [
        ([[1, 1, 1], np.array([1, 1, 1]) + r * u], cubic),
        ([[L - 0.4, 5, 5], [r - 0.4, 5, 5]], cubic),                      # across the periodic boundary
        ([[0.2, 39.9, 0.1], np.array([0.2, 39.9, 0.1]) - r * u], cubic),  # stored positions outside the box (R5)
        ([[3, 3, 3], np.array([3, 3, 3]) + r * shear[1] / np.linalg.norm(shear[1])], shear),  # along a sheared axis
        ([shear[1] * 0.99 + 1.0, shear[1] * 0.99 + 1.0 + r * shear[1] / np.linalg.norm(shear[1]) - shear[1]], shear),
    ]
    for pos, cell in cases:
        out = orc.energy_forces(_dimer_batch(pos, cell, pot))
        assert out["E"][0] == pytest.approx(lj(r) - lj(RC), rel=1e-11, abs=1e-16)
        f = np.linalg.norm(out["F"], axis=1)
        assert f[0] == pytest.approx(abs(dlj(r)), rel=1e-10, abs=1e-15)
        assert np.allclose(out["F"][0], -out["F"][1], rtol=0, atol=1e-18)
        # attractive beyond r_min: force on atom 0 points to its partner's nearest image
        assert np.allclose(np.trace(out["W"][0]), -dlj(r) * r, rtol=1e-10)


def _fcc_shells(a, rc):
    """Shell distances and multiplicities of FCC by explicit lattice enumeration (numpy only)."""
    n = int(np.ceil(rc / a)) + 1
    g = np.stack(np.meshgrid(*[np.arange(-n, n + 1)] * 3, indexing="ij"), -1).reshape(-1, 3)
    pts = (g[:, None, :] + wl._FCC[None]).reshape(-1, 3) * a
    d = np.linalg.norm(pts, axis=1)
    d = d[(d > 1e-9) & (d < rc)]
    return d


def test_fcc_lattice_sum_cfg1(orc):
    a = 5.26
    base, cell = wl.lattice(wl._FCC, a, (4, 4, 4))
    b = wl.cfg1(n_systems=1, clean=False)
    b.pos = base
    out = orc.energy_forces(b)
    # textbook FCC shells: 12, 6, 24, 12, 24 at d = a sqrt(n/2), n = 1..5 inside 8.5 A
    c = np.array([12, 6, 24, 12, 24]); d = a * np.sqrt(np.arange(1, 6) / 2)
    assert d[-1] < RC < a * np.sqrt(3.0)
    e_atom = 0.5 * np.sum(c * (lj(d) - lj(RC)))
    assert e_atom == pytest.approx(-0.07760965343, rel=1e-9)                 # SURVEY 8(c) value
    assert out["E"][0] / 256 == pytest.approx(e_atom, rel=1e-13)
    assert 0.5 * np.sum(c * lj(d)) == pytest.approx(-0.08422778448, rel=1e-9)
    assert np.abs(out["F"]).max() < 1e-14
    W = out["W"][0]
    trw = -0.5 * np.sum(c * dlj(d) * d)
    assert trw == pytest.approx(0.01011606978, rel=1e-9)
    assert np.trace(W) / 256 == pytest.approx(trw, rel=1e-12)
    assert np.allclose(W, np.eye(3) * np.trace(W) / 3, atol=1e-13)            # isotropic
    for R, nn in ((8.5, 78), (9.5, 86)):
        i, j, S, r2 = orc.pairs(base, cell, R)
        assert np.all(np.bincount(i, minlength=256) == nn)
    assert _fcc_shells(a, 8.5).size == 78 and _fcc_shells(a, 9.5).size == 86


def test_fcc_textbook_lattice_sums(orc):
    """A12 = 12.13188, A6 = 14.45392 (Kittel): E/atom = 2 eps [A12 (s/d)^12 - A6 (s/d)^6]."""
    sig, eps = 1.0, 1.0
    d_nn = 1.09017 * sig
    a = d_nn * np.sqrt(2.0)
    rc = 3.99 * a                                      # box 8a > 2 rc not needed: images handled
    base, cell = wl.lattice(wl._FCC, a, (2, 2, 2))     # box SMALLER than rc: multi-image path
    pot = wl._single_type("lj", eps, sig, 0.0, rc, shift=False)
    b = wl._finish("fcc", [(base, np.zeros_like(base), np.ones(32), np.zeros(32, np.int32), cell)], pot, 1.0, 1.0, 0.0, "f64", [0])
    out = orc.energy_forces(b)
    d = _fcc_shells(a, rc) / d_nn
    A12, A6 = np.sum(d ** -12.0), np.sum(d ** -6.0)
    assert A12 == pytest.approx(12.13188, abs=2e-4)
    tail6 = 4 * np.pi * np.sqrt(2.0) / 3.0 * (rc / d_nn) ** -3.0          # integral of the continuum beyond rc
    assert A6 + tail6 == pytest.approx(14.45392, abs=2e-2)
    e_atom = 2 * eps * (A12 * (sig / d_nn) ** 12 - A6 * (sig / d_nn) ** 6)
    assert out["E"][0] / 32 == pytest.approx(e_atom, rel=1e-12)
    assert -eps * 14.45392 ** 2 / (2 * 12.13188) == pytest.approx(-8.6102, abs=1e-4)
    assert np.abs(out["F"]).max() < 1e-12


def test_type_table_and_per_pair_cutoff(orc):
    """Binary soft-sphere (R13): sigma_ij in {1.0, 1.2, 1.4}, cutoff = pair sigma."""
    pot = wl.soft_sphere_binary()
    L = 10.0
    for (ti, tj, sij) in ((0, 0, 1.0), (0, 1, 1.2), (1, 1, 1.4)):
        for r in (0.5 * sij, 0.95 * sij, 1.01 * sij):
            pos = np.array([[1, 1, 1], [1 + r, 1, 1]], float)
            b = wl._finish("d", [(pos, np.zeros_like(pos), np.ones(2), np.array([ti, tj], np.int32), np.eye(3) * L)], pot, 1.0, 1.0, 0.0, "f64", [0])
            out = orc.energy_forces(b)
            exp = 0.5 * (1 - r / sij) ** 2 if r < sij else 0.0
            assert out["E"][0] == pytest.approx(exp, rel=1e-13, abs=1e-18)
            fx = (1 - r / sij) / sij if r < sij else 0.0
            assert out["F"][0, 0] == pytest.approx(-fx, rel=1e-13, abs=1e-18)     # repulsive: pushed away from j
