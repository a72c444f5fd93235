"""Pins for oracle O1 (pair set, image logic): brute force over a fixed image cube on tiny boxes,
supercell / re-basis / lattice-translation / permutation invariances (SURVEY.md 8(c) pins)."""
import copy

import numpy as np
import pytest

import workloads as wl


def _brute(pos, cell, R, nimg=4):
    """Triple loop over a generous FIXED image range, numpy only."""
    n = pos.shape[0]
    out = set()
    rng = range(-nimg, nimg + 1)
    for s0 in rng:
        for s1 in rng:
            for s2 in rng:
                sh = s0 * cell[0] + s1 * cell[1] + s2 * cell[2]
                d = pos[None, :, :] - pos[:, None, :] + sh       # [i, j] = x_j - x_i + S.h
                r2 = (d ** 2).sum(-1)
                ii, jj = np.nonzero(r2 < R * R)
                for i, j in zip(ii, jj):
                    if i == j and s0 == 0 and s1 == 0 and s2 == 0:
                        continue
                    out.add((int(i), int(j), s0, s1, s2))
    return out


@pytest.mark.parametrize("seed", range(6))
def test_pairs_brute_force_tiny_boxes(orc, seed):
    rng = np.random.default_rng(100 + seed)
    R = 2.5
    n = int(rng.integers(1, 33))
    heights = rng.uniform(0.6 * R, 2.6 * R, size=3)            # from 0.6 rc up: self- and multi-images
    cell = np.diag(heights)
    if seed % 2:                                               # sheared
        cell[1, 0] = rng.uniform(-0.4, 0.4) * heights[0]
        cell[2, 0] = rng.uniform(-0.4, 0.4) * heights[0]
        cell[2, 1] = rng.uniform(-0.4, 0.4) * heights[1]
    pos = rng.uniform(-0.5, 1.5, size=(n, 3)) @ cell           # stored positions may lie outside the cell
    i, j, S, r2 = orc.pairs(pos, cell, R)
    got = set(zip(i.tolist(), j.tolist(), S[:, 0].tolist(), S[:, 1].tolist(), S[:, 2].tolist()))
    assert len(got) == len(i)                                  # no duplicates
    assert got == _brute(pos, cell, R)
    # r2 reported equals the definition
    d = pos[j] - pos[i] + S @ cell
    assert np.allclose((d ** 2).sum(1), r2, rtol=1e-14)


def _lj_small():
    b = wl.cfg1(n_systems=1, reps=1, clean=False)              # 4 atoms, box 5.26 A << rc = 8.5 A
    return b


def test_supercell_invariance_box_smaller_than_cutoff(orc):
    b = _lj_small()
    o1 = orc.energy_forces(b)
    bb = copy.deepcopy(b)
    shift = b.cell[0, 0]
    bb.pos = np.concatenate([b.pos, b.pos + shift])
    n = b.n_atoms
    big = wl._finish("x", [(bb.pos, np.zeros((2 * n, 3)), np.tile(b.mass, 2), np.tile(b.type, 2), b.cell[0] * np.array([[2], [1], [1]]))],
                     b.potential, b.mass_conv, b.kB, 0.0, "f64", [0])
    o2 = orc.energy_forces(big)
    assert o2["E"][0] == pytest.approx(2 * o1["E"][0], rel=1e-13)
    assert np.allclose(o2["F"][:n], o1["F"], atol=1e-13) and np.allclose(o2["F"][n:], o1["F"], atol=1e-13)
    assert np.allclose(o2["W"][0], 2 * o1["W"][0], rtol=1e-12, atol=1e-15)


def test_rebasis_translation_permutation(orc):
    b = wl.cfg3(system_ids=[7], dtype="f64", clean=False, n_range=(32, 80))
    o = orc.energy_forces(b)
    # a1 -> a1 + a2 describes the same lattice
    bb = copy.deepcopy(b)
    bb.cell[0, 0] = b.cell[0, 0] + b.cell[0, 1]
    o2 = orc.energy_forces(bb)
    assert o2["E"][0] == pytest.approx(o["E"][0], rel=1e-13)
    assert np.allclose(o2["F"], o["F"], atol=1e-12) and np.allclose(o2["W"], o["W"], rtol=1e-11, atol=1e-13)
    # translating one atom by a lattice vector changes only S
    bb = copy.deepcopy(b)
    bb.pos[3] += 2 * b.cell[0, 1] - b.cell[0, 2]
    o3 = orc.energy_forces(bb)
    assert o3["E"][0] == pytest.approx(o["E"][0], rel=1e-13) and np.allclose(o3["F"], o["F"], atol=1e-11)
    R = b.potential.rc_max
    i0, j0, S0, _ = orc.pairs(b.pos, b.cell[0], R)
    i1, j1, S1, _ = orc.pairs(bb.pos, bb.cell[0], R)
    assert np.array_equal(i0, i1) and np.array_equal(j0, j1)
    dS = S1 - S0
    t = np.array([0, 2, -1])
    assert np.array_equal(dS[(i0 == 3) & (j0 != 3)], np.tile(t, (np.sum((i0 == 3) & (j0 != 3)), 1)))
    assert np.array_equal(dS[(j0 == 3) & (i0 != 3)], np.tile(-t, (np.sum((j0 == 3) & (i0 != 3)), 1)))
    assert not dS[(i0 != 3) & (j0 != 3)].any() and not dS[(i0 == 3) & (j0 == 3)].any()
    # permutation of atoms permutes forces
    perm = np.random.default_rng(1).permutation(b.n_atoms)
    bb = copy.deepcopy(b)
    bb.pos = b.pos[perm]
    o4 = orc.energy_forces(bb)
    assert np.allclose(o4["F"], o["F"][perm], atol=1e-12) and o4["E"][0] == pytest.approx(o["E"][0], rel=1e-13)


def test_generators_reject_near_cutoff_pairs(orc):
    """R28: no pair within w of r_c or r_c + skin, verified with the ORACLE's own search."""
    for b, w in ((wl.cfg1(n_systems=2), 1e-6), (wl.cfg2(n_systems=1, dtype="f32"), 1e-4), (wl.cfg4([0, 1]), 1e-6)):
        radii = sorted(set(np.unique(b.potential.rc).tolist() + [b.r_list]))
        for s in range(b.n_systems):
            a0, a1 = b.sys_offset[s], b.sys_offset[s + 1]
            _, _, _, r2 = orc.pairs(b.pos[a0:a1], b.cell[s], radii[-1] + 2 * w)
            r = np.sqrt(r2)
            for R in radii:
                assert np.abs(r - R).min() >= w * (1 - 1e-9)
