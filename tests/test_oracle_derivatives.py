"""Pins for oracle O2: F = -dE/dx and W = -dE/dstrain by central differences, Newton's third law.
Inputs use the wide R28 window (w >= 10 delta, O8) so no pair crosses r_c inside the stencil."""
import copy

import numpy as np
import pytest

import workloads as wl


def _cases():
    return {
        "lj_fcc": wl.cfg1(n_systems=1, reps=3, w=2e-4),                    # box 15.78 < 2 rc: multi-image
        "morse_triclinic": wl.cfg3(system_ids=[1, 7], dtype="f64", w=2e-4, n_range=(32, 120)),
        "soft_binary": wl.cfg4([0], n_atoms=64, w=2e-4),
    }


@pytest.mark.parametrize("name", ["lj_fcc", "morse_triclinic", "soft_binary"])
def test_force_is_minus_energy_gradient(orc, name):
    b = _cases()[name]
    out = orc.energy_forces(b)
    F = out["F"]
    # Newton's third law: zero net force per system
    for s in range(b.n_systems):
        a0, a1 = b.sys_offset[s], b.sys_offset[s + 1]
        assert np.abs(F[a0:a1].sum(0)).max() < 1e-12 * max(1.0, np.abs(F[a0:a1]).max())
    rng = np.random.default_rng(0)
    delta = 1e-5
    for i in rng.choice(b.n_atoms, size=6, replace=False):
        s = int(b.system_idx[i])
        for k in range(3):
            e = []
            for sgn in (+1, -1):
                bb = copy.deepcopy(b)
                bb.pos[i, k] += sgn * delta
                e.append(orc.energy_forces(bb)["E"][s])
            fd = -(e[0] - e[1]) / (2 * delta)
            assert fd == pytest.approx(F[i, k], abs=1e-8 * max(1.0, abs(F[i, k])))


@pytest.mark.parametrize("name", ["lj_fcc", "morse_triclinic", "soft_binary"])
def test_virial_is_minus_strain_derivative(orc, name):
    b = _cases()[name]
    W = orc.energy_forces(b)["W"]
    assert np.allclose(W, np.swapaxes(W, 1, 2), atol=1e-12 * np.abs(W).max())       # symmetric
    delta = 1e-6
    for a in range(3):
        for c in range(a, 3):
            e = []
            for sgn in (+1, -1):
                eps = np.zeros((3, 3)); eps[a, c] += 0.5 * sgn * delta; eps[c, a] += 0.5 * sgn * delta
                bb = copy.deepcopy(b)
                M = np.eye(3) + eps
                bb.pos = b.pos @ M
                bb.cell = b.cell @ M
                e.append(orc.energy_forces(bb)["E"])
            fd = -(e[0] - e[1]) / (2 * delta)
            assert np.allclose(fd, W[:, a, c], rtol=2e-6, atol=2e-7 * np.abs(W).max())
