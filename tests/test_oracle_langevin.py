"""Pins of the oracle's Langevin integrator O9 (reading S27/S28): the counter-based generator against
its published known-answer vectors, the normals' moments, the zero-friction limit (velocity-Verlet),
and thermalisation of free particles by the O step."""
import numpy as np
import pytest

import oracle
from paper_2412_18271_b200 import workloads as W

KB = 8.617333262e-5
ACC = 9.648533216e-3
MASS = np.array([1.008, 12.011, 14.007, 15.999])


def test_philox_known_answers():
    """P13: Philox4x32-10 known-answer vectors of the Random123 distribution (Salmon et al., SC'11)."""
    kat = [
        ([0, 0, 0, 0], [0, 0], [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]),
        ([0xffffffff] * 4, [0xffffffff] * 2, [0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd]),
        ([0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344], [0xa4093822, 0x299f31d0],
         [0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1]),
    ]
    for ctr, key, want in kat:
        assert [int(x) for x in oracle.philox4x32_10(ctr, key)] == want


def test_normals_moments_and_independence():
    """P14: the Box-Muller normals have mean 0, variance 1, kurtosis 3, no correlation between
    components, atoms or steps; a different seed gives a different stream."""
    xi = np.array([oracle.langevin_normals(a, s, 77) for a in range(200) for s in range(1, 101)])
    n = xi.shape[0]
    assert np.abs(xi.mean(0)).max() < 4.0 / np.sqrt(n)
    assert np.abs(xi.var(0) - 1.0).max() < 4.0 * np.sqrt(2.0 / n)
    assert np.abs((xi ** 4).mean(0) - 3.0).max() < 0.15
    c = np.corrcoef(xi.T)
    assert np.abs(c - np.eye(3)).max() < 4.0 / np.sqrt(n)
    lag = (xi[1:, 0] * xi[:-1, 0]).mean()
    assert abs(lag) < 4.0 / np.sqrt(n)
    assert not np.allclose(oracle.langevin_normals(3, 5, 77), oracle.langevin_normals(3, 5, 78))
    assert np.array_equal(oracle.langevin_normals(3, 5, 77), oracle.langevin_normals(3, 5, 77))


def test_zero_friction_is_velocity_verlet():
    """P15: gamma = 0 gives c1 = 1, c2 = 0: BAOAB is O8 (two half drifts = one drift up to rounding)."""
    wl, w = W.config0(), W.make_weights()
    a = oracle.step(wl.pos, wl.vel, wl.species, wl.sys_offsets, w, 0.5, 10)
    b = oracle.step_langevin(wl.pos, wl.vel, wl.species, wl.sys_offsets, w, 0.5, 10, 0.0, 300.0, 1)
    assert np.abs(a["pos"] - b["pos"]).max() < 1e-12
    assert np.abs(a["vel"] - b["vel"]).max() < 1e-13
    assert np.abs(a["F"] - b["F"]).max() < 1e-9


def test_free_particles_thermalise():
    """P16: without forces the O step is an exact Ornstein-Uhlenbeck update: after many relaxation
    times <m v^2 / ACC> = kB T per component for every element, whatever the start."""
    n = 4000
    species = (np.arange(n) % 4).astype(np.int32)
    pos = np.zeros((n, 3)); vel = np.full((n, 3), 0.05)
    off = np.array([0, n], dtype=np.int32)
    T, gamma, dt = 450.0, 0.05, 1.0                      # 20 fs relaxation time, 400 fs run
    out = oracle.step_langevin(pos, vel, species, off, None, dt, 400, gamma, T, 5, free=True)
    for z in range(4):
        v = out["vel"][species == z]
        kt = MASS[z] * (v ** 2).mean() / ACC
        assert abs(kt / (KB * T) - 1.0) < 4.0 * np.sqrt(2.0 / v.size)
    # one O step from rest: variance (1 - c1^2) kB T ACC / m exactly
    out1 = oracle.step_langevin(pos, 0 * vel, species, off, None, dt, 1, gamma, T, 9, free=True)
    c1 = np.exp(-gamma * dt)
    v = out1["vel"][species == 0]
    assert abs((v ** 2).mean() / ((1 - c1 ** 2) * KB * T * ACC / MASS[0]) - 1.0) < 4.0 * np.sqrt(2.0 / v.size)
    # and the drift uses the half-updated velocities: x = dt/2 (v_before + v_after) with v_before = 0
    assert np.allclose(out1["pos"], 0.5 * dt * out1["vel"], atol=1e-15)
