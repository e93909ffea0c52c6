"""Pins of the oracle's velocity-Verlet map (O8): SURVEY.md §8(c) P8-P11."""
import math

import numpy as np

import oracle
from paper_2412_18271_b200 import workloads as W


def test_p10_harmonic_oscillator_period_and_dt2():
    """Textbook special case: two atoms (H, C) on a spring E = k/2 (r-r0)^2.
    omega^2 = k*ACC/mu.  After exactly one period the bond length returns to its
    start with an error ~ dt^2, and the energy error scales as dt^2."""
    k, r0, amp = 30.0, 1.1, 0.05
    m = oracle.MASSES_AMU
    mu = m[0] * m[1] / (m[0] + m[1])
    period = 2 * math.pi * math.sqrt(mu / (k * oracle.ACC))
    pos = np.array([[0.0, 0, 0], [r0 + amp, 0, 0]])
    vel = np.zeros((2, 3))
    errs, derr = [], []
    for n in (400, 800):
        dt = period / n
        out = oracle.step(pos, vel, [0, 1], [0, 2], None, dt, n, harmonic=(k, r0))
        r = np.linalg.norm(out["pos"][1] - out["pos"][0])
        errs.append(abs(r - (r0 + amp)))
        H = out["pe"][:, 0] + out["ke"][:, 0]
        derr.append(np.abs(H - H[0]).max())
        # centre of mass does not move, momentum conserved
        assert np.abs((m[[0, 1], None] * out["vel"]).sum(0)).max() < 1e-12
    assert errs[0] < 1e-4 * amp * 50 and errs[1] < errs[0]
    assert 3.5 < derr[0] / derr[1] < 4.5
    # measured period from the first return of (r - r0) to a maximum
    n = 2000
    dt = 1.25 * period / n
    out = [oracle.step(pos, vel, [0, 1], [0, 2], None, dt, s, harmonic=(k, r0)) for s in (0,)]
    traj = []
    p, v = pos, vel
    for _ in range(n):
        o = oracle.step(p, v, [0, 1], [0, 2], None, dt, 1, harmonic=(k, r0))
        p, v = o["pos"], o["vel"]
        traj.append(np.linalg.norm(p[1] - p[0]) - r0)
    traj = np.array(traj)
    i_max = n // 2 + int(np.argmax(traj[n // 2:]))
    assert abs((i_max + 1) * dt - period) < 2 * dt


def test_p8_nve_second_order_and_bounded_drift(weights):
    """max_t |H(t)-H(0)| over 50 fs at dt = 0.5 vs 0.25 fs has ratio ~4 (the
    integrator is second order); no secular drift over 200 steps (configs[0])."""
    c = W.config0()
    a = oracle.step(c.pos, c.vel, c.species, c.sys_offsets, weights, 0.5, 100)
    b = oracle.step(c.pos, c.vel, c.species, c.sys_offsets, weights, 0.25, 200)
    Ha = (a["pe"] + a["ke"])[:, 0]
    Hb = (b["pe"] + b["ke"])[:, 0]
    da, db = np.abs(Ha - Ha[0]).max(), np.abs(Hb - Hb[0]).max()
    assert 3.0 < da / db < 5.0
    long = oracle.step(c.pos, c.vel, c.species, c.sys_offsets, weights, 0.5, 200)
    H = (long["pe"] + long["ke"])[:, 0]
    osc = np.abs(H[:100] - H[0]).max()
    assert abs(H[100:].mean() - H[:100].mean()) < 2 * osc
    # P11 context: sigma_H/|H| of order 1e-4 or better over 100 steps
    assert H[:101].std() / max(abs(H[:101].mean()), 1.0) < 1e-3


def test_p9_time_reversibility(weights):
    c = W.config0()
    fwd = oracle.step(c.pos, c.vel, c.species, c.sys_offsets, weights, 0.5, 50)
    back = oracle.step(fwd["pos"], -fwd["vel"], c.species, c.sys_offsets, weights, 0.5, 50)
    assert np.abs(back["pos"] - c.pos.astype(np.float64)).max() < 1e-9
    assert np.abs(back["vel"] + c.vel.astype(np.float64)).max() < 1e-9


def test_step_forces_and_energy_bookkeeping(weights):
    """F returned by step() is the force at the returned positions; pe[0] is the
    energy of the start; KE uses the element masses (S12) and ACC."""
    c = W.config1(n_replicas=3)
    out = oracle.step(c.pos, c.vel, c.species, c.sys_offsets, weights, 0.5, 3)
    ef = oracle.energy_forces(out["pos"], c.species, c.sys_offsets, weights)
    np.testing.assert_allclose(out["F"], ef["F"], rtol=0, atol=1e-13)
    np.testing.assert_allclose(out["pe"][-1], ef["E"], rtol=0, atol=1e-12)
    e0 = oracle.energy_forces(c.pos, c.species, c.sys_offsets, weights)
    np.testing.assert_allclose(out["pe"][0], e0["E"], rtol=0, atol=1e-12)
    v = c.vel.astype(np.float64)
    ke = 0.5 * oracle.MASSES_AMU[c.species] * (v * v).sum(1) / oracle.ACC
    want = [ke[c.sys_offsets[s]:c.sys_offsets[s + 1]].sum() for s in range(3)]
    np.testing.assert_allclose(out["ke"][0], want, rtol=1e-13)
    # replicas are independent: stepping replica 1 alone gives the same trajectory
    sl = slice(c.sys_offsets[1], c.sys_offsets[2])
    solo = oracle.step(c.pos[sl], c.vel[sl], c.species[sl], [0, 22], weights, 0.5, 3)
    np.testing.assert_allclose(solo["pos"], out["pos"][sl], rtol=0, atol=1e-13)
