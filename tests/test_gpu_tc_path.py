"""GPU parity of the tensor-core K3 (tcgen05 kind::tf32, 3-term split)
against the fp64 oracle, at the SAME bars as the FP32 path (north_star allows 5e-3 eV/A for a
reduced-precision MLP; the split meets the FP32 bars, so those are the ones asserted), and the
evidence that plain TF32 (one term) does not.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle                                                    # noqa: E402
from paper_2412_18271_b200 import workloads as W                 # noqa: E402

E_RTOL = 1e-5
F_ATOL = 1e-3                # FP32-path bar of north_star
F_ATOL_INTERNAL = 5e-5
G_ATOL = 2e-6
RMSD_TOL = 1e-4


@pytest.fixture(scope="module")
def pfc():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2412_18271_b200 import pfc as m
    m.load_library()
    return m


def _dev(pfc, a3):
    return torch.from_numpy(pfc.pack4(a3)).cuda()


def _errors(pfc, weights, wl, path, cell=False):
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights, mlp_path=path)
    E, F = p.energy_forces(_dev(pfc, wl.pos))
    assert p.status() == 0
    ref = oracle.energy_forces(wl.pos.astype(np.float64), wl.species, wl.sys_offsets, weights, cell=cell,
                               want_intermediates=True)
    _, g = p.intermediates()
    Eh, Fh = E.cpu().numpy().astype(np.float64), F.cpu().numpy().astype(np.float64)
    p.close()
    return {"E": float((np.abs(Eh - ref["E"]) / np.maximum(np.abs(ref["E"]), 1.0)).max()),
            "F": float(np.abs(Fh[:, :3] - ref["F"]).max()),
            "e": float(np.abs(Fh[:, 3] - ref["e"]).max()),
            "g": float(np.abs(g - ref["g"]).max())}


@pytest.mark.parametrize("k", [0, 1, 2, 3, 4])
def test_tf32x3_step0_energy_forces_full_size(pfc, weights, k):
    wl = W.make_config(k)
    err = _errors(pfc, weights, wl, pfc.MLP_TENSOR, cell=(k == 3))
    assert err["E"] <= E_RTOL, err
    assert err["F"] <= F_ATOL_INTERNAL, err
    assert err["e"] <= 1e-5, err
    assert err["g"] <= G_ATOL, err


def test_tf32x3_matches_fp32_path_closely(pfc, weights):
    """The two K3 implementations share no code; their g and F agree to fp32 rounding."""
    wl = W.config4(n_replicas=300)
    out = []
    for path in (pfc.MLP_FP32, pfc.MLP_TENSOR):
        p = pfc.Pfc(wl.species, wl.sys_offsets, weights, mlp_path=path)
        E, F = p.energy_forces(_dev(pfc, wl.pos))
        _, g = p.intermediates()
        out.append((F.cpu().numpy().copy(), g.copy()))
        p.close()
    assert np.abs(out[0][0] - out[1][0]).max() <= 2e-5
    assert np.abs(out[0][1] - out[1][1]).max() <= 2e-6


def test_plain_tf32_misses_the_fp32_bars(pfc, weights):
    """Evidence for the tensor-core decision (north_star (3)): one-term TF32 is 2-3 orders of
    magnitude less accurate in g than the split and misses the internal force target."""
    wl = W.make_config(1)
    e1 = _errors(pfc, weights, wl, pfc.MLP_TENSOR_1TERM)
    e3 = _errors(pfc, weights, wl, pfc.MLP_TENSOR)
    assert e3["g"] <= G_ATOL and e3["F"] <= F_ATOL_INTERNAL
    assert e1["g"] > 50 * e3["g"], (e1, e3)
    assert e1["F"] > F_ATOL_INTERNAL, e1
    assert e1["F"] <= 5e-2                    # still the right function, just coarser


def _trajectory(pfc, weights, wl, n_steps, cell=False, allow_outliers=0):
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights, mlp_path=pfc.MLP_TENSOR)
    pos, vel = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
    E, F = p.set_state(pos, vel)
    p.step(n_steps, wl.dt_fs)
    torch.cuda.synchronize()
    assert p.status() == 0
    ref = oracle.step(wl.pos, wl.vel, wl.species, wl.sys_offsets, weights, wl.dt_fs, n_steps, cell=cell)
    x = pos.cpu().numpy()[:, :3].astype(np.float64)
    d2 = ((x - ref["pos"]) ** 2).sum(1)
    off = wl.sys_offsets
    per_sys = np.sort([float(np.sqrt(d2[off[s]:off[s + 1]].mean())) for s in range(len(off) - 1)])[::-1]
    assert per_sys[allow_outliers] <= RMSD_TOL, per_sys[:4]
    if allow_outliers:
        assert per_sys[0] <= 1e-3, per_sys[:4]
    xf = pos.cpu().numpy()[:, :3]
    at = oracle.energy_forces(xf.astype(np.float64), wl.species, off, weights, cell=cell)
    Fh = F.cpu().numpy().astype(np.float64)
    assert np.abs(Fh[:, :3] - at["F"]).max() <= F_ATOL
    p.close()


def test_tf32x3_trajectory_config0(pfc, weights):
    _trajectory(pfc, weights, W.make_config(0), 100)


def test_tf32x3_trajectory_config1(pfc, weights):
    """The decision case.  Without the truncation compensation 255 of the 256
    replicas stay within 1e-4 A but the most chaotic one (2.0e-5 A on the FP32 path) reaches 4.6e-4 A:
    the accumulator's round-toward-zero loss is one-sided and integrates coherently.  With the
    compensation (the shipped path) every replica stays within the bar (worst 3.8e-5 A)."""
    _trajectory(pfc, weights, W.make_config(1), 100)


def test_uncompensated_tf32x3_misses_the_trajectory_bar(pfc, weights):
    """Evidence for the compensation: switched off (pfc_tuning_t.tc_comp_override with both factors 0)
    the worst replica of config 1 leaves the 1e-4 A bar while all the others keep it."""
    wl = W.make_config(1)
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights, mlp_path=pfc.MLP_TENSOR,
                tuning=pfc.Tuning(tc_comp_override=1, tc_comp_forward=0.0, tc_comp_backward=0.0))
    pos, vel = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
    p.set_state(pos, vel)
    p.step(100, wl.dt_fs)
    torch.cuda.synchronize()
    ref = oracle.step(wl.pos, wl.vel, wl.species, wl.sys_offsets, weights, wl.dt_fs, 100)
    d2 = ((pos.cpu().numpy()[:, :3].astype(np.float64) - ref["pos"]) ** 2).sum(1)
    off = wl.sys_offsets
    per_sys = np.sort([float(np.sqrt(d2[off[s]:off[s + 1]].mean())) for s in range(len(off) - 1)])[::-1]
    assert per_sys[0] > RMSD_TOL and per_sys[1] <= RMSD_TOL, per_sys[:4]
    p.close()


def test_tf32x3_trajectory_config2(pfc, weights):
    _trajectory(pfc, weights, W.make_config(2), 100)


def test_tf32x3_trajectory_config4_subset(pfc, weights):
    _trajectory(pfc, weights, W.config4(n_replicas=64), 100)


def test_tf32x3_bitwise_determinism(pfc, weights):
    wl = W.config4(n_replicas=300)                       # > 148 tiles? no: ~17k rows = 135 tiles + padding
    outs = []
    for _ in range(2):
        p = pfc.Pfc(wl.species, wl.sys_offsets, weights, mlp_path=pfc.MLP_TENSOR)
        pos, vel = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
        E, F = p.set_state(pos, vel)
        p.step(10, 0.5)
        torch.cuda.synchronize()
        outs.append((pos.cpu().numpy().copy(), F.cpu().numpy().copy()))
        p.close()
    for a, b in zip(*outs):
        assert np.array_equal(a, b)


def test_compensation_holds_for_another_weight_draw(pfc):
    """The compensation constants were fitted with the weights of seed 2412.  With
    a different draw (seed 7) the one-sided error of g stays an order of magnitude below the
    uncompensated -2.2e-6 and the 100-step trajectories of 64 replicas of config 1 stay within the bar."""
    w7 = W.make_weights(7)
    wl = W.config1(n_replicas=64)
    ref = oracle.energy_forces(wl.pos.astype(np.float64), wl.species, wl.sys_offsets, w7, want_intermediates=True)
    p = pfc.Pfc(wl.species, wl.sys_offsets, w7, mlp_path=pfc.MLP_TENSOR)
    pos, vel = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
    E, F = p.energy_forces(pos)
    torch.cuda.synchronize()
    _, g = p.intermediates()
    dg = g.astype(np.float64) - ref["g"]
    slope = float(np.sum(dg * ref["g"]) / np.sum(ref["g"] ** 2))
    assert abs(slope) <= 5e-7, slope
    assert np.abs(dg).max() <= G_ATOL
    p.set_state(pos, vel)
    p.step(100, wl.dt_fs)
    torch.cuda.synchronize()
    r = oracle.step(wl.pos, wl.vel, wl.species, wl.sys_offsets, w7, wl.dt_fs, 100)
    d2 = ((pos.cpu().numpy()[:, :3].astype(np.float64) - r["pos"]) ** 2).sum(1)
    off = wl.sys_offsets
    worst = max(float(np.sqrt(d2[off[s]:off[s + 1]].mean())) for s in range(len(off) - 1))
    assert worst <= RMSD_TOL, worst
    p.close()
