"""GPU parity of the tensor-core K3 (tcgen05 kind::f16, fp16 hi|lo 3-term split, fp32 accumulate;
DESIGN.md section 5) against the fp64 oracle, at the SAME bars as the FP32 path (north_star allows
5e-3 eV/A for a reduced-precision MLP; the split meets the FP32 bars, so those are the ones asserted),
the evidence that one 16-bit term does not, and the truncation compensation: calibrated by the library
against its own FP32 MLP, checked here against the oracle -- on the standard weights, on other draws and
on weight sets that are not iid (all-positive, rescaled, low-rank, sign-alternating).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle                                                    # noqa: E402
from paper_2412_18271_b200 import workloads as W                 # noqa: E402

E_RTOL = 1e-5
F_ATOL = 1e-3                # FP32-path bar of north_star
F_ATOL_INTERNAL = 5e-5       # other weight sets
G_ATOL = 2e-6                # other weight sets
F_ATOL_STEP0 = 6e-6          # standard weights, the five configs: <= 3x the measured worst case
G_ATOL_STEP0 = 1.2e-6
E_ATOM_ATOL = 3e-6
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
def test_f16x3_step0_energy_forces_full_size(pfc, weights, k):
    wl = W.make_config(k)
    err = _errors(pfc, weights, wl, pfc.MLP_TENSOR, cell=(k == 3))
    assert err["E"] <= E_RTOL, err
    assert err["F"] <= F_ATOL_STEP0, err
    assert err["e"] <= E_ATOM_ATOL, err
    assert err["g"] <= G_ATOL_STEP0, err


def test_f16x3_matches_fp32_path_closely(pfc, weights):
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


def test_plain_fp16_misses_the_fp32_bars(pfc, weights):
    """Evidence for the tensor-core decision (north_star (3)): one fp16 term is 2-3 orders of
    magnitude less accurate in g than the split and misses the internal force target."""
    wl = W.make_config(1)
    e1 = _errors(pfc, weights, wl, pfc.MLP_TENSOR_1TERM)
    e3 = _errors(pfc, weights, wl, pfc.MLP_TENSOR)
    assert e3["g"] <= G_ATOL and e3["F"] <= F_ATOL_INTERNAL
    assert e1["g"] > 50 * e3["g"], (e1, e3)
    assert e1["F"] > F_ATOL_INTERNAL, e1
    assert e1["F"] <= 5e-2                    # still the right function, just coarser


COND_FACTOR = 4.0


def _conditioning(k):
    """tests/golden/cfg{k}_conditioning.txt: the oracle's own one-ulp sensitivity per replica (reading S30)."""
    import os
    t = np.loadtxt(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"cfg{k}_conditioning.txt"))
    return t[:, 2:].max(axis=1)


def _rmsd(x, xref, off):
    d2 = ((x - xref) ** 2).sum(1)
    return np.array([float(np.sqrt(d2[off[s]:off[s + 1]].mean())) for s in range(len(off) - 1)])


def _trajectory(pfc, weights, wl, n_steps, cell=False, cond=None, tuning=None):
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights, mlp_path=pfc.MLP_TENSOR, tuning=tuning)
    pos, vel = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
    E, F = p.set_state(pos, vel)
    p.step(n_steps, wl.dt_fs)
    torch.cuda.synchronize()
    assert p.status() == 0
    assert p.mlp_path() == pfc.MLP_TENSOR
    ref = oracle.step(wl.pos, wl.vel, wl.species, wl.sys_offsets, weights, wl.dt_fs, n_steps, cell=cell)
    per_sys = _rmsd(pos.cpu().numpy()[:, :3].astype(np.float64), ref["pos"], wl.sys_offsets)
    bound = np.full(wl.n_systems, RMSD_TOL)
    if cond is not None:
        bound = np.maximum(RMSD_TOL, COND_FACTOR * _conditioning(cond)[:wl.n_systems])
    assert (per_sys <= bound).all(), np.sort(per_sys / bound)[::-1][:4]
    xf = pos.cpu().numpy()[:, :3]
    at = oracle.energy_forces(xf.astype(np.float64), wl.species, wl.sys_offsets, weights, cell=cell)
    Fh = F.cpu().numpy().astype(np.float64)
    assert np.abs(Fh[:, :3] - at["F"]).max() <= F_ATOL
    p.close()
    return per_sys


def test_f16x3_trajectory_config0(pfc, weights):
    _trajectory(pfc, weights, W.make_config(0), 100)


def test_f16x3_trajectory_config1(pfc, weights):
    """All 256 replicas.  255 of them stay below 1e-5 A; replica 68 is the one whose fp64 trajectory itself
    moves by 1.1e-4 A under a one-ulp input error (tests/golden/cfg1_conditioning.txt), so its bar is
    COND_FACTOR times that (reading S30); with the calibrated compensation it lands at about 3e-5 A."""
    per_sys = _trajectory(pfc, weights, W.make_config(1), 100, cond=1)
    assert np.sort(per_sys)[-2] <= 2e-5 and np.median(per_sys) <= 2e-6, np.sort(per_sys)[-4:]


def test_f16x3_trajectory_config2(pfc, weights):
    _trajectory(pfc, weights, W.make_config(2), 100)


def test_f16x3_trajectory_config4_subset(pfc, weights):
    _trajectory(pfc, weights, W.config4(n_replicas=64), 100, cond=4)


def test_f16x3_bitwise_determinism(pfc, weights):
    wl = W.config4(n_replicas=300)                       # ~17k rows = 135 tiles + padding
    outs = []
    for _ in range(2):
        p = pfc.Pfc(wl.species, wl.sys_offsets, weights, mlp_path=pfc.MLP_TENSOR)
        pos, vel = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
        E, F = p.set_state(pos, vel)
        p.step(10, 0.5)
        torch.cuda.synchronize()
        outs.append((pos.cpu().numpy().copy(), F.cpu().numpy().copy(), p.tc_calibration()))
        p.close()
    for a, b in zip(*outs):
        assert np.array_equal(a, b)


# ---- the truncation compensation ----------------------------------------
def _slopes(pfc, w, wl, path, tuning=None):
    """First evaluation of a fresh handle: least-squares slopes of the errors of e_i and g on the oracle's
    values, largest errors, the path the handle ended up on and its calibration table."""
    ref = oracle.energy_forces(wl.pos.astype(np.float64), wl.species, wl.sys_offsets, w, want_intermediates=True)
    p = pfc.Pfc(wl.species, wl.sys_offsets, w, mlp_path=path, tuning=tuning)
    E, F = p.energy_forces(_dev(pfc, wl.pos))
    torch.cuda.synchronize()
    assert p.status() == 0
    _, g = p.intermediates()
    Eh, Fh = E.cpu().numpy().astype(np.float64), F.cpu().numpy().astype(np.float64)
    de, dg = Fh[:, 3] - ref["e"], g.astype(np.float64) - ref["g"]
    out = {"slope_e": float((de * ref["e"]).sum() / (ref["e"] ** 2).sum()),
           "slope_g": float((dg * ref["g"]).sum() / (ref["g"] ** 2).sum()),
           "g": float(np.abs(dg).max()), "F": float(np.abs(Fh[:, :3] - ref["F"]).max()),
           "E": float((np.abs(Eh - ref["E"]) / np.maximum(np.abs(ref["E"]), 1.0)).max()),
           "path": p.mlp_path(), "calib": p.tc_calibration()}
    p.close()
    return out


def test_uncompensated_split_shrinks_and_the_calibration_removes_it(pfc, weights):
    """Evidence for the compensation.  The tensor core's accumulate step rounds toward zero: switched off
    (pfc_tuning_t.tc_comp_override with both factors 0) e_i and g come out systematically too small --
    slopes of about -7e-7 and -1.1e-6 against the fp64 oracle, where the FP32 MLP shows +-1e-8.  The
    library calibrates two scales per element against its OWN FP32 MLP on the first batch; checked here
    against the oracle, which the library never sees: |slope| <= 1e-7 on both."""
    wl = W.make_config(1)
    raw = _slopes(pfc, weights, wl, pfc.MLP_TENSOR, tuning=pfc.Tuning(tc_comp_override=1, tc_comp_forward=0.0,
                                                                     tc_comp_backward=0.0))
    assert raw["slope_g"] < -5e-7 and raw["slope_e"] < -2e-7, raw
    cal = _slopes(pfc, weights, wl, pfc.MLP_TENSOR)
    assert abs(cal["slope_g"]) <= 1e-7 and abs(cal["slope_e"]) <= 1e-7, cal
    assert cal["g"] <= G_ATOL and cal["F"] <= F_ATOL_INTERNAL and cal["E"] <= E_RTOL, cal
    t = cal["calib"]
    assert (t[:, 6] == 1).all() and (t[:, 7] == 0).all()                  # final, no fallback
    assert (t[:, 1] >= 0.3).all() and (t[:, 1] <= 1.6).all(), t[:, :2]    # lambda_b: the mean-field estimate is 1
    assert (np.abs(t[:, 2:4]) <= 3e-7).all(), t                           # residual slopes against the FP32 MLP
    fp = _slopes(pfc, weights, wl, pfc.MLP_FP32)
    assert abs(fp["slope_g"]) <= 5e-8 and abs(fp["slope_e"]) <= 5e-8, fp


def _weights_variant(kind):
    """Weight sets that break the iid N(0, 1/fan_in) statistics the round-1 constants were fitted on."""
    if kind in ("seed7", "seed99"):
        return W.make_weights(int(kind[4:]))
    w = W.make_weights().copy()
    D0, D1, D2, D3, per = 384, 160, 128, 96, 94689
    for e in range(4):
        b = w[e * per:(e + 1) * per]
        o2 = D1 * D0 + D1
        o3 = o2 + D2 * D1 + D2
        W1, W2, W3 = b[:D1 * D0].reshape(D1, D0), b[o2:o2 + D2 * D1].reshape(D2, D1), b[o3:o3 + D3 * D2].reshape(D3, D2)
        if kind == "positive_W2":
            W2[:] = np.abs(W2) * 0.3
        elif kind == "W1_times_8_W2_over_8":
            W1 *= 8
            W2 /= 8
        elif kind == "rank4_W1":
            rng = np.random.Generator(np.random.PCG64(5 + e))
            W1[:] = (rng.standard_normal((D1, 4)) @ rng.standard_normal((4, D0)) / np.sqrt(4 * D0)).astype(np.float32)
        elif kind == "alternating_W3":
            W3[:] = np.abs(W3) * np.where(np.arange(D2) % 2 == 0, 1.0, -1.0)[None, :]
        elif kind == "all_positive":
            W1[:] = np.abs(W1) * 0.2
            W2[:] = np.abs(W2) * 0.2
            W3[:] = np.abs(W3) * 0.3
    return w


@pytest.mark.parametrize("kind", ["seed7", "seed99", "positive_W2", "W1_times_8_W2_over_8", "rank4_W1",
                                  "alternating_W3", "all_positive"])
def test_compensation_on_other_weight_sets(pfc, kind):
    """PFC_MLP_AUTO on 256 replicas of config 1 (5,632 atoms: the tensor path) with weights the compensation
    was never tuned on.  Whatever path the handle ends up on after its calibration check must hold, against the
    oracle: slope of the g error <= 2e-7 in magnitude (uncompensated: -1e-6 .. -2.3e-6), max|dg| <= 2e-6, the
    energy and force bars; and the 100-step trajectories stay within max(1e-4 A, COND_FACTOR x the oracle's own
    one-ulp sensitivity on THESE weights) -- several of these potentials are chaotic enough that the FP32 MLP
    misses 1e-4 A on a replica or two as well."""
    w = _weights_variant(kind)
    wl = W.make_config(1)
    off = wl.sys_offsets
    out = _slopes(pfc, w, wl, pfc.MLP_AUTO)
    assert out["path"] in (pfc.MLP_TENSOR, pfc.MLP_FP32)
    if out["path"] == pfc.MLP_TENSOR:
        assert (out["calib"][:, 7] == 0).all()
    assert abs(out["slope_g"]) <= 2e-7 and abs(out["slope_e"]) <= 2e-7, out
    assert out["g"] <= G_ATOL and out["F"] <= F_ATOL_INTERNAL and out["E"] <= E_RTOL, out
    # conditioning of the trajectory bar on these weights: the oracle against itself, inputs moved by one ulp
    ref = oracle.step(wl.pos, wl.vel, wl.species, off, w, wl.dt_fs, 100)["pos"]
    sgn = np.random.Generator(np.random.PCG64(1)).integers(0, 2, size=wl.pos.shape) * 2 - 1
    moved = np.where(sgn > 0, np.nextafter(wl.pos, np.float32(np.inf)), np.nextafter(wl.pos, np.float32(-np.inf)))
    sens = _rmsd(oracle.step(moved.astype(np.float32), wl.vel, wl.species, off, w, wl.dt_fs, 100)["pos"], ref, off)
    p = pfc.Pfc(wl.species, off, w, mlp_path=pfc.MLP_AUTO)
    pos, vel = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
    p.set_state(pos, vel)
    p.step(100, wl.dt_fs)
    torch.cuda.synchronize()
    assert p.status() == 0
    per_sys = _rmsd(pos.cpu().numpy()[:, :3].astype(np.float64), ref, off)
    p.close()
    bound = np.maximum(RMSD_TOL, COND_FACTOR * sens)
    assert (per_sys <= bound).all(), (kind, np.sort(per_sys / bound)[::-1][:4])
    assert np.median(per_sys) <= 1e-5, np.median(per_sys)


def test_auto_goes_back_to_fp32_when_the_calibration_check_fails(pfc, weights):
    """A weight set the fp16-split operands cannot carry: with a bias of 1e6 on the second hidden layer the
    activations h2 (the A operand of the third GEMM) exceed fp16's range.  The FP32 MLP evaluates it without
    trouble; the tensor MLP returns non-finite values on the calibration batch, the check fails, and a
    PFC_MLP_AUTO handle continues on the FP32 MLP -- whose results are then held to the usual bars."""
    w = weights.copy()
    D0, D1, D2, per = 384, 160, 128, 94689
    for e in range(4):
        o_b2 = e * per + D1 * D0 + D1 + D2 * D1
        w[o_b2:o_b2 + D2] += 1.0e6
    wl = W.make_config(1)
    p = pfc.Pfc(wl.species, wl.sys_offsets, w, mlp_path=pfc.MLP_AUTO)
    assert p.mlp_path() == pfc.MLP_TENSOR                      # before the first evaluation: by size
    E, F = p.energy_forces(_dev(pfc, wl.pos))
    torch.cuda.synchronize()
    assert p.mlp_path() == pfc.MLP_FP32 and (p.tc_calibration()[:, 7] == 1).all()
    assert p.status() == 0
    ref = oracle.energy_forces(wl.pos.astype(np.float64), wl.species, wl.sys_offsets, w)
    Eh, Fh = E.cpu().numpy().astype(np.float64), F.cpu().numpy().astype(np.float64)
    assert (np.abs(Eh - ref["E"]) <= E_RTOL * np.maximum(np.abs(ref["E"]), 1.0)).all()
    assert np.abs(Fh[:, :3] - ref["F"]).max() <= F_ATOL_INTERNAL * max(1.0, np.abs(ref["F"]).max())
    p.close()
    # asked for explicitly, the tensor path stays (and reports what the check saw)
    q = pfc.Pfc(wl.species, wl.sys_offsets, w, mlp_path=pfc.MLP_TENSOR)
    q.energy_forces(_dev(pfc, wl.pos))
    torch.cuda.synchronize()
    assert q.mlp_path() == pfc.MLP_TENSOR and (q.tc_calibration()[:, 7] == 0).all()
    q.close()
