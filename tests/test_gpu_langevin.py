"""GPU parity of the Langevin integrator and trajectory frames (O9)
against the fp64 oracle: same Philox4x32-10 counter-based normals on both sides (each side's own
implementation), same BAOAB splitting.  Bars: per-system RMSD <= 1e-4 A after 100 steps (the
north_star trajectory bar), velocities within the DESIGN.md bound; frames equal the positions the
oracle has at those steps."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle                                                    # noqa: E402
from paper_2412_18271_b200 import workloads as W                 # noqa: E402

RMSD_TOL = 1e-4
VEL_TOL = 4e-5
GAMMA = 1e-4          # 0.1 ps^-1, the paper's protocol


@pytest.fixture(scope="module")
def pfc():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2412_18271_b200 import pfc as m
    m.load_library()
    return m


def _dev(pfc, a3):
    return torch.from_numpy(pfc.pack4(a3)).cuda()


def _rmsd(x, xref, off):
    d2 = ((x - xref) ** 2).sum(1)
    return np.array([np.sqrt(d2[off[s]:off[s + 1]].mean()) for s in range(len(off) - 1)])


def _batch():
    a, b = W.config0(), W.config1(n_replicas=6)
    pos = np.concatenate([a.pos, b.pos]); vel = np.concatenate([a.vel, b.vel])
    species = np.concatenate([a.species, b.species])
    off = np.concatenate([a.sys_offsets, b.sys_offsets[1:] + a.n_atoms]).astype(np.int32)
    return pos, vel, species, off


@pytest.mark.parametrize("gamma,T", [(GAMMA, 300.0), (0.02, 500.0)])
def test_langevin_trajectory_matches_oracle(pfc, gamma, T):
    """100 steps of 0.5 fs; the strong-friction case makes the random kicks dominate the motion,
    so a wrong generator, counter or noise amplitude cannot hide."""
    pos, vel, species, off = _batch()
    w = W.make_weights()
    p = pfc.Pfc(species, off, w)
    x, v = _dev(pfc, pos), _dev(pfc, vel)
    p.set_state(x, v)
    p.step_langevin(60, 0.5, gamma, T, seed=2412)
    p.step_langevin(40, 0.5, gamma, T, seed=2412)     # the step counter continues across calls
    torch.cuda.synchronize()
    ref = oracle.step_langevin(pos, vel, species, off, w, 0.5, 100, gamma, T, 2412)
    xh, vh = x.cpu().numpy()[:, :3].astype(np.float64), v.cpu().numpy()[:, :3].astype(np.float64)
    assert _rmsd(xh, ref["pos"], off).max() <= RMSD_TOL
    assert np.abs(vh - ref["vel"]).max() <= VEL_TOL
    assert p.status() == 0
    # the noise really moved the system: against plain velocity-Verlet the trajectories differ
    nve = oracle.step(pos, vel, species, off, w, 0.5, 100)
    assert _rmsd(ref["pos"], nve["pos"], off).min() > (1e-3 if gamma > 1e-3 else 1e-5)
    p.close()


def test_zero_friction_equals_verlet_on_device(pfc):
    pos, vel, species, off = _batch()
    w = W.make_weights()
    out = []
    for lang in (False, True):
        p = pfc.Pfc(species, off, w)
        x, v = _dev(pfc, pos), _dev(pfc, vel)
        p.set_state(x, v)
        if lang:
            p.step_langevin(50, 0.5, 0.0, 300.0, seed=1)
        else:
            p.step(50, 0.5)
        torch.cuda.synchronize()
        out.append((x.cpu().numpy()[:, :3].astype(np.float64), v.cpu().numpy()[:, :3].astype(np.float64)))
        p.close()
    assert _rmsd(out[0][0], out[1][0], off).max() <= 2e-6      # two half drifts vs one: fp32 rounding only
    assert np.abs(out[0][1] - out[1][1]).max() <= 2e-6


def test_seed_and_reset_semantics(pfc):
    """Same seed after pfc_set_state replays the same noise bit for bit; another seed does not."""
    pos, vel, species, off = _batch()
    w = W.make_weights()
    p = pfc.Pfc(species, off, w)
    res = []
    for seed in (7, 7, 8):
        x, v = _dev(pfc, pos), _dev(pfc, vel)
        p.set_state(x, v)
        p.step_langevin(20, 0.5, 0.01, 300.0, seed=seed)
        torch.cuda.synchronize()
        res.append(x.cpu().numpy().copy())
    assert np.array_equal(res[0], res[1])
    assert not np.array_equal(res[0], res[2])
    p.close()


def test_frames_hold_the_positions_of_their_steps(pfc):
    """Frames every 10 steps of a 50-step NVE run and of a Langevin run: frame k = x after step 10(k+1)."""
    pos, vel, species, off = _batch()
    w = W.make_weights()
    p = pfc.Pfc(species, off, w)
    n = pos.shape[0]
    for lang in (False, True):
        x, v = _dev(pfc, pos), _dev(pfc, vel)
        frames = torch.zeros(4, n, 4, dtype=torch.float32, device="cuda")     # room for 4 of the 5 frames
        p.set_state(x, v)
        p.set_frames(frames, 10)
        for _ in range(5):
            if lang:
                p.step_langevin(10, 0.5, GAMMA, 300.0, seed=3)
            else:
                p.step(10, 0.5)
        torch.cuda.synchronize()
        assert p.frames_written() == 4                                        # capped at max_frames
        fh = frames.cpu().numpy()[:, :, :3].astype(np.float64)
        for k in range(4):
            if lang:
                ref = oracle.step_langevin(pos, vel, species, off, w, 0.5, 10 * (k + 1), GAMMA, 300.0, 3)
            else:
                ref = oracle.step(pos, vel, species, off, w, 0.5, 10 * (k + 1))
            assert _rmsd(fh[k], ref["pos"], off).max() <= RMSD_TOL, (lang, k)
        p.set_frames(None, 0)
    p.close()
