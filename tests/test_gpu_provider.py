"""GPU parity of the provider-style entry point in the paper's units (
PAPER.md:47, :62, :67, :102, :121): positions in nm in, kJ/mol and kJ/mol/nm out, against the fp64
oracle converted with 1 nm = 10 A, 1 eV = 96.485332 kJ/mol."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle                                                    # noqa: E402
from paper_2412_18271_b200 import workloads as W                 # noqa: E402

EV_KJ = 96.485332


@pytest.fixture(scope="module")
def pfc():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2412_18271_b200 import pfc as m
    m.load_library()
    return m


def test_energy_and_forces_in_openmm_units(pfc):
    wl, w = W.config1(n_replicas=12), W.make_weights()
    p = pfc.Pfc(wl.species, wl.sys_offsets, w)
    pos_nm = torch.from_numpy(np.ascontiguousarray(wl.pos / np.float32(10.0), dtype=np.float32)).cuda()
    E, F = p.energy_forces_nm(pos_nm)
    E2, F2 = p.energy_forces_nm(pos_nm, want_forces=False)           # RETURN_ENERGY mode
    torch.cuda.synchronize()
    assert F2 is None and torch.equal(E, E2)
    # the oracle sees exactly the positions the library computes with: fl(10 * fl(x / 10))
    x = (pos_nm.cpu().numpy() * np.float32(10.0)).astype(np.float64)
    ref = oracle.energy_forces(x, wl.species, wl.sys_offsets, w)
    Eh, Fh = E.cpu().numpy().astype(np.float64), F.cpu().numpy().astype(np.float64)
    assert (np.abs(Eh - EV_KJ * ref["E"]) <= 1e-5 * EV_KJ * np.maximum(np.abs(ref["E"]), 1.0)).all()
    assert np.abs(Fh - 10.0 * EV_KJ * ref["F"]).max() <= 1e-3 * 10.0 * EV_KJ
    assert np.abs(Fh - 10.0 * EV_KJ * ref["F"]).max() <= 5e-5 * 10.0 * EV_KJ      # the internal FP32 target
    assert p.status() == 0
    p.close()


def test_provider_call_is_refused_while_a_host_state_is_bound(pfc):
    wl, w = W.config0(), W.make_weights()
    p = pfc.Pfc(wl.species, wl.sys_offsets, w)
    ph = torch.from_numpy(pfc.pack4(wl.pos)).pin_memory()
    vh = torch.from_numpy(pfc.pack4(wl.vel)).pin_memory()
    Eh = torch.empty(1, dtype=torch.float32).pin_memory()
    p.run_host(ph, vh, 1, 0.5, Eh)
    pos_nm = torch.from_numpy(np.ascontiguousarray(wl.pos / np.float32(10.0))).cuda()
    with pytest.raises(pfc.PfcError):
        p.energy_forces_nm(pos_nm)
    p.close()


# ---- the provider call as a graph replay, per-handle state, steps per graph ----------------------
def _dev(pfc, a3):
    return torch.from_numpy(pfc.pack4(a3)).cuda()


def test_energy_forces_is_a_cached_graph_replay(pfc):
    """pfc_energy_forces replays one CUDA graph per (pos, E, F) buffer triple (the
    paper's CUDA-Graph finding applied to the provider call itself).  Same buffers, new contents ->
    the replay sees the new positions; more distinct triples than cache slots -> eviction and
    re-capture stay correct; results equal the kernel-by-kernel sequence of pfc_profile_stages."""
    wl, w = W.config1(n_replicas=6), W.make_weights()
    p = pfc.Pfc(wl.species, wl.sys_offsets, w)
    ref0 = oracle.energy_forces(wl.pos.astype(np.float64), wl.species, wl.sys_offsets, w)
    pos2 = (wl.pos + np.float32(0.01) * np.sin(np.arange(wl.pos.size, dtype=np.float32)).reshape(wl.pos.shape)).astype(np.float32)
    ref2 = oracle.energy_forces(pos2.astype(np.float64), wl.species, wl.sys_offsets, w)
    x = _dev(pfc, wl.pos)
    E = torch.empty(wl.n_systems, device="cuda"); F = torch.empty(wl.n_atoms, 4, device="cuda")
    p.energy_forces(x, E, F)                                   # capture + replay
    F0 = F.cpu().numpy().copy()
    assert np.abs(F0[:, :3] - ref0["F"]).max() <= 5e-5
    x.copy_(_dev(pfc, pos2))
    p.energy_forces(x, E, F)                                   # replay of the cached graph on new contents
    assert np.abs(F.cpu().numpy()[:, :3] - ref2["F"]).max() <= 5e-5
    assert np.abs(E.cpu().numpy() - ref2["E"]).max() <= 1e-5 * np.maximum(np.abs(ref2["E"]), 1.0).max()
    outs = []
    for k in range(7):                                         # 7 distinct triples > 4 cache slots
        xs_ = _dev(pfc, wl.pos if k % 2 == 0 else pos2)
        Ek, Fk = p.energy_forces(xs_)
        outs.append((xs_, Ek, Fk))
    for k, (_, Ek, Fk) in enumerate(outs):
        r = ref0 if k % 2 == 0 else ref2
        assert np.abs(Fk.cpu().numpy()[:, :3] - r["F"]).max() <= 5e-5
    x.copy_(_dev(pfc, wl.pos))
    p.energy_forces(x, E, F)                                   # the first triple again (evicted: re-captured)
    assert np.array_equal(F.cpu().numpy(), F0)                 # bit-reproducible
    E2 = torch.empty_like(E); F2 = torch.empty_like(F)
    p.profile_stages(x, E2, F2)                                # raw launches, no graph
    assert torch.equal(F, F2) and torch.equal(E, E2)
    assert p.status() == 0
    p.close()


def test_two_live_handles_with_different_masses(pfc):
    """pfc_desc_t.masses_amu is per handle (hydrogen mass repartitioning next to standard masses):
    interleaved stepping of two live handles, each against oracle.step with its own masses."""
    wl, w = W.config1(n_replicas=4), W.make_weights()
    m_std = np.array([1.008, 12.011, 14.007, 15.999])
    m_hmr = np.array([3.024, 9.995, 11.991, 13.983])
    handles = []
    for m in (m_std, m_hmr):
        p = pfc.Pfc(wl.species, wl.sys_offsets, w, masses_amu=m)
        x, v = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
        p.set_state(x, v)
        handles.append((p, x, v, m))
    for _ in range(4):                                         # interleave: 4 x 10 steps each
        for p, _, _, _ in handles:
            p.step(10, 0.5)
    torch.cuda.synchronize()
    for p, x, v, m in handles:
        ref = oracle.step(wl.pos, wl.vel, wl.species, wl.sys_offsets, w, 0.5, 40, masses=m)
        d2 = ((x.cpu().numpy()[:, :3].astype(np.float64) - ref["pos"]) ** 2).sum(1)
        off = wl.sys_offsets
        assert max(np.sqrt(d2[off[s]:off[s + 1]].mean()) for s in range(len(off) - 1)) <= 2e-5
        assert np.abs(v.cpu().numpy()[:, :3] - ref["vel"]).max() <= 2e-5
        p.close()
    # the two trajectories really differ (a shared mass table would make them equal)
    a, b = handles[0][1].cpu().numpy(), handles[1][1].cpu().numpy()
    assert np.abs(a - b).max() > 1e-3


@pytest.mark.parametrize("langevin", [False, True])
def test_steps_per_graph_is_bitwise_neutral(pfc, langevin):
    """pfc_step captures several MD steps per CUDA graph (default 16; fewer host launches in the
    launch-bound regime of PAPER.md:94).  The trajectory is bit-identical to one graph per step,
    frames included (a frame boundary falls back to single-step graphs)."""
    wl, w = W.config1(n_replicas=5), W.make_weights()
    res = []
    for k in (1, 16, 5):
        p = pfc.Pfc(wl.species, wl.sys_offsets, w, tuning=pfc.Tuning(steps_per_graph=k))
        assert p.steps_per_graph() == k
        x, v = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
        frames = torch.zeros(4, wl.n_atoms, 4, device="cuda")
        E, F = p.set_state(x, v)
        p.set_frames(frames, 20)
        for n in (50, 37):
            if langevin:
                p.step_langevin(n, 0.5, 1e-3, 300.0, seed=11)
            else:
                p.step(n, 0.5)
        torch.cuda.synchronize()
        assert p.frames_written() == 4 and p.status() == 0
        res.append([t.cpu().numpy().copy() for t in (x, v, E, F, frames)])
        p.close()
    for other in res[1:]:
        for a, b in zip(res[0], other):
            assert np.array_equal(a, b)
