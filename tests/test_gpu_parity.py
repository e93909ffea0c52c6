"""GPU parity: the CUDA path (through the C ABI, libpfc.so) against the fp64 oracle on
the same seeded inputs.  Bars (BASELINE.json:north_star):
  * neighbour lists bit-exact (int32 CSR arrays equal);
  * per-system energy |dE| <= 1e-5 * max(|E_ref|, 1 eV)          (S14);
  * forces max|dF| <= 1e-3 eV/A (FP32 path; we also hold a 5e-5 internal target);
  * trajectories: RMSD <= 1e-4 A per system after 100 steps of 0.5 fs.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle                                                    # noqa: E402
from paper_2412_18271_b200 import workloads as W                 # noqa: E402

E_RTOL = 1e-5
F_ATOL = 1e-3
F_ATOL_INTERNAL = 5e-5       # dense / unusual test geometries
RMSD_TOL = 1e-4
VEL_TOL = 4e-5
# Builder-set bounds on the five configs at step 0, each <= 3x the worst value measured on either MLP path
# (max|dF| 1.9e-6, max|daev| 5.3e-6, max|dg| 3.9e-7, max|de_i| 8.8e-7)
F_ATOL_STEP0 = 6e-6
AEV_ATOL = 1e-5
G_ATOL = 1.2e-6
E_ATOM_ATOL = 3e-6


@pytest.fixture(scope="module")
def pfc():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2412_18271_b200 import pfc as m
    m.load_library()
    return m


def _cfg(k):
    if k == 4:
        return W.config4()
    return W.make_config(k)


_cache = {}


def cfg(k):
    if k not in _cache:
        _cache[k] = _cfg(k)
    return _cache[k]


def _dev(pfc, a3):
    return torch.from_numpy(pfc.pack4(a3)).cuda()


def _rmsd_per_system(x, xref, off):
    d2 = ((x - xref) ** 2).sum(1)
    return np.array([np.sqrt(d2[off[s]:off[s + 1]].mean()) for s in range(len(off) - 1)])


def _assert_lists_equal(got, ref):
    for name, a, b in zip(("r_off", "r_idx", "a_off", "a_idx"), got, ref):
        assert a.dtype == np.int32 and a.shape == b.shape, name
        assert np.array_equal(a, b), f"{name} differs"


def _check_energy_forces(E, F, ref, tight=True):
    Eh = E.cpu().numpy().astype(np.float64)
    Fh = F.cpu().numpy().astype(np.float64)
    tol_e = E_RTOL * np.maximum(np.abs(ref["E"]), 1.0)
    assert (np.abs(Eh - ref["E"]) <= tol_e).all(), float((np.abs(Eh - ref["E"]) / tol_e).max())
    dF = np.abs(Fh[:, :3] - ref["F"]).max()
    assert dF <= F_ATOL, dF
    de = np.abs(Fh[:, 3] - ref["e"]).max()
    if tight:                                                    # the generators' states (step 0)
        assert dF <= F_ATOL_STEP0, dF
        assert de <= E_ATOM_ATOL, de
    else:                                                        # evolved states: atoms in close contacts carry larger e_i
        assert de <= 1e-5 * max(1.0, np.abs(ref["e"]).max()), de
    return dF


# ---- step 0 on every config at full size: lists, E, F --------------------------------
# (the default MLP path is PFC_MLP_AUTO: the calibrated tensor-core MLP from 1,024 atoms on -- configs 1 to 4 --,
# the FP32 cluster kernel on config 0; "fp32" pins the FP32 kernels on the larger configs as well)
@pytest.mark.parametrize("k,path", [(0, "auto"), (1, "auto"), (2, "auto"), (3, "auto"), (4, "auto"),
                                    (1, "fp32"), (2, "fp32"), (3, "fp32"), (4, "fp32")])
def test_step0_lists_energy_forces_full_size(pfc, weights, k, path):
    wl = cfg(k)
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights, mlp_path=pfc.MLP_AUTO if path == "auto" else pfc.MLP_FP32)
    assert p.mlp_path() == (pfc.MLP_TENSOR if (path == "auto" and wl.n_atoms >= 1024) else pfc.MLP_FP32)
    E, F = p.energy_forces(_dev(pfc, wl.pos))
    assert p.status() == 0
    # the definition is the O(N^2) enumeration; config 3 (20,000 atoms) goes through the
    # oracle's cell list, which test_oracle_pins pins to the enumeration (P7)
    _assert_lists_equal(p.neighbors(), oracle.neighbors(wl.pos, wl.sys_offsets, cell=(k == 3)))
    ref = oracle.energy_forces(wl.pos.astype(np.float64), wl.species, wl.sys_offsets, weights,
                               cell=(k == 3), want_intermediates=True)
    _check_energy_forces(E, F, ref)
    aev, g = p.intermediates()
    assert np.abs(aev - ref["aev"]).max() <= AEV_ATOL
    assert np.abs(g - ref["g"]).max() <= G_ATOL
    p.close()


def test_config3_brute_force_enumeration_matches_cell_path(pfc, weights):
    """K1's cell list against the O(N^2) definition directly, on a cut of config 3 that is
    still above BRUTE_MAX (so the GPU uses cells) -- independent of the oracle's cell list."""
    wl = W.config3(n_atoms=5000)
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights)
    p.energy_forces(_dev(pfc, wl.pos))
    _assert_lists_equal(p.neighbors(), oracle.neighbors(wl.pos, wl.sys_offsets, cell=False))
    p.close()


# ---- 100-step trajectories -----------------------------------------------------------
COND_FACTOR = 4.0     # a replica may miss 1e-4 A only within this factor of its own one-ulp sensitivity (S30)


def _conditioning(k):
    """tests/golden/cfg{k}_conditioning.txt (written by make_conditioning.py from the oracle alone): per
    replica of config k (1 or 4), how far the fp64 oracle's own 100-step trajectory moves when its inputs
    are disturbed by one fp32 ulp -- the worst of the recorded disturbances."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"cfg{k}_conditioning.txt")
    t = np.loadtxt(path)
    assert np.array_equal(t[:, 0], np.arange(t.shape[0]))
    return t[:, 1].astype(int), t[:, 2:].max(axis=1)


def _trajectory(pfc, weights, wl, n_steps, cell=False, mlp_path=None, cond=None):
    """cond = config index with a conditioning table (reading S30): the bar of system s is then
    max(1e-4 A, COND_FACTOR * its one-ulp sensitivity) -- on config 1 that matters for one replica (68),
    whose fp64 trajectory itself moves by 1.1e-4 A under a one-ulp input error."""
    floor = np.zeros(wl.n_systems)
    if cond is not None:
        sizes, sens = _conditioning(cond)
        assert np.array_equal(sizes[:wl.n_systems], np.diff(wl.sys_offsets))
        floor = COND_FACTOR * sens[:wl.n_systems]
    rel = np.maximum(1.0, floor / RMSD_TOL)                      # 1 wherever the plain bar applies
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights, mlp_path=pfc.MLP_AUTO if mlp_path is None else mlp_path)
    pos, vel = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
    E, F = p.set_state(pos, vel)
    p.step(n_steps, wl.dt_fs)
    torch.cuda.synchronize()
    assert p.status() == 0
    ref = oracle.step(wl.pos, wl.vel, wl.species, wl.sys_offsets, weights, wl.dt_fs, n_steps, cell=cell)
    x = pos.cpu().numpy()[:, :3].astype(np.float64)
    v = vel.cpu().numpy()[:, :3].astype(np.float64)
    rmsd = _rmsd_per_system(x, ref["pos"], wl.sys_offsets)
    assert (rmsd <= RMSD_TOL * rel).all(), (rmsd / rel).max()
    # velocities: north_star states no bound; DESIGN.md "Tolerances" derives one from the position
    # bound: an error that reaches 1e-4 A while growing with e-folding time tau moves at 1e-4/tau;
    # measured tau >= 2.5 fs (config 3, steps 80-100: 3.4 fs) gives 4e-5 A/fs, taken like the
    # position bound as a root mean square over the atoms of a system (reading S29: this potential
    # has no core repulsion; single atoms in a 0.08 A contact at step 100 of config 2 are
    # ill-conditioned).  Thermal H speed is 1.6e-2 A/fs.
    vrms = _rmsd_per_system(v, ref["vel"], wl.sys_offsets)
    assert (vrms <= VEL_TOL * rel).all(), (vrms / rel).max()
    # synchronous state: F and E are those of the FINAL GPU positions -- checked by evaluating
    # the oracle at exactly those fp32 positions (the paper's frame replay), so the
    # force bound is not blurred by the 1e-6..1e-5 A by which the two trajectories differ
    xf = pos.cpu().numpy()[:, :3]
    _assert_lists_equal(p.neighbors(), oracle.neighbors(xf, wl.sys_offsets, cell=cell))
    at = oracle.energy_forces(xf.astype(np.float64), wl.species, wl.sys_offsets, weights, cell=cell)
    _check_energy_forces(E, F, at, tight=False)
    # and the oracle's own final energy is reached to fp32 trajectory accuracy
    Eh = E.cpu().numpy().astype(np.float64)
    assert (np.abs(Eh - ref["pe"][-1]) <= 10 * E_RTOL * np.maximum(np.abs(ref["pe"][-1]), 1.0)).all()
    assert (pos.cpu().numpy()[:, 3] == 0).all() and (vel.cpu().numpy()[:, 3] == 0).all()   # .w untouched
    p.close()
    return rmsd.max()


def test_trajectory_config0(pfc, weights):
    _trajectory(pfc, weights, cfg(0), 100)


def test_trajectory_config1_all_256_replicas(pfc, weights):
    _trajectory(pfc, weights, cfg(1), 100, cond=1)


def test_trajectory_config2(pfc, weights):
    _trajectory(pfc, weights, cfg(2), 100)


def test_trajectory_config3_full_size(pfc, weights):
    _trajectory(pfc, weights, cfg(3), 100, cell=True)


def test_trajectory_fp32_path_configs_1_2_3(pfc, weights):
    """The FP32 MLP on the configs whose default is the tensor-core MLP (config 4: the all-replica test)."""
    _trajectory(pfc, weights, cfg(1), 100, mlp_path=pfc.MLP_FP32, cond=1)
    _trajectory(pfc, weights, cfg(2), 100, mlp_path=pfc.MLP_FP32)
    _trajectory(pfc, weights, cfg(3), 100, cell=True, mlp_path=pfc.MLP_FP32)


def test_trajectory_config4_subset_of_64_replicas(pfc, weights):
    """100 steps on the first 64 replicas of config 4 with every check of _trajectory (velocities, final
    lists, E, F); all 4,096 replicas are integrated by the next test."""
    _trajectory(pfc, weights, W.config4(n_replicas=64), 100, cond=4)


# ---- all 4,096 replicas of config 4, both MLP paths, with the conditioning of the bar (reading S30) ----
_cfg4_ref = {}


def _cfg4_oracle(weights):
    if "pos" not in _cfg4_ref:
        wl = cfg(4)
        _cfg4_ref["pos"] = oracle.step(wl.pos, wl.vel, wl.species, wl.sys_offsets, weights, wl.dt_fs, 100)["pos"]
    return _cfg4_ref["pos"]




@pytest.mark.slow
@pytest.mark.parametrize("path", ["fp32", "tensor"])
def test_trajectory_config4_all_4096_replicas(pfc, weights, path):
    """north_star: trajectories within 1e-4 A RMSD after 100 steps "on all five configs".  On config 4 the
    bar itself is ill-conditioned for a handful of replicas (this random-weight potential has no core
    repulsion; atoms in sub-0.1 A contacts amplify any perturbation): the fp64 oracle, rerun with its fp32
    inputs moved by ONE ulp, leaves the bar on 26 of the 4,096 replicas (tests/golden/cfg4_conditioning.txt).
    Asserted here, per replica s:   RMSD_s <= max(1e-4 A, COND_FACTOR * sensitivity_s),
    i.e. every replica either meets the bar or is within a small factor of what an exact evaluation of the
    same trajectory does under a one-ulp input error; and no more replicas miss the bar than the disturbed
    oracle itself.  The floor (second term) is active for the replicas reported in the message."""
    wl = cfg(4)
    sizes, sens = _conditioning(4)
    assert np.array_equal(sizes, np.diff(wl.sys_offsets))
    ref = _cfg4_oracle(weights)
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights, mlp_path=pfc.MLP_FP32 if path == "fp32" else pfc.MLP_TENSOR)
    pos, vel = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
    p.set_state(pos, vel)
    p.step(100, wl.dt_fs)
    torch.cuda.synchronize()
    assert p.status() == 0
    rmsd = _rmsd_per_system(pos.cpu().numpy()[:, :3].astype(np.float64), ref, wl.sys_offsets)
    p.close()
    bound = np.maximum(RMSD_TOL, COND_FACTOR * sens)
    miss = np.where(rmsd > RMSD_TOL)[0]
    report = (f"{path}: {len(miss)} of 4096 replicas above 1e-4 A (disturbed oracle: {int((sens > RMSD_TOL).sum())}); "
              f"median {np.median(rmsd):.2e}, worst {rmsd.max():.2e}; worst ratio to the bound {(rmsd / bound).max():.2f}; "
              f"replicas on the floor: {[(int(s), float(f'{rmsd[s]:.2e}'), float(f'{sens[s]:.2e}')) for s in miss]}")
    print(report)
    assert (rmsd <= bound).all(), report
    assert len(miss) <= int((sens > RMSD_TOL).sum()), report
    assert np.median(rmsd) <= 5e-6, report


# ---- frame replay (Fig. 4): oracle frames through pfc_energy_forces -------
@pytest.mark.parametrize("k", [0, 2])
def test_frame_replay(pfc, weights, k):
    wl = cfg(k)
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights)
    x, v = wl.pos.astype(np.float64), wl.vel.astype(np.float64)
    done = 0
    for frame in (10, 50, 100):
        out = oracle.step(x, v, wl.species, wl.sys_offsets, weights, wl.dt_fs, frame - done)
        x, v, done = out["pos"], out["vel"], frame
        xf = x.astype(np.float32)                                # the frame as a PDB-like fp32 record
        E, F = p.energy_forces(_dev(pfc, xf))
        _assert_lists_equal(p.neighbors(), oracle.neighbors(xf, wl.sys_offsets))
        ref = oracle.energy_forces(xf.astype(np.float64), wl.species, wl.sys_offsets, weights)
        _check_energy_forces(E, F, ref)
    assert p.status() == 0
    p.close()


# ---- determinism ------------------------------------------------------------------------
def test_bitwise_determinism(pfc, weights):
    wl = W.config4(n_replicas=48)
    outs = []
    for _ in range(2):
        p = pfc.Pfc(wl.species, wl.sys_offsets, weights)
        pos, vel = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
        E, F = p.set_state(pos, vel)
        p.step(25, 0.5)
        torch.cuda.synchronize()
        outs.append((pos.cpu().numpy().copy(), vel.cpu().numpy().copy(), E.cpu().numpy().copy(),
                     F.cpu().numpy().copy()))
        p.close()
    for a, b in zip(*outs):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("what", ["tensor", "cluster"])
def test_repeated_evaluations_are_bit_identical(pfc, weights, what):
    """Stands in for racecheck (compute-sanitizer is closed on this pool, profiles/r2_sanitizer.md): a race in the
    tensor kernel's mbarrier / TMEM pipeline (three warp roles, TMEM columns reused under live readers), in the
    cluster kernel's distributed-shared-memory exchange or in the graph replay shows as a run-to-run difference.
    40 evaluations of one batch, every output identical bit for bit; then a second handle reproduces them."""
    if what == "tensor":
        wl = W.config4(n_replicas=300)                            # 135 tiles + padding on 148 persistent CTAs
        mk = lambda: pfc.Pfc(wl.species, wl.sys_offsets, weights, mlp_path=pfc.MLP_TENSOR)
    else:
        wl = W.config1(n_replicas=8)                              # 12 tiles of 16 rows: the cluster kernel
        mk = lambda: pfc.Pfc(wl.species, wl.sys_offsets, weights, mlp_path=pfc.MLP_FP32, tuning=pfc.Tuning(k3_cluster=2))
    pos = _dev(pfc, wl.pos)
    ref = None
    for handle in range(2):
        p = mk()
        for _ in range(40 if handle == 0 else 3):
            E, F = p.energy_forces(pos)
            torch.cuda.synchronize()
            _, g = p.intermediates()
            out = (E.cpu().numpy().copy(), F.cpu().numpy().copy(), g.copy())
            if ref is None:
                ref = out
            for a, b in zip(out, ref):
                assert np.array_equal(a, b)
        assert p.status() == 0
        p.close()


def test_step_splits_are_equivalent(pfc, weights):
    """pfc_step(60) == pfc_step(25) + pfc_step(35) bit for bit (the state at exit is synchronous)."""
    wl = W.config1(n_replicas=8)
    res = []
    for parts in ((60,), (25, 35)):
        p = pfc.Pfc(wl.species, wl.sys_offsets, weights)
        pos, vel = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
        p.set_state(pos, vel)
        for n in parts:
            p.step(n, 0.5)
        torch.cuda.synchronize()
        res.append(pos.cpu().numpy().copy())
        p.close()
    # the fused kick (dt*a) and two half kicks round differently: equal to fp32 rounding, not bitwise
    assert np.abs(res[0] - res[1]).max() <= 2e-6


# ---- host-buffer entry point ----------------------------------------------------------------
def test_run_host_matches_device_path(pfc, weights):
    wl = W.config1(n_replicas=4)
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights)
    pos, vel = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
    E, F = p.set_state(pos, vel)
    p.step(10, 0.5)
    torch.cuda.synchronize()
    ph = torch.from_numpy(pfc.pack4(wl.pos)).pin_memory()
    vh = torch.from_numpy(pfc.pack4(wl.vel)).pin_memory()
    Eh = torch.empty(wl.n_systems, dtype=torch.float32).pin_memory()
    Fh = torch.empty(wl.n_atoms, 4, dtype=torch.float32).pin_memory()
    p2 = pfc.Pfc(wl.species, wl.sys_offsets, weights)
    p2.run_host(ph, vh, 10, 0.5, Eh, Fh)
    assert np.array_equal(ph.numpy(), pos.cpu().numpy())
    assert np.array_equal(Eh.numpy(), E.cpu().numpy())
    assert np.array_equal(Fh.numpy(), F.cpu().numpy())
    p.close(); p2.close()


def test_run_host_resume_one_force_evaluation_per_call(pfc, weights):
    """The callback regime: state on the host, one step per call, forces carried over by the caller."""
    wl = W.config1(n_replicas=4)
    ph = torch.from_numpy(pfc.pack4(wl.pos)).pin_memory()
    vh = torch.from_numpy(pfc.pack4(wl.vel)).pin_memory()
    Eh = torch.empty(wl.n_systems, dtype=torch.float32).pin_memory()
    Fh = torch.empty(wl.n_atoms, 4, dtype=torch.float32).pin_memory()
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights)
    p.run_host(ph, vh, 0, 0.5, Eh, Fh)                        # forces at the start
    ef, step = p.launch_counts()
    for _ in range(20):
        p.run_host_resume(ph, vh, Fh, 1, 0.5, Eh)
    ref = oracle.step(wl.pos, wl.vel, wl.species, wl.sys_offsets, weights, 0.5, 20)
    x = ph.numpy()[:, :3].astype(np.float64)
    assert _rmsd_per_system(x, ref["pos"], wl.sys_offsets).max() <= RMSD_TOL
    assert np.abs(vh.numpy()[:, :3] - ref["vel"]).max() <= VEL_TOL
    assert np.abs(Fh.numpy()[:, :3] - ref["F"]).max() <= F_ATOL_INTERNAL
    assert np.abs(Eh.numpy() - ref["pe"][-1]).max() <= E_RTOL * np.maximum(np.abs(ref["pe"][-1]), 1.0).max()
    p.close()


# ---- edge and degenerate cases ------------------------------------------------------------
def _eval(pfc, weights, pos, species, off):
    p = pfc.Pfc(species, off, weights)
    E, F = p.energy_forces(_dev(pfc, pos))
    lists = p.neighbors()
    st = p.status()
    ref = oracle.energy_forces(np.asarray(pos, np.float64), species, off, weights)
    p.close()
    return E, F, lists, st, ref


def test_isolated_atoms_and_pairs(pfc, weights):
    """Systems of one atom (empty rows, AEV = 0, E = MLP(0), F = 0), pairs beyond and inside the
    cutoffs, and a pair straddling each cutoff by one fp32 ulp of d2."""
    pos = np.zeros((10, 3), np.float32)
    species = np.array([0, 1, 2, 3, 0, 0, 1, 3, 0, 0], np.int32)
    off = np.array([0, 1, 2, 3, 4, 6, 8, 10], np.int32)
    pos[5] = [6.0, 0, 0]                      # H-H beyond both cutoffs
    pos[7] = [0, 3.0, 0]                      # C-O inside both
    pos[9] = [0, 0, 4.0]                      # H-H radial only
    E, F, lists, st, ref = _eval(pfc, weights, pos, species, off)
    assert st == 0
    _assert_lists_equal(lists, oracle.neighbors(pos, off))
    assert list(np.diff(lists[0])) == [0, 0, 0, 0, 0, 0, 1, 1, 1, 1]
    assert list(np.diff(lists[2])) == [0, 0, 0, 0, 0, 0, 1, 1, 0, 0]
    _check_energy_forces(E, F, ref)
    assert np.abs(F.cpu().numpy()[:6, :3]).max() == 0.0


def test_cutoff_boundary_is_the_fp32_predicate(pfc, weights):
    """d2 == RC2 exactly is excluded, one ulp below is included (S6), for both cutoffs."""
    rc2 = {"r": np.float32(27.04), "a": np.float32(12.25)}
    rows = []
    pos, off = [], [0]
    for key in ("r", "a"):
        for ulps in (-1, 0, 1):
            target = np.nextafter(rc2[key], np.float32(np.inf if ulps > 0 else -np.inf)) if ulps else rc2[key]
            # find an x whose fp32 square is exactly `target` if one exists, else nearest below/above
            x = np.float32(np.sqrt(np.float64(target)))
            pos += [[0, 0, 0], [float(x), 0, 0]]
            off.append(off[-1] + 2)
            rows.append((key, float(np.float32(x) * np.float32(x))))
    pos = np.array(pos, np.float32)
    species = np.zeros(len(pos), np.int32)
    E, F, lists, st, ref = _eval(pfc, weights, pos, species, np.array(off, np.int32))
    _assert_lists_equal(lists, oracle.neighbors(pos, np.array(off, np.int32)))
    nr, na = np.diff(lists[0])[::2], np.diff(lists[2])[::2]
    for (key, d2), r, a in zip(rows, nr, na):
        assert r == int(np.float32(d2) < np.float32(27.04))
        assert a == int(np.float32(d2) < np.float32(12.25))
    _check_energy_forces(E, F, ref)


def test_brute_force_to_cell_list_switch(pfc, weights):
    """2,048 atoms -> brute force, 2,049 -> cell list; both bit-exact against the enumeration."""
    for n in (2048, 2049):
        wl = W.config3(n_atoms=n)
        p = pfc.Pfc(wl.species, wl.sys_offsets, weights)
        E, F = p.energy_forces(_dev(pfc, wl.pos))
        n_launch, _ = p.launch_counts()
        _assert_lists_equal(p.neighbors(), oracle.neighbors(wl.pos, wl.sys_offsets))
        _check_energy_forces(E, F, oracle.energy_forces(wl.pos.astype(np.float64), wl.species,
                                                        wl.sys_offsets, weights))
        assert (n_launch > 6) == (n > 2048)         # cell path: grid, assign, scan, fill, rows
        p.close()


def test_skin_list_reuse_keeps_the_lists_bit_exact(pfc, weights):
    """pfc_tuning_t.skin_list = 1: cell-list systems keep candidate rows (cutoff 5.2 + 0.5 A) and rebuild them only
    when an atom has moved more than 0.25 A since the build; every step the exact predicate runs on the candidates.  The lists must be
    the O(N^2) definition's, bit for bit, at the positions the GPU has reached -- after a stretch of steps that
    reused the candidates, after the export (which invalidates them) and after a jump of all positions."""
    wl = W.config3(n_atoms=5000)
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights, tuning=pfc.Tuning(skin_list=1))
    pos, vel = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
    p.set_state(pos, vel)
    p.step(40, wl.dt_fs)
    torch.cuda.synchronize()
    builds = p.work_counts()["skin_builds"]
    assert 1 <= builds <= 12, builds                            # 41 evaluations, a handful of builds
    _assert_lists_equal(p.neighbors(), oracle.neighbors(pos.cpu().numpy()[:, :3], wl.sys_offsets, cell=False))
    p.step(25, wl.dt_fs)
    torch.cuda.synchronize()
    _assert_lists_equal(p.neighbors(), oracle.neighbors(pos.cpu().numpy()[:, :3], wl.sys_offsets, cell=False))
    # a jump: every atom displaced by up to 0.6 A -> the check must trigger a rebuild
    rng = np.random.default_rng(5)
    moved = (pos.cpu().numpy()[:, :3] + rng.uniform(-0.35, 0.35, size=(wl.n_atoms, 3))).astype(np.float32)
    before = p.work_counts()["skin_builds"]
    p.energy_forces(_dev(pfc, moved))
    torch.cuda.synchronize()
    assert p.work_counts()["skin_builds"] == before + 1
    _assert_lists_equal(p.neighbors(), oracle.neighbors(moved, wl.sys_offsets, cell=False))
    assert p.status() == 0
    p.close()


def test_mixed_batch_of_cell_and_brute_systems(pfc, weights):
    """One handle holding a 2,500-atom cluster (cell list), small molecules and a 1-atom system."""
    big = W.config3(n_atoms=2500)
    small = W.config4(n_replicas=5)
    small.pos[:] += (np.repeat(np.arange(5), np.diff(small.sys_offsets))[:, None] * np.float32(4.0))   # molecules 4 A apart
    pos = np.concatenate([small.pos[:40], big.pos, small.pos[40:], [[0, 0, 0]]]).astype(np.float32)
    species = np.concatenate([small.species[:40], big.species, small.species[40:], [2]]).astype(np.int32)
    # four systems: 40 small-molecule atoms | the cluster | the remaining small atoms | one atom
    off = np.array([0, 40, 40 + 2500, 40 + 2500 + (small.n_atoms - 40), len(pos)], np.int32)
    E, F, lists, st, ref = _eval(pfc, weights, pos, species, off)
    assert st == 0
    _assert_lists_equal(lists, oracle.neighbors(pos, off))
    _check_energy_forces(E, F, ref, tight=False)


def test_dense_cluster_sets_status_bits_and_does_not_fault(pfc, weights):
    """More than PFC_MAX_ANGULAR atoms within 3.5 A of one atom: reported through the status word, not
    silently wrong, and no out-of-bounds access.  The rows (119 <= 128 entries per atom) still fit, so
    all four list arrays stay bit-exact."""
    rng = np.random.Generator(np.random.PCG64(5))
    n = 120
    pos = (rng.random((n, 3)) * 1.6).astype(np.float32)
    species = np.zeros(n, np.int32)
    off = np.array([0, n], np.int32)
    p = pfc.Pfc(species, off, weights)
    p.energy_forces(_dev(pfc, pos))
    st = p.status()
    assert st & 4 and not st & 1
    _assert_lists_equal(p.neighbors(), oracle.neighbors(pos, off))
    p.close()
    # row capacity exceeded as well (199 > 192 entries per atom): flagged, no fault, handle stays usable
    n = 200
    pos = (rng.random((n, 3)) * 1.6).astype(np.float32)
    p = pfc.Pfc(np.zeros(n, np.int32), np.array([0, n], np.int32), weights)
    p.energy_forces(_dev(pfc, pos))
    assert p.status() & 1
    p.close()


def test_bad_arguments_are_rejected(pfc, weights):
    with pytest.raises(pfc.PfcError):
        pfc.Pfc(np.array([0, 4], np.int32), np.array([0, 2], np.int32), weights)       # species 4
    with pytest.raises(pfc.PfcError):
        pfc.Pfc(np.array([0, 1], np.int32), np.array([0, 1, 1, 2], np.int32), weights)  # empty system
    with pytest.raises(pfc.PfcError):
        pfc.Pfc(np.array([0, 1], np.int32), np.array([0, 2], np.int32), weights[:-1])
    p = pfc.Pfc(np.array([0, 1], np.int32), np.array([0, 2], np.int32), weights)
    with pytest.raises(pfc.PfcError):
        p.step(1, 0.5)                                                                    # not bound
    with pytest.raises(pfc.PfcError):
        p.energy_forces(torch.zeros(3, 4, device="cuda"))
    p.close()


def test_nve_energy_conservation_on_gpu(pfc, weights):
    """PAPER.md:75 (Fig. 2): the Hamiltonian is flat over 100 NVE steps.  Here: |H(t)-H(0)| stays
    within 5e-4 eV for config 0 at dt = 0.5 fs, and the GPU H(t) tracks the oracle's."""
    wl = cfg(0)
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights)
    pos, vel = _dev(pfc, wl.pos), _dev(pfc, wl.vel)
    E, F = p.set_state(pos, vel)
    m = W.MASSES_AMU[wl.species]
    H = []
    for _ in range(101):
        p.step(1 if H else 0, 0.5)             # step(0) only evaluates E, F at the bound state
        torch.cuda.synchronize()
        v = vel.cpu().numpy()[:, :3].astype(np.float64)
        ke = (0.5 * m[:, None] * v * v).sum() / W.ACC
        H.append(float(E.cpu().numpy()[0]) + ke)
    ref = oracle.step(wl.pos, wl.vel, wl.species, wl.sys_offsets, weights, 0.5, 100)
    Href = ref["pe"][:, 0] + ref["ke"][:, 0]
    H = np.array(H)
    assert np.abs(H - H[0]).max() < 5e-4
    assert np.abs(H - Href).max() < 2e-5
    p.close()


# ---- every K3 tile variant, on element blocks that end inside a warp's rows / a tile ----------------
@pytest.mark.parametrize("tm,deep", [(0, 0), (16, 0), (16, 1), (32, 0), (32, 1), (64, 0), (128, 0)])
def test_k3_tile_variants_on_ragged_element_blocks(pfc, weights, tm, deep):
    """pfc_create picks one FP32 MLP kernel per batch; pfc_tuning_t.k3_tile_rows / k3_deep_ring / k3_cluster
    force the others (tm = 0: the cluster kernel for single small molecules, 8 CTAs per 16-row tile, which is
    what this 84-atom batch gets by default).  Element counts 1 / 9 / 33 / 41 end inside an 8-row warp
    group, a 16-row and a 32-row tile."""
    rng = np.random.default_rng(20241218)
    counts = [33, 41, 1, 9]                                     # H, C, N, O
    species = np.repeat(np.arange(4, dtype=np.int32), counts)
    rng.shuffle(species)
    n = species.size
    pts = []
    while len(pts) < n:                                          # >= 1.0 A apart in a ball at 0.1 / A^3
        c = rng.normal(size=3); c *= 5.8 * rng.random() ** (1 / 3) / np.linalg.norm(c)
        if all(np.linalg.norm(c - q) >= 1.0 for q in pts):
            pts.append(c)
    pos = np.asarray(pts, dtype=np.float32)
    off = np.array([0, 30, n], dtype=np.int32)                   # two systems
    tuning = pfc.Tuning(k3_cluster=2) if tm == 0 else pfc.Tuning(k3_tile_rows=tm, k3_deep_ring=2 if deep else 1)
    p = pfc.Pfc(species, off, weights, mlp_path=pfc.MLP_FP32, tuning=tuning)
    E, F = p.energy_forces(_dev(pfc, pos))
    torch.cuda.synchronize()
    ref = oracle.energy_forces(pos.astype(np.float64), species, off, weights, want_intermediates=True)
    assert np.abs(p.intermediates()[1] - ref["g"]).max() <= 2e-6
    Eh, Fh = E.cpu().numpy().astype(np.float64), F.cpu().numpy().astype(np.float64)
    assert (np.abs(Eh - ref["E"]) <= E_RTOL * np.maximum(np.abs(ref["E"]), 1.0)).all()
    assert np.abs(Fh[:, :3] - ref["F"]).max() <= F_ATOL_INTERNAL
    assert np.abs(Fh[:, 3] - ref["e"]).max() <= 1e-5 * max(1.0, np.abs(ref["e"]).max())   # per-atom energies
    assert p.status() == 0
    p.close()
