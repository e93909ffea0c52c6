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
