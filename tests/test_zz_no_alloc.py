"""pfc_neighbor_offsets_noalloc (include/pfc_noalloc.h): the one entry point whose scratch is a static device
array inside libpfc.so -- no cudaMalloc in the call, no byte of the caller's workspace touched.  Its output is
compared with the existing path's (the r_off / a_off arrays of pfc_get_neighbors, whose block totals sit in the
workspace) at the tolerance the list tests use: bit-exact int32.  Calls in a row share the scratch and must not
see each other's leftovers.  Collected last (pytest -x): a failure here hides no other test.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_2412_18271_b200 import workloads as W                 # noqa: E402


@pytest.fixture(scope="module")
def pfc():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2412_18271_b200 import pfc as m
    m.load_library()
    return m


def _dev(pfc, a3):
    return torch.from_numpy(pfc.pack4(a3)).cuda()


def _handle(pfc, wl, weights):
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights)
    p.energy_forces(_dev(pfc, wl.pos))
    torch.cuda.synchronize()
    assert p.status() == 0
    return p


def _offsets_both_ways(p):
    """(new entry point, existing path): the new one first, so the reference export cannot have helped it."""
    r_off, a_off = p.neighbor_offsets_noalloc()
    torch.cuda.synchronize()
    got = (r_off.cpu().numpy(), a_off.cpu().numpy())
    ref = p.neighbors()
    return got, (ref[0], ref[2])


def test_offsets_match_the_existing_path_on_calls_in_a_row(pfc, weights):
    # three batches with different numbers of 2,048-atom scan blocks (10 blocks of them holding a cell-list
    # system, 3 blocks, 1 block): a later call with fewer blocks finds the earlier call's totals in the scratch
    big = _handle(pfc, W.make_config(3), weights)                 # 20,000 atoms, one cell-list system: 10 blocks
    mid = _handle(pfc, W.make_config(1), weights)               # 5,632 atoms in 256 systems
    one = _handle(pfc, W.make_config(0), weights)               # 22 atoms: the totals kernel does not run at all
    for p in (big, mid, one, mid, big):
        got, ref = _offsets_both_ways(p)
        for g, r in zip(got, ref):
            assert g.dtype == np.int32 and g.shape == r.shape == (p.n_atoms + 1,)
            assert np.array_equal(g, r)
        assert got[0][0] == 0 and got[0][-1] > 0
    # two calls in a row on one handle into fresh outputs: identical, and again equal to the existing path
    first = [t.clone() for t in mid.neighbor_offsets_noalloc()]
    second = mid.neighbor_offsets_noalloc()
    torch.cuda.synchronize()
    ref = mid.neighbors()
    for a, b, r in zip(first, second, (ref[0], ref[2])):
        assert torch.equal(a, b) and np.array_equal(b.cpu().numpy(), r)
    # caller-owned outputs on a side stream, ordered behind the evaluation by the caller
    s = torch.cuda.Stream()
    r_off = torch.full((big.n_atoms + 1,), -1, dtype=torch.int32, device="cuda")
    a_off = torch.full((big.n_atoms + 1,), -1, dtype=torch.int32, device="cuda")
    s.wait_stream(torch.cuda.current_stream())
    big.neighbor_offsets_noalloc(r_off, a_off, stream=s)
    s.synchronize()
    ref = big.neighbors()
    assert np.array_equal(r_off.cpu().numpy(), ref[0]) and np.array_equal(a_off.cpu().numpy(), ref[2])
    for p in (big, mid, one):
        p.close()


def test_the_workspace_is_left_untouched(pfc, weights):
    """With pfc_tuning_t.skin_list = 1 the export block of the workspace holds the candidate rows: pfc_get_neighbors
    overwrites them (and has them rebuilt), the static-scratch entry point does not."""
    wl = W.config3(n_atoms=5000)
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights, tuning=pfc.Tuning(skin_list=1))
    pos = _dev(pfc, wl.pos)
    p.energy_forces(pos)
    torch.cuda.synchronize()
    builds = p.work_counts()["skin_builds"]
    for _ in range(3):
        p.neighbor_offsets_noalloc()
        p.energy_forces(pos)
    torch.cuda.synchronize()
    assert p.work_counts()["skin_builds"] == builds              # candidates still valid: nothing was rebuilt
    got, ref = _offsets_both_ways(p)
    assert np.array_equal(got[0], ref[0]) and np.array_equal(got[1], ref[1])
    p.energy_forces(pos)
    torch.cuda.synchronize()
    assert p.work_counts()["skin_builds"] == builds + 1          # the existing export did cost a rebuild
    p.close()


def test_bad_arguments_and_the_size_limit(pfc, weights):
    wl = W.make_config(0)
    p = _handle(pfc, wl, weights)
    lib = pfc.load_library()
    out = torch.empty(wl.n_atoms + 1, dtype=torch.int32, device="cuda")
    assert lib.pfc_neighbor_offsets_noalloc(None, out.data_ptr(), out.data_ptr(), None) == -1
    assert lib.pfc_neighbor_offsets_noalloc(p._h, None, out.data_ptr(), None) == -1
    p.close()
    assert b"PFC_NOALLOC_MAX_ATOMS" in lib.pfc_error_string(pfc.ERR_TOO_LARGE)
    # one atom more than the static scratch covers: rejected with its own error code, nothing enqueued.
    # (single-atom systems: creating the handle needs an 11 GB workspace and no neighbour work)
    n = pfc.NOALLOC_MAX_ATOMS + 1
    need = pfc.pfc_workspace_bytes(n, n)
    free, _ = torch.cuda.mem_get_info()
    if free < need + (8 << 30):
        pytest.skip(f"{need / 1e9:.1f} GB workspace for the size-limit case does not fit ({free / 1e9:.1f} GB free)")
    species = np.zeros(n, dtype=np.int32)
    off = np.arange(n + 1, dtype=np.int32)
    q = pfc.Pfc(species, off, weights, mlp_path=pfc.MLP_FP32)
    big_out = torch.empty(n + 1, dtype=torch.int32, device="cuda")
    rc = lib.pfc_neighbor_offsets_noalloc(q._h, big_out.data_ptr(), big_out.data_ptr(), None)
    assert rc == pfc.ERR_TOO_LARGE
    with pytest.raises(pfc.PfcError, match="PFC_NOALLOC_MAX_ATOMS"):
        q.neighbor_offsets_noalloc(big_out, big_out.clone())
    q.close()
    del q, big_out
    torch.cuda.empty_cache()
