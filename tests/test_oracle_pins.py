"""Pins of the fp64 oracle (oracle/pfc_oracle.c) against things other than
itself: SURVEY.md §8(c) P1-P7.  CPU only."""
import math
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2412_18271_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    out = []
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].strip()
        if line:
            out.append(line.split())
    return out


def _aev_of(pos, species):
    pos = np.asarray(pos, float)
    lists = oracle.neighbors(pos.astype(np.float32), [0, len(pos)])
    return oracle.aev(pos, species, *lists)


# ---------------------------------------------------------------- O2 predicate
def test_predicate_is_uncontracted_fp32():
    """O2/S6: d2 = fl(fl(fl(dx*dx)+fl(dy*dy))+fl(dz*dz)) with every operation
    rounded to fp32.  numpy float32 scalars round every operation, and are a
    different implementation (not the oracle's C)."""
    rng = np.random.default_rng(1)
    a = (rng.random((20000, 3)) * 40 - 20).astype(np.float32)
    b = (a + rng.normal(size=(20000, 3)) * 3).astype(np.float32)
    d = a - b
    sq = d * d
    want = (sq[:, 0] + sq[:, 1]) + sq[:, 2]
    got = np.array([oracle.dist2_f32(a[i], b[i]) for i in range(2000)], np.float32)
    assert (got == want[:2000]).all()
    # the check has power: an FMA-contracted evaluation differs on some of these pairs
    d64 = d.astype(np.float64)
    fma = (d64[:, 0] * d64[:, 0] + sq[:, 1].astype(np.float64)).astype(np.float32)  # fl(dx*dx + fl(dy*dy))
    fma = (fma + sq[:, 2]).astype(np.float32)
    assert (fma[:2000] != want[:2000]).any()


def test_cutoff_literal_and_straddle():
    """S6: RC2_R = 27.04f = 0x41d851ec (not 5.2f*5.2f); strict '<'.  P7 hand
    example: atoms at 5.1999 / 5.2001 and 3.4999 / 3.5001 from the centre."""
    assert np.float32(27.04).view(np.uint32) == 0x41D851EC
    assert (np.float32(5.2) * np.float32(5.2)).view(np.uint32) != 0x41D851EC
    pos = np.array([[0, 0, 0], [5.1999, 0, 0], [0, 5.2001, 0], [0, 0, 3.4999], [0, 0, -3.5001]], np.float32)
    r_off, r_idx, a_off, a_idx = oracle.neighbors(pos, [0, 5])
    assert list(r_idx[r_off[0]:r_off[1]]) == [1, 3, 4]
    assert list(a_idx[a_off[0]:a_off[1]]) == [3]
    # exactly on the cutoff is excluded (strict): d2 == 12.25 for (3.5,0,0)
    pos = np.array([[0, 0, 0], [3.5, 0, 0]], np.float32)
    r_off, r_idx, a_off, a_idx = oracle.neighbors(pos, [0, 2])
    assert a_off[-1] == 0 and r_off[-1] == 2


def test_no_cross_system_pairs():
    """S22: the search is confined to the atom's own system."""
    pos = np.array([[0, 0, 0], [1, 0, 0], [1.5, 0, 0], [0, 1, 0]], np.float32)
    r_off, r_idx, _, _ = oracle.neighbors(pos, [0, 2, 4])
    rows = [list(r_idx[r_off[i]:r_off[i + 1]]) for i in range(4)]
    assert rows == [[1], [0], [3], [2]]


# ---------------------------------------------------------------- P1 / P2 golden
def test_p1_radial_golden():
    for row in _rows("p1_radial.txt"):
        r, _fc, *vals = map(float, row)
        aev = _aev_of([[0, 0, 0], [r, 0, 0]], [0, 0])
        np.testing.assert_allclose(aev[0, :4], vals, rtol=2e-6)
        np.testing.assert_allclose(aev[1, :4], vals, rtol=2e-6)
        assert np.abs(aev[:, 16:]).max() == 0.0          # only the H radial block is populated


def test_p1_radial_species_blocks():
    """O3: a neighbour of species s fills aev[16 s : 16 s + 16] and nothing else."""
    ref = _aev_of([[0, 0, 0], [1.5, 0, 0]], [0, 0])[0, :16]
    for s in range(4):
        aev = _aev_of([[0, 0, 0], [1.5, 0, 0]], [0, s])
        np.testing.assert_allclose(aev[0, 16 * s:16 * s + 16], ref, rtol=1e-14)
        mask = np.ones(384, bool)
        mask[16 * s:16 * s + 16] = False
        assert np.abs(aev[0, mask]).max() == 0.0


def test_p2_angular_golden():
    for row in _rows("p2_angular.txt"):
        name = row[0]
        vj = list(map(float, row[1:4]))
        vk = list(map(float, row[4:7]))
        aev = _aev_of([[0, 0, 0], vj, vk], [0, 0, 0])
        if name.startswith("ratio"):
            a, bn, bd, val = int(row[7]), int(row[8]), int(row[9]), float(row[10])
            got = aev[0, 64 + 8 * a + bn] / aev[0, 64 + 8 * a + bd]
            np.testing.assert_allclose(got, val, rtol=2e-6)
        else:
            a, b, val = int(row[7]), int(row[8]), float(row[9])
            np.testing.assert_allclose(aev[0, 64 + 8 * a + b], val, rtol=2e-6)


def test_pair_block_order():
    """O4/S23: a triple with leg species (s1,s2) fills block p of the golden table only."""
    for s1, s2, p in (tuple(map(int, r)) for r in _rows("pair_blocks.txt")):
        assert oracle.pair_index(s1, s2) == p and oracle.pair_index(s2, s1) == p
        aev = _aev_of([[0, 0, 0], [1.1, 0, 0], [0, 1.2, 0]], [1, s1, s2])
        ang = aev[0, 64:].reshape(10, 32)
        nz = np.nonzero(np.abs(ang).sum(1))[0]
        assert list(nz) == [p]


# ---------------------------------------------------------------- P5 MLP vs torch
def test_p5_mlp_matches_torch_fp64(weights):
    rng = np.random.default_rng(3)
    n = 12
    x = rng.random((n, 384)) * 0.8
    species = rng.integers(0, 4, n).astype(np.int32)
    e, g = oracle.mlp(species, x, weights)
    alpha = float(np.float32(0.1))
    dims = W.LAYER_DIMS
    per = W.WEIGHTS_PER_ELEMENT
    for i in range(n):
        w = torch.tensor(weights[species[i] * per:(species[i] + 1) * per], dtype=torch.float64)
        xi = torch.tensor(x[i], requires_grad=True)
        h, o = xi, 0
        for li, (fi, fo) in enumerate(zip(dims[:-1], dims[1:])):
            Wm = w[o:o + fo * fi].reshape(fo, fi); o += fo * fi
            b = w[o:o + fo]; o += fo
            h = Wm @ h + b
            if li < 3:
                h = torch.nn.functional.celu(h, alpha=alpha)
        (gi,) = torch.autograd.grad(h[0], xi)
        assert abs(h.item() - e[i]) < 1e-12 * max(1, abs(e[i]))
        np.testing.assert_allclose(g[i], gi.numpy(), rtol=0, atol=1e-12)


def test_p5_celu_values_and_zero_weights():
    """CELU(-0.1)=-0.0632120559, CELU(-0.05)=-0.0393469340 (alpha=0.1); with
    all-zero weights and b4=c the energy is c per atom."""
    per = W.WEIGHTS_PER_ELEMENT
    w = np.zeros(4 * per, np.float32)
    # make layer 1 the identity on the first input with bias 0, chain to output: e = celu(celu(celu(x)))
    w[0] = 1.0                                            # W1[0][0]
    o2 = 160 * 384 + 160
    w[o2] = 1.0                                           # W2[0][0]
    o3 = o2 + 128 * 160 + 128
    w[o3] = 1.0                                           # W3[0][0]
    o4 = o3 + 96 * 128 + 96
    w[o4] = 1.0                                           # W4[0][0]
    w[o4 + 96] = 0.25                                     # b4
    x = np.zeros((2, 384)); x[0, 0] = -0.1; x[1, 0] = 0.7
    e, g = oracle.mlp([0, 0], x, w)
    a = float(np.float32(0.1))
    c1 = a * math.expm1(-0.1 / a)
    assert abs(c1 - (-0.0632120559)) < 1e-8               # golden CELU(-0.1) up to alpha=0.1f
    c3 = a * math.expm1(a * math.expm1(c1 / a) / a)
    assert abs(e[0] - (c3 + 0.25)) < 1e-14
    assert abs(e[1] - 0.95) < 1e-14 and abs(g[1, 0] - 1.0) < 1e-14
    w[:] = 0; w[o4 + 96] = 0.25
    e, g = oracle.mlp([0, 0], x, w)
    assert (e == 0.25).all() and (g == 0).all()


# ---------------------------------------------------------------- P6 independent torch autograd
_PAIR = torch.tensor([[0, 1, 2, 3], [1, 4, 5, 6], [2, 5, 7, 8], [3, 6, 8, 9]])   # golden/pair_blocks.txt


def torch_energy(pos32, species, weights):
    """The potential re-derived as vectorised torch.float64 ops (dense N^3
    tensors), forces by autograd.  Test-only; shares nothing with the C file."""
    x32 = torch.tensor(np.asarray(pos32, np.float32))
    d32 = x32[:, None, :] - x32[None, :, :]
    sq = d32 * d32
    d2 = (sq[..., 0] + sq[..., 1]) + sq[..., 2]           # fp32, each op rounded
    n = x32.shape[0]
    eye = torch.eye(n, dtype=torch.bool)
    mr = (d2 < torch.tensor(27.04, dtype=torch.float32)) & ~eye
    ma = (d2 < torch.tensor(12.25, dtype=torch.float32)) & ~eye
    x = x32.double().requires_grad_(True)
    f32 = lambda v: torch.tensor(np.asarray(v, np.float32)).double()
    spc = torch.tensor(np.asarray(species, np.int64))
    v = x[None, :, :] - x[:, None, :]                      # v[i,j] = x_j - x_i
    r = torch.sqrt((v * v).sum(-1) + eye.double())         # avoid sqrt(0) grad on the diagonal
    rc_r, rc_a = f32(5.2), f32(3.5)
    fc_r = 0.5 * torch.cos(math.pi * r / rc_r) + 0.5
    shf_r = f32([0.9, 1.16875, 1.4375, 1.70625, 1.975, 2.24375, 2.5125, 2.78125,
                 3.05, 3.31875, 3.5875, 3.85625, 4.125, 4.39375, 4.6625, 4.93125])
    rad_terms = 0.25 * torch.exp(-16.0 * (r[..., None] - shf_r) ** 2) * fc_r[..., None] * mr[..., None]
    onehot = torch.nn.functional.one_hot(spc, 4).double()  # [N,4]
    radial = torch.einsum("ijk,js->isk", rad_terms, onehot).reshape(n, 64)
    # angular
    fc_a = 0.5 * torch.cos(math.pi * r / rc_a) + 0.5
    u = v / r[..., None]
    cosphi = torch.einsum("ijc,ikc->ijk", u, u)
    theta = torch.acos(f32(0.95) * cosphi)
    rbar = 0.5 * (r[:, :, None] + r[:, None, :])
    shf_a = f32([0.9, 1.55, 2.2, 2.85])
    shf_z = f32([0.19634954, 0.58904862, 0.98174770, 1.37444679, 1.76714587, 2.15984495, 2.55254403, 2.94524311])
    A = ((1 + torch.cos(theta[..., None] - shf_z)) / 2) ** 32                 # [N,N,N,8]
    B = torch.exp(-8.0 * (rbar[..., None] - shf_a) ** 2)                      # [N,N,N,4]
    jj, kk = torch.meshgrid(torch.arange(n), torch.arange(n), indexing="ij")
    tri = (jj < kk)[None] & ma[:, :, None] & ma[:, None, :]
    wgt = 2.0 * fc_a[:, :, None] * fc_a[:, None, :] * tri
    terms = wgt[..., None, None] * B[..., :, None] * A[..., None, :]          # [N,N,N,4,8]
    p = _PAIR[spc[:, None], spc[None, :]]                                      # [N,N]
    ph = torch.nn.functional.one_hot(p, 10).double()                           # [N,N,10]
    angular = torch.einsum("ijkab,jkp->ipab", terms, ph).reshape(n, 320)
    aev = torch.cat([radial, angular], 1)
    alpha = float(np.float32(0.1))
    per = W.WEIGHTS_PER_ELEMENT
    E = 0.0
    for i in range(n):
        w = torch.tensor(weights[int(spc[i]) * per:(int(spc[i]) + 1) * per], dtype=torch.float64)
        h, o = aev[i], 0
        for li, (fi, fo) in enumerate(zip(W.LAYER_DIMS[:-1], W.LAYER_DIMS[1:])):
            Wm = w[o:o + fo * fi].reshape(fo, fi); o += fo * fi
            b = w[o:o + fo]; o += fo
            h = Wm @ h + b
            if li < 3:
                h = torch.nn.functional.celu(h, alpha=alpha)
        E = E + h[0]
    (grad,) = torch.autograd.grad(E, x)
    return float(E.detach()), -grad.numpy(), aev.detach().numpy()


@pytest.mark.parametrize("case", ["cfg0", "cfg4_small", "water"])
def test_p6_independent_torch_autograd(case, weights):
    if case == "cfg0":
        c = W.config0()
        pos, spc = c.pos, c.species
    elif case == "cfg4_small":
        c = W.config4(n_replicas=3)
        s = int(np.argmin(np.diff(c.sys_offsets)))
        sl = slice(c.sys_offsets[s], c.sys_offsets[s + 1])
        pos, spc = c.pos[sl], c.species[sl]
    else:
        c = W.config2(n_mol=12)
        pos, spc = c.pos, c.species
    out = oracle.energy_forces(pos, spc, [0, len(spc)], weights, want_intermediates=True)
    E, F, aev = torch_energy(pos, spc, weights)
    np.testing.assert_allclose(out["aev"], aev, rtol=0, atol=1e-12)
    assert abs(out["E"][0] - E) <= 1e-10 * max(1.0, abs(E))
    np.testing.assert_allclose(out["F"], F, rtol=0, atol=1e-9)


# ---------------------------------------------------------------- P3 finite differences
def _fd_check(pos, spc, off, weights, atoms, h=1e-4):
    pos = np.asarray(pos, np.float64)
    base = oracle.energy_forces(pos, spc, off, weights)
    fmax = np.abs(base["F"]).max()
    worst = 0.0
    for i in atoms:
        for c in range(3):
            e = []
            for k in (-2, -1, 1, 2):
                p = pos.copy(); p[i, c] += k * h
                e.append(oracle.energy_forces(p, spc, off, weights)["E"].sum())
            dEdx = (e[0] - 8 * e[1] + 8 * e[2] - e[3]) / (12 * h)
            worst = max(worst, abs(base["F"][i, c] + dEdx))
    return worst / fmax


def test_p3_forces_are_minus_gradient_cfg0(weights):
    c = W.config0()
    assert _fd_check(c.pos, c.species, c.sys_offsets, weights, range(22)) <= 1e-6


def test_p3_forces_are_minus_gradient_water_and_ragged(weights):
    c = W.config2(n_mol=60)
    assert _fd_check(c.pos, c.species, c.sys_offsets, weights, [0, 1, 2, 91, 179]) <= 1e-6
    c = W.config4(n_replicas=24)
    s = int(np.argmax(np.diff(c.sys_offsets)))
    sl = slice(c.sys_offsets[s], c.sys_offsets[s + 1])
    n = sl.stop - sl.start
    assert _fd_check(c.pos[sl], c.species[sl], [0, n], weights, [0, n // 2, n - 1]) <= 1e-6


# ---------------------------------------------------------------- P4 invariances
def _rot(rng):
    q = rng.normal(size=4); q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def test_p4_invariances(weights):
    """E invariant under translation / rotation / within-element permutation;
    forces co-rotate; sum F = 0 and sum x cross F = 0.  The cutoff predicate is
    fp32, so transformed copies must not move a pair across a cutoff: checked by
    comparing list sizes."""
    rng = np.random.default_rng(5)
    c = W.config0()
    pos = c.pos.astype(np.float64)
    off = c.sys_offsets
    base = oracle.energy_forces(pos, c.species, off, weights)
    n_pairs = oracle.neighbors(c.pos, off)[0][-1]
    E0, F0 = base["E"][0], base["F"]
    assert np.abs(F0.sum(0)).max() < 1e-10
    assert np.abs(np.cross(pos, F0).sum(0)).max() < 1e-10
    tol = 1e-10 * max(1.0, abs(E0))
    t = oracle.energy_forces(pos + np.array([0.3, -1.7, 2.2]), c.species, off, weights)
    R = _rot(rng)
    r = oracle.energy_forces(pos @ R.T, c.species, off, weights)
    for arr in (pos + np.array([0.3, -1.7, 2.2]), pos @ R.T):
        assert oracle.neighbors(arr.astype(np.float32), off)[0][-1] == n_pairs
    assert abs(t["E"][0] - E0) < tol and np.abs(t["F"] - F0).max() < 1e-9
    assert abs(r["E"][0] - E0) < tol and np.abs(r["F"] - F0 @ R.T).max() < 1e-9
    perm = np.arange(22)
    for s in range(4):
        idx = np.nonzero(c.species == s)[0]
        perm[idx] = rng.permutation(idx)
    assert (c.species[perm] == c.species).all() and (perm != np.arange(22)).any()
    p = oracle.energy_forces(pos[perm], c.species, off, weights)
    assert abs(p["E"][0] - E0) < tol and np.abs(p["F"] - F0[perm]).max() < 1e-9


# ---------------------------------------------------------------- P7 neighbour lists
def _brute_numpy(pos32, off):
    """Independent O(N^2) enumeration with numpy float32 ops."""
    rows_r, rows_a = [], []
    for s in range(len(off) - 1):
        x = pos32[off[s]:off[s + 1]]
        d = x[:, None, :] - x[None, :, :]
        sq = d * d
        d2 = (sq[..., 0] + sq[..., 1]) + sq[..., 2]
        np.fill_diagonal(d2, np.inf)
        for i in range(x.shape[0]):
            rows_r.append(np.nonzero(d2[i] < np.float32(27.04))[0] + off[s])
            rows_a.append(np.nonzero(d2[i] < np.float32(12.25))[0] + off[s])
    return rows_r, rows_a


def _check_lists(lists, rows_r, rows_a):
    r_off, r_idx, a_off, a_idx = lists
    assert r_off[-1] == sum(map(len, rows_r)) and a_off[-1] == sum(map(len, rows_a))
    for i in range(len(rows_r)):
        assert (r_idx[r_off[i]:r_off[i + 1]] == rows_r[i]).all()
        assert (a_idx[a_off[i]:a_off[i + 1]] == rows_a[i]).all()


def test_p7_brute_force_matches_numpy_and_cell():
    for c in (W.config0(), W.config1(n_replicas=8), W.config2(), W.config4(n_replicas=40)):
        rows_r, rows_a = _brute_numpy(c.pos, c.sys_offsets)
        lists = oracle.neighbors(c.pos, c.sys_offsets)
        _check_lists(lists, rows_r, rows_a)
        cell = oracle.neighbors(c.pos, c.sys_offsets, cell=True)
        for a, b in zip(lists, cell):
            assert (a == b).all()
        # symmetry, sortedness, NL_A subset of NL_R
        r_off, r_idx, a_off, a_idx = lists
        pairs = set()
        for i in range(c.n_atoms):
            row = r_idx[r_off[i]:r_off[i + 1]]
            assert (np.diff(row) > 0).all()
            pairs.update((i, int(j)) for j in row)
            assert set(a_idx[a_off[i]:a_off[i + 1]]) <= set(row)
        assert all((j, i) in pairs for (i, j) in pairs)


def test_p7_cell_list_equals_enumeration_cfg3_and_shifted_copies():
    c = W.config3()
    brute = oracle.neighbors(c.pos, c.sys_offsets)
    cell = oracle.neighbors(c.pos, c.sys_offsets, cell=True)
    for a, b in zip(brute, cell):
        assert (a == b).all()
    # mean row lengths near the uniform-ball estimates of SURVEY.md §8 (54.1 / 17.0), hard-core excluded
    assert abs(brute[0][-1] / c.n_atoms - 54.1) < 3.0
    assert abs(brute[2][-1] / c.n_atoms - 17.0) < 1.5
    rng = np.random.default_rng(9)
    c0 = W.config0()
    for _ in range(200):
        x = (c0.pos.astype(np.float64) @ _rot(rng).T + rng.normal(size=3) * 30).astype(np.float32)
        a = oracle.neighbors(x, c0.sys_offsets)
        b = oracle.neighbors(x, c0.sys_offsets, cell=True, cell_edge=5.2 * (1 + 2.0 ** -16))
        assert all((p == q).all() for p, q in zip(a, b))
