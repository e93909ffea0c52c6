"""The seeded input recipe: shapes, composition,
spacing, determinism."""
import numpy as np

from paper_2412_18271_b200 import workloads as W


def _min_dist(pos):
    d = pos[:, None, :].astype(np.float64) - pos[None, :, :]
    d2 = (d * d).sum(-1)
    np.fill_diagonal(d2, np.inf)
    return np.sqrt(d2.min())


def test_config0_and_1():
    c = W.config0()
    assert c.n_atoms == 22 and c.n_systems == 1
    assert [int((c.species == s).sum()) for s in range(4)] == [12, 6, 2, 2]
    assert _min_dist(c.pos) >= 1.0 - 1e-6 and np.linalg.norm(c.pos, axis=1).max() <= 4.0 + 1e-5
    c1 = W.config1(n_replicas=6)
    assert c1.n_atoms == 132 and list(c1.sys_offsets) == [0, 22, 44, 66, 88, 110, 132]
    for s in range(6):
        sl = slice(22 * s, 22 * s + 22)
        assert [int((c1.species[sl] == k).sum()) for k in range(4)] == [12, 6, 2, 2]
        assert _min_dist(c1.pos[sl]) >= 1.0 - 1e-6
    assert not np.allclose(c1.pos[:22], c1.pos[22:44])
    again = W.config1(n_replicas=6)
    assert (again.pos == c1.pos).all() and (again.vel == c1.vel).all()
    assert c1.pos.dtype == np.float32 and c1.vel.dtype == np.float32 and c1.species.dtype == np.int32


def test_config2_geometry():
    c = W.config2()
    assert c.n_atoms == 1500 and list(c.species[:3]) == [3, 0, 0]
    o, h1, h2 = c.pos[0::3].astype(np.float64), c.pos[1::3].astype(np.float64), c.pos[2::3].astype(np.float64)
    np.testing.assert_allclose(np.linalg.norm(h1 - o, axis=1), 0.96, atol=1e-5)
    np.testing.assert_allclose(np.linalg.norm(h2 - o, axis=1), 0.96, atol=1e-5)
    cosang = ((h1 - o) * (h2 - o)).sum(1) / 0.96 ** 2
    np.testing.assert_allclose(np.degrees(np.arccos(cosang)), 104.5, atol=1e-3)
    assert _min_dist(o) >= 2.5 - 1e-5


def test_config3_and_4_shapes():
    c = W.config3()
    assert c.n_atoms == 20000
    assert [int((c.species == s).sum()) for s in range(4)] == [10000, 6000, 2000, 2000]
    r = np.linalg.norm(c.pos, axis=1).max()
    assert 36.0 < r <= 36.279
    c4 = W.config4(n_replicas=64)
    sizes = np.diff(c4.sys_offsets)
    assert sizes.min() >= 16 and sizes.max() <= 96
    full_sizes = np.random.Generator(np.random.PCG64(13)).integers(16, 97, size=4096)
    assert (sizes == full_sizes[:64]).all()
    for s in range(0, 64, 7):
        sl = slice(c4.sys_offsets[s], c4.sys_offsets[s + 1])
        assert _min_dist(c4.pos[sl]) >= 1.0 - 1e-6


def test_velocities_are_300K():
    """S13: <m v^2>/ACC = kB T per component (no rescaling, so statistical)."""
    c = W.config3()
    v = c.vel.astype(np.float64)
    kt = (W.MASSES_AMU[c.species][:, None] * v * v / W.ACC).mean()
    assert abs(kt / (W.KB_EV_PER_K * 300.0) - 1) < 0.02


def test_weights_layout():
    w = W.make_weights()
    assert w.shape == (378756,) and w.dtype == np.float32
    per = W.WEIGHTS_PER_ELEMENT
    assert per == 94689
    w1 = w[:160 * 384]
    assert abs(w1.std() - 384 ** -0.5) < 0.02 * 384 ** -0.5
    assert not np.allclose(w[:per], w[per:2 * per])
