"""Seeded synthetic inputs for the five workloads of BASELINE.json:configs.

This module is the ONE thing the fp64 oracle's tests and the CUDA path share.
It holds none of the method's arithmetic (no neighbour search, no symmetry
functions, no MLP, no integrator): it only draws positions, velocities,
species and weights.  The recipe is SURVEY.md §8(d) G1-G6 with the readings
S9-S13 and S16; DESIGN.md §"Input recipe" restates it.

Every array is drawn in fp64 from ``numpy.random.Generator(PCG64(seed))`` and
rounded once to fp32; both sides receive the fp32 arrays.

Stand-in statement: the paper's workload (one ethanol molecule, BAMBOO MLFF,
PAPER.md:73) is not reproducible here; these gas-phase systems keep its shape
(isolated molecule/cluster, no periodic box, 300 K Maxwell-Boltzmann start).
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

# -- constants of the input recipe (not of the potential) ---------------------
N_SPECIES = 4                                   # H, C, N, O  (configs[0])
MASSES_AMU = np.array([1.008, 12.011, 14.007, 15.999])        # S12
KB_EV_PER_K = 8.617333262e-5
ACC = 9.648533216e-3                            # (Å/fs²) per (eV/Å/amu)
TEMPERATURE_K = 300.0
WEIGHT_SEED = 2412                              # S9: one potential for all configs
LAYER_DIMS = (384, 160, 128, 96, 1)             # configs[0]
WEIGHTS_PER_ELEMENT = sum(o * i + o for i, o in zip(LAYER_DIMS[:-1], LAYER_DIMS[1:]))
N_WEIGHTS = N_SPECIES * WEIGHTS_PER_ELEMENT     # 378,756
_BLOCK = 64                                     # candidates drawn per RNG call


@dataclass
class Workload:
    """fp32 inputs of one config.  pos/vel are [N,3]; species int32 [N];
    sys_offsets int32 [n_systems+1] (atoms of system s are the contiguous
    range sys_offsets[s]:sys_offsets[s+1])."""
    name: str
    pos: np.ndarray
    vel: np.ndarray
    species: np.ndarray
    sys_offsets: np.ndarray
    dt_fs: float = 0.5
    steps_timed: int = 0

    @property
    def n_atoms(self) -> int:
        return int(self.species.shape[0])

    @property
    def n_systems(self) -> int:
        return int(self.sys_offsets.shape[0] - 1)


def make_weights(seed: int = WEIGHT_SEED) -> np.ndarray:
    """G6 / S9: per element e=0..3, per layer, W[out][in] then b[out], each
    standard_normal * fan_in**-0.5, concatenated (layout SURVEY.md §8c-O5)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    parts = []
    for _e in range(N_SPECIES):
        for fan_in, fan_out in zip(LAYER_DIMS[:-1], LAYER_DIMS[1:]):
            s = fan_in ** -0.5
            parts.append((rng.standard_normal((fan_out, fan_in)) * s).ravel())
            parts.append(rng.standard_normal(fan_out) * s)
    w = np.concatenate(parts).astype(np.float32)
    assert w.shape[0] == N_WEIGHTS
    return w


def _sample_ball(rng, n: int, radius: float, spacing: float) -> np.ndarray:
    """S16 sequential rejection: candidate = R * u^(1/3) * n_hat, accepted iff
    at least `spacing` from every accepted site.  Candidates are drawn
    _BLOCK at a time (normals first, then uniforms) and consumed in order; the
    unused tail of the last block is discarded."""
    pts = np.empty((n, 3))
    k = 0
    s2 = spacing * spacing
    if n > 4096:                      # same accept/reject decisions, O(1) lookup
        return _sample_ball_grid(rng, n, radius, spacing)
    while k < n:
        g = rng.standard_normal((_BLOCK, 3))
        u = rng.random(_BLOCK)
        cand = (radius * np.cbrt(u) / np.sqrt((g * g).sum(1)))[:, None] * g
        for c in cand:
            if k == n:
                break
            if k == 0:
                ok = True
            else:
                d = pts[:k] - c
                ok = (d * d).sum(1).min() >= s2
            if ok:
                pts[k] = c
                k += 1
    return pts


def _sample_ball_grid(rng, n: int, radius: float, spacing: float) -> np.ndarray:
    """_sample_ball with the accepted sites binned on a grid of edge `spacing`
    (27-cell lookup).  Same RNG consumption and the same decisions."""
    pts = np.empty((n, 3))
    k = 0
    s2 = spacing * spacing
    cells: dict = {}
    inv = 1.0 / spacing
    while k < n:
        g = rng.standard_normal((_BLOCK, 3))
        u = rng.random(_BLOCK)
        cand = (radius * np.cbrt(u) / np.sqrt((g * g).sum(1)))[:, None] * g
        keys = np.floor(cand * inv).astype(np.int64)
        for c, key in zip(cand, keys):
            if k == n:
                break
            cx, cy, cz = int(key[0]), int(key[1]), int(key[2])
            ok = True
            for ax in (cx - 1, cx, cx + 1):
                for ay in (cy - 1, cy, cy + 1):
                    for az in (cz - 1, cz, cz + 1):
                        lst = cells.get((ax, ay, az))
                        if lst is None:
                            continue
                        for q in lst:
                            d = pts[q] - c
                            if d[0] * d[0] + d[1] * d[1] + d[2] * d[2] < s2:
                                ok = False
                                break
                        if not ok:
                            break
                    if not ok:
                        break
                if not ok:
                    break
            if ok:
                pts[k] = c
                cells.setdefault((cx, cy, cz), []).append(k)
                k += 1
    return pts


def _velocities(rng, species: np.ndarray) -> np.ndarray:
    """S13: each component ~ N(0, kB*T*ACC/m) in (Å/fs)²; no COM removal,
    no rescaling."""
    sigma = np.sqrt(KB_EV_PER_K * TEMPERATURE_K * ACC / MASSES_AMU)
    return rng.standard_normal((species.shape[0], 3)) * sigma[species][:, None]


def _ball_radius(n: int, density: float) -> float:
    return (3.0 * n / (4.0 * math.pi * density)) ** (1.0 / 3.0)


def _small_molecule(seed: int):
    """configs[0]/[1]: 22 atoms (12 H, 6 C, 2 N, 2 O) permuted, 4 Å ball,
    >= 1.0 Å spacing (S11, S16)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    base = np.array([0] * 12 + [1] * 6 + [2] * 2 + [3] * 2, dtype=np.int32)
    species = base[rng.permutation(22)]
    pos = _sample_ball(rng, 22, 4.0, 1.0)
    vel = _velocities(rng, species)
    return pos, vel, species


def _pack(name, pos_l, vel_l, spc_l, steps) -> Workload:
    sizes = np.array([p.shape[0] for p in pos_l], dtype=np.int64)
    off = np.zeros(len(pos_l) + 1, dtype=np.int32)
    off[1:] = np.cumsum(sizes)
    return Workload(
        name=name,
        pos=np.concatenate(pos_l).astype(np.float32),
        vel=np.concatenate(vel_l).astype(np.float32),
        species=np.concatenate(spc_l).astype(np.int32),
        sys_offsets=off,
        steps_timed=steps,
    )


def config0() -> Workload:
    p, v, s = _small_molecule(0)
    return _pack("cfg0_molecule22", [p], [v], [s], 200)


def config1(n_replicas: int = 256) -> Workload:
    """configs[1]: replica r uses seed r (1..256)."""
    out = [_small_molecule(r) for r in range(1, n_replicas + 1)]
    return _pack("cfg1_256x22", [o[0] for o in out], [o[1] for o in out],
                 [o[2] for o in out], 1000)


def config2(n_mol: int = 500) -> Workload:
    """configs[2]: water-like triples O,H,H; O sites in a ball sized for
    1.0 g/cm³ (29.9146 Å³ per molecule), O-O >= 2.5 Å, O-H 0.96 Å, HOH 104.5°,
    orientation from a uniform unit quaternion; seed 7."""
    rng = np.random.Generator(np.random.PCG64(7))
    radius = (3.0 * n_mol * 29.9146 / (4.0 * math.pi)) ** (1.0 / 3.0)
    sites = _sample_ball(rng, n_mol, radius, 2.5)
    q = rng.standard_normal((n_mol, 4))
    q /= np.sqrt((q * q).sum(1))[:, None]
    w, x, y, z = q.T
    rot = np.empty((n_mol, 3, 3))
    rot[:, 0, 0] = 1 - 2 * (y * y + z * z)
    rot[:, 0, 1] = 2 * (x * y - z * w)
    rot[:, 0, 2] = 2 * (x * z + y * w)
    rot[:, 1, 0] = 2 * (x * y + z * w)
    rot[:, 1, 1] = 1 - 2 * (x * x + z * z)
    rot[:, 1, 2] = 2 * (y * z - x * w)
    rot[:, 2, 0] = 2 * (x * z - y * w)
    rot[:, 2, 1] = 2 * (y * z + x * w)
    rot[:, 2, 2] = 1 - 2 * (x * x + y * y)
    half = math.radians(104.5) / 2.0
    h_local = 0.96 * np.array([[math.sin(half), math.cos(half), 0.0],
                               [-math.sin(half), math.cos(half), 0.0]])
    pos = np.empty((n_mol, 3, 3))
    pos[:, 0] = sites
    pos[:, 1] = sites + rot @ h_local[0]
    pos[:, 2] = sites + rot @ h_local[1]
    pos = pos.reshape(-1, 3)
    species = np.tile(np.array([3, 0, 0], dtype=np.int32), n_mol)
    vel = _velocities(rng, species)
    return _pack("cfg2_water1500", [pos], [vel], [species], 1000)


def config3(n_atoms: int = 20000) -> Workload:
    """configs[3]: droplet, exact composition 50:30:10:10 permuted, ball at
    0.1 atoms/Å³, >= 1.0 Å spacing, seed 11."""
    rng = np.random.Generator(np.random.PCG64(11))
    counts = [n_atoms * 5 // 10, n_atoms * 3 // 10, n_atoms // 10]
    counts.append(n_atoms - sum(counts))
    base = np.repeat(np.arange(4, dtype=np.int32), counts)
    species = base[rng.permutation(n_atoms)]
    pos = _sample_ball(rng, n_atoms, _ball_radius(n_atoms, 0.1), 1.0)
    vel = _velocities(rng, species)
    return _pack("cfg3_droplet20000", [pos], [vel], [species], 500)


def config4(n_replicas: int = 4096) -> Workload:
    """configs[4]: sizes iid U{16..96} from PCG64(13); replica r draws from
    child r of SeedSequence(13).spawn(n); species iid p=(.5,.3,.1,.1)."""
    sizes = np.random.Generator(np.random.PCG64(13)).integers(16, 97, size=4096)[:n_replicas]
    children = np.random.SeedSequence(13).spawn(4096)[:n_replicas]
    cum = np.array([0.5, 0.8, 0.9])
    pos_l, vel_l, spc_l = [], [], []
    for n, child in zip(sizes, children):
        rng = np.random.Generator(np.random.PCG64(child))
        species = np.searchsorted(cum, rng.random(int(n)), side="right").astype(np.int32)
        pos = _sample_ball(rng, int(n), _ball_radius(int(n), 0.1), 1.0)
        vel = _velocities(rng, species)
        pos_l.append(pos); vel_l.append(vel); spc_l.append(species)
    return _pack("cfg4_ragged4096", pos_l, vel_l, spc_l, 1000)


CONFIGS = (config0, config1, config2, config3, config4)


def make_config(k: int, **kw) -> Workload:
    return CONFIGS[k](**kw)
