"""ctypes front of oracle/pfc_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

The fp64 CPU definition of the `pfc` hot path (see the header of
pfc_oracle.c for what it follows and how it is pinned).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2412_18271_b200.

All functions take and return numpy arrays; positions are [N,3].
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from ctypes import POINTER, c_double, c_float, c_int, c_int32, c_int64

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pfc_oracle.c")
_LIB = os.path.join(_HERE, "libpfc_oracle.so")

AEV_LEN = 384
MASSES_AMU = np.array([1.008, 12.011, 14.007, 15.999])      # S12
ACC = 9.648533216e-3


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-ffp-contract=off is part of its definition)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
               "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _L():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        pi32, pf, pd = POINTER(c_int32), POINTER(c_float), POINTER(c_double)
        lib.oracle_neighbors.argtypes = [c_int, c_int, pi32, pf, pi32, pi32, c_int64, pi32, pi32, c_int64]
        lib.oracle_neighbors.restype = c_int
        lib.oracle_neighbors_cell.argtypes = [c_int, c_int, pi32, pf, c_double,
                                              pi32, pi32, c_int64, pi32, pi32, c_int64]
        lib.oracle_neighbors_cell.restype = c_int
        lib.oracle_aev.argtypes = [c_int, pd, pi32, pi32, pi32, pi32, pi32, pd]
        lib.oracle_aev.restype = None
        lib.oracle_mlp.argtypes = [c_int, pi32, pd, pf, pd, pd]
        lib.oracle_mlp.restype = None
        lib.oracle_energy_forces.argtypes = [c_int, c_int, pi32, pd, pi32, pf, c_int, pd, pd, pd, pd, pd]
        lib.oracle_energy_forces.restype = c_int
        lib.oracle_step.argtypes = [c_int, c_int, pi32, pd, pd, pi32, pf, pd, c_double, c_int, c_int,
                                    c_int, c_double, c_double, pd, pd, pd]
        lib.oracle_step.restype = c_int
        lib.oracle_dist2_f32.argtypes = [pf, pf]
        lib.oracle_dist2_f32.restype = c_float
        lib.oracle_pair_index.argtypes = [c_int, c_int]
        lib.oracle_pair_index.restype = c_int
        lib.oracle_num_threads.restype = c_int
        lib.oracle_set_num_threads.argtypes = [c_int]
        _lib = lib
    return _lib


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(POINTER(ct))


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def num_threads() -> int:
    return int(_L().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _L().oracle_set_num_threads(int(n))


def dist2_f32(a, b) -> float:
    a = np.ascontiguousarray(a, dtype=np.float32)
    b = np.ascontiguousarray(b, dtype=np.float32)
    return float(_L().oracle_dist2_f32(_p(a, c_float), _p(b, c_float)))


def pair_index(za: int, zb: int) -> int:
    return int(_L().oracle_pair_index(int(za), int(zb)))


def neighbors(pos_f32, sys_offsets, cell: bool = False, cell_edge: float = 5.25):
    """O2.  Returns (r_off, r_idx, a_off, a_idx) int32 CSR, rows ascending."""
    pos = np.ascontiguousarray(pos_f32, dtype=np.float32)
    off = _i32(sys_offsets)
    n, ns = pos.shape[0], off.shape[0] - 1
    r_off = np.zeros(n + 1, np.int32)
    a_off = np.zeros(n + 1, np.int32)
    L = _L()

    def call(r_idx, cr, a_idx, ca):
        if cell:
            return L.oracle_neighbors_cell(n, ns, _p(off, c_int32), _p(pos, c_float), float(cell_edge),
                                           _p(r_off, c_int32), _p(r_idx, c_int32), cr,
                                           _p(a_off, c_int32), _p(a_idx, c_int32), ca)
        return L.oracle_neighbors(n, ns, _p(off, c_int32), _p(pos, c_float),
                                  _p(r_off, c_int32), _p(r_idx, c_int32), cr,
                                  _p(a_off, c_int32), _p(a_idx, c_int32), ca)
    assert call(None, 0, None, 0) == 0
    r_idx = np.zeros(max(int(r_off[-1]), 1), np.int32)
    a_idx = np.zeros(max(int(a_off[-1]), 1), np.int32)
    assert call(r_idx, int(r_off[-1]), a_idx, int(a_off[-1])) == 0
    return r_off, r_idx[: r_off[-1]], a_off, a_idx[: a_off[-1]]


def aev(pos, species, r_off, r_idx, a_off, a_idx):
    """O3/O4 on given lists.  Returns [N,384] fp64."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    spc = _i32(species)
    n = pos.shape[0]
    out = np.zeros((n, AEV_LEN))
    ri = _i32(r_idx) if len(r_idx) else np.zeros(1, np.int32)
    ai = _i32(a_idx) if len(a_idx) else np.zeros(1, np.int32)
    _L().oracle_aev(n, _p(pos, c_double), _p(spc, c_int32), _p(_i32(r_off), c_int32), _p(ri, c_int32),
                    _p(_i32(a_off), c_int32), _p(ai, c_int32), _p(out, c_double))
    return out


def mlp(species, aev_rows, weights):
    """O5.  Returns (e[N], g[N,384]) fp64 for the given AEV rows."""
    spc = _i32(species)
    a = np.ascontiguousarray(aev_rows, dtype=np.float64)
    w = np.ascontiguousarray(weights, dtype=np.float32)
    n = a.shape[0]
    e = np.zeros(n)
    g = np.zeros((n, AEV_LEN))
    _L().oracle_mlp(n, _p(spc, c_int32), _p(a, c_double), _p(w, c_float), _p(e, c_double), _p(g, c_double))
    return e, g


def energy_forces(pos, species, sys_offsets, weights, cell: bool = False, want_intermediates: bool = False):
    """O1-O7.  Returns dict(E[n_sys], F[N,3], e[N]) (+ aev, g if asked)."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    spc, off = _i32(species), _i32(sys_offsets)
    w = np.ascontiguousarray(weights, dtype=np.float32)
    n, ns = pos.shape[0], off.shape[0] - 1
    E = np.zeros(ns)
    F = np.zeros((n, 3))
    e = np.zeros(n)
    av = np.zeros((n, AEV_LEN)) if want_intermediates else None
    g = np.zeros((n, AEV_LEN)) if want_intermediates else None
    rc = _L().oracle_energy_forces(n, ns, _p(off, c_int32), _p(pos, c_double), _p(spc, c_int32),
                                   _p(w, c_float), int(cell), _p(E, c_double), _p(F, c_double),
                                   _p(e, c_double), _p(av, c_double), _p(g, c_double))
    assert rc == 0
    out = {"E": E, "F": F, "e": e}
    if want_intermediates:
        out["aev"], out["g"] = av, g
    return out


def step(pos, vel, species, sys_offsets, weights, dt, n_steps, cell: bool = False,
         masses=None, harmonic=None):
    """O8.  Returns dict(pos, vel, F, pe[(n_steps+1),n_sys], ke[...]).
    harmonic=(k, r0) swaps in the P10 test potential."""
    pos = np.array(pos, dtype=np.float64, order="C", copy=True)
    vel = np.array(vel, dtype=np.float64, order="C", copy=True)
    spc, off = _i32(species), _i32(sys_offsets)
    n, ns = pos.shape[0], off.shape[0] - 1
    m = np.ascontiguousarray(MASSES_AMU if masses is None else masses, dtype=np.float64)
    w = np.ascontiguousarray(weights if weights is not None else np.zeros(1), dtype=np.float32)
    F = np.zeros((n, 3))
    pe = np.zeros((n_steps + 1, ns))
    ke = np.zeros((n_steps + 1, ns))
    kind, k, r0 = (1, float(harmonic[0]), float(harmonic[1])) if harmonic else (0, 0.0, 0.0)
    rc = _L().oracle_step(n, ns, _p(off, c_int32), _p(pos, c_double), _p(vel, c_double), _p(spc, c_int32),
                          _p(w, c_float), _p(m, c_double), float(dt), int(n_steps), int(cell), kind, k, r0,
                          _p(F, c_double), _p(pe, c_double), _p(ke, c_double))
    assert rc == 0
    return {"pos": pos, "vel": vel, "F": F, "pe": pe, "ke": ke}


def philox4x32_10(ctr, key):
    """Philox4x32-10 block (O9 / reading S28): ctr[4], key[2] uint32 -> 4 uint32."""
    from ctypes import c_uint32
    L = _L()
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    L.oracle_philox4x32_10.restype = None
    L.oracle_philox4x32_10(_p(c, c_uint32), _p(k, c_uint32), _p(out, c_uint32))
    return out


def langevin_normals(atom: int, step: int, seed: int):
    """The three standard normals of (atom, step) (O9)."""
    from ctypes import c_uint32, c_uint64
    L = _L()
    xi = np.zeros(3)
    L.oracle_langevin_normals.restype = None
    L.oracle_langevin_normals.argtypes = [c_uint32, c_uint32, c_uint64, ctypes.POINTER(c_double)]
    L.oracle_langevin_normals(int(atom), int(step), int(seed), _p(xi, c_double))
    return xi


def step_langevin(pos, vel, species, sys_offsets, weights, dt, n_steps, gamma, temperature, seed,
                  step0: int = 0, cell: bool = False, masses=None, free: bool = False):
    """O9: n_steps of BAOAB Langevin dynamics.  free=True drops the forces (pins).
    Returns dict(pos, vel, F)."""
    from ctypes import c_uint32, c_uint64
    pos = np.array(pos, dtype=np.float64, order="C", copy=True)
    vel = np.array(vel, dtype=np.float64, order="C", copy=True)
    spc, off = _i32(species), _i32(sys_offsets)
    n, ns = pos.shape[0], off.shape[0] - 1
    m = np.ascontiguousarray(MASSES_AMU if masses is None else masses, dtype=np.float64)
    w = np.ascontiguousarray(weights if weights is not None else np.zeros(1), dtype=np.float32)
    F = np.zeros((n, 3))
    L = _L()
    L.oracle_step_langevin.restype = c_int
    L.oracle_step_langevin.argtypes = [c_int, c_int, ctypes.POINTER(c_int32), ctypes.POINTER(c_double),
                                       ctypes.POINTER(c_double), ctypes.POINTER(c_int32),
                                       ctypes.POINTER(c_float), ctypes.POINTER(c_double), c_double, c_int, c_int,
                                       c_int, c_double, c_double, c_uint64, c_uint32, ctypes.POINTER(c_double)]
    rc = L.oracle_step_langevin(n, ns, _p(off, c_int32), _p(pos, c_double), _p(vel, c_double), _p(spc, c_int32),
                                _p(w, c_float), _p(m, c_double), float(dt), int(n_steps), int(cell),
                                2 if free else 0, float(gamma), float(temperature), int(seed), int(step0),
                                _p(F, c_double))
    assert rc == 0
    return {"pos": pos, "vel": vel, "F": F}
