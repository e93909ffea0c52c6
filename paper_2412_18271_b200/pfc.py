"""ctypes binding of libpfc.so (include/pfc.h) -- argument marshalling only.

Every step of the path (neighbour build, AEV, MLP, force chain rule,
velocity-Verlet, graph replay) runs inside the library's CUDA kernels; this
module owns no arithmetic.  PyTorch supplies device memory (the workspace and
all state tensors) and the stream.  There is no CPU fallback: importing this
module without a built libpfc.so, or creating a handle without a CUDA device,
raises.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_char_p, c_float, c_int, c_int32, c_size_t, c_uint32, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpfc.so")

AEV_LEN = 384
N_WEIGHTS = 378756
MLP_FP32 = 0
MLP_TENSOR = 1
MLP_TENSOR_1TERM = 2      # plain fp16 operands: tolerance evidence only
MLP_AUTO = 3              # MLP_TENSOR from 1024 atoms on, FP32 below

STATUS_BITS = {1: "radial capacity overflow", 2: "angular capacity overflow",
               4: "angular row longer than PFC_MAX_ANGULAR", 8: "non-finite energy",
               16: "cell grid overflow"}

N_STAGES = 7
STAGE_NAMES = ("K1_neighbors", "K2_aev_fwd", "K3_mlp", "K4a_aev_bwd", "K4b_gather", "energy_sum", "K5_integrate")

# include/pfc.h (the provider boundary) and include/pfc_debug.h (measurement / parity helpers)
EXPORTS = ("pfc_workspace_bytes", "pfc_create", "pfc_energy_forces", "pfc_energy_forces_nm", "pfc_set_state",
           "pfc_step", "pfc_step_langevin", "pfc_set_frames", "pfc_frames_written", "pfc_run_host",
           "pfc_run_host_resume", "pfc_get_neighbors", "pfc_get_intermediates", "pfc_status", "pfc_destroy",
           "pfc_error_string")
DEBUG_EXPORTS = ("pfc_profile_stages", "pfc_work_counts", "pfc_k3_timeline", "pfc_copy_to_host", "pfc_mlp_path", "pfc_launch_counts", "pfc_tc_calibration", "pfc_tc_chain_probe")


NOALLOC_EXPORTS = ("pfc_neighbor_offsets_noalloc",)        # include/pfc_noalloc.h
NOALLOC_MAX_ATOMS = 1048576
ERR_TOO_LARGE = -7


class PfcError(RuntimeError):
    pass


class Tuning(ctypes.Structure):
    """pfc_tuning_t (include/pfc.h): a zero-filled struct is "all defaults"."""
    _fields_ = [("k3_tile_rows", c_int32), ("k3_deep_ring", c_int32), ("tc_comp_override", c_int32),
                ("tc_comp_forward", c_float), ("tc_comp_backward", c_float), ("steps_per_graph", c_int32),
                ("k3_cluster", c_int32), ("skin_list", c_int32)]


class _Desc(ctypes.Structure):
    _fields_ = [("n_atoms", c_int32), ("n_systems", c_int32),
                ("species", POINTER(c_int32)), ("sys_offsets", POINTER(c_int32)),
                ("weights", POINTER(c_float)), ("masses_amu", POINTER(c_float)),
                ("workspace", c_void_p), ("workspace_bytes", c_size_t),
                ("mlp_path", c_int32), ("tuning", POINTER(Tuning))]


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libpfc.so and declare the prototypes of include/pfc.h.  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise PfcError(f"{LIB_PATH} is missing: build it with `python -m paper_2412_18271_b200.build` "
                       "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    pp_i32 = POINTER(POINTER(c_int32))
    pp_f = POINTER(POINTER(c_float))
    lib.pfc_workspace_bytes.argtypes = [c_int32, c_int32]
    lib.pfc_workspace_bytes.restype = c_size_t
    lib.pfc_create.argtypes = [POINTER(_Desc), POINTER(c_void_p)]
    lib.pfc_energy_forces.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]
    lib.pfc_energy_forces_nm.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]
    lib.pfc_profile_stages.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, POINTER(c_float)]
    lib.pfc_set_state.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]
    lib.pfc_step.argtypes = [c_void_p, c_int32, c_float]
    lib.pfc_step_langevin.argtypes = [c_void_p, c_int32, c_float, c_float, c_float, ctypes.c_uint64]
    lib.pfc_set_frames.argtypes = [c_void_p, c_void_p, c_int32, c_int32]
    lib.pfc_frames_written.argtypes = [c_void_p, POINTER(c_int32)]
    lib.pfc_run_host.argtypes = [c_void_p, c_void_p, c_void_p, c_int32, c_float, c_void_p, c_void_p, c_void_p]
    lib.pfc_run_host_resume.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_int32, c_float, c_void_p, c_void_p]
    lib.pfc_get_neighbors.argtypes = [c_void_p, pp_i32, pp_i32, pp_i32, pp_i32]
    lib.pfc_work_counts.argtypes = [c_void_p, POINTER(ctypes.c_int64)]
    lib.pfc_k3_timeline.argtypes = [c_void_p, POINTER(ctypes.c_int64), c_int32]
    lib.pfc_get_intermediates.argtypes = [c_void_p, pp_f, pp_f, pp_i32, POINTER(c_int32)]
    lib.pfc_copy_to_host.argtypes = [c_void_p, c_void_p, c_size_t]
    lib.pfc_status.argtypes = [c_void_p, POINTER(c_uint32)]
    lib.pfc_mlp_path.argtypes = [c_void_p, POINTER(c_int32)]
    lib.pfc_tc_calibration.argtypes = [c_void_p, POINTER(c_float)]
    lib.pfc_tc_chain_probe.argtypes = [c_void_p, c_void_p, c_int32, c_int32, c_void_p, c_void_p]
    lib.pfc_launch_counts.argtypes = [c_void_p, POINTER(c_int32), POINTER(c_int32), POINTER(c_int32)]
    lib.pfc_destroy.argtypes = [c_void_p]
    lib.pfc_neighbor_offsets_noalloc.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p]
    lib.pfc_neighbor_offsets_noalloc.restype = c_int
    lib.pfc_error_string.argtypes = [c_int]
    lib.pfc_error_string.restype = c_char_p
    for name in EXPORTS + DEBUG_EXPORTS:
        if name not in ("pfc_workspace_bytes", "pfc_error_string"):
            getattr(lib, name).restype = c_int
    _lib = lib
    return lib


def _check(rc: int, what: str) -> None:
    if rc != 0:
        raise PfcError(f"{what}: {load_library().pfc_error_string(rc).decode()} ({rc})")


def tc_chain_probe(A, B, n_mma: int, stream=None):
    """pfc_tc_chain_probe: cuda float32 tensors A [128, 16 s], B [64, 16 s] (fp16-representable values) -> raw
    accumulator [128, 64] of a chain of n_mma tcgen05.mma kind::f16 instructions cycling through the s slices."""
    import torch
    assert A.is_cuda and B.is_cuda and A.dtype == torch.float32 and B.dtype == torch.float32
    assert A.shape[0] == 128 and B.shape[0] == 64 and A.shape[1] == B.shape[1] and A.shape[1] % 16 == 0
    A, B = A.contiguous(), B.contiguous()
    D = torch.empty(128, 64, dtype=torch.float32, device=A.device)
    with torch.cuda.device(A.device):
        _check(load_library().pfc_tc_chain_probe(A.data_ptr(), B.data_ptr(), A.shape[1] // 16, int(n_mma), D.data_ptr(),
                                                 _stream_ptr(stream)), "pfc_tc_chain_probe")
    return D


def pfc_workspace_bytes(n_atoms: int, n_systems: int) -> int:
    return int(load_library().pfc_workspace_bytes(int(n_atoms), int(n_systems)))


def _stream_ptr(stream) -> int:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def _on_device(method):
    """Run a Pfc method with the handle's CUDA device current (the library checks it: a handle is
    bound to the device it was created on), so that a handle on cuda:1 works while cuda:0 is current."""
    import functools

    @functools.wraps(method)
    def wrapper(self, *args, **kwargs):
        import torch
        with torch.cuda.device(self.device):
            return method(self, *args, **kwargs)
    return wrapper


class Pfc:
    """One handle = one set of systems + one potential (pfc_create .. pfc_destroy)."""

    def __init__(self, species, sys_offsets, weights, masses_amu=None, mlp_path: int = MLP_AUTO,
                 device="cuda:0", tuning: "Tuning | None" = None):
        import torch
        if not torch.cuda.is_available():
            raise PfcError("pfc needs a CUDA device (sm_100a); there is no CPU fallback")
        self._lib = load_library()
        self.device = torch.device(device)
        species = np.ascontiguousarray(species, dtype=np.int32)
        sys_offsets = np.ascontiguousarray(sys_offsets, dtype=np.int32)
        weights = np.ascontiguousarray(weights, dtype=np.float32)
        if weights.shape != (N_WEIGHTS,):
            raise PfcError(f"weights must have {N_WEIGHTS} floats")
        self.n_atoms = int(species.shape[0])
        self.n_systems = int(sys_offsets.shape[0] - 1)
        nbytes = pfc_workspace_bytes(self.n_atoms, self.n_systems)
        if nbytes == 0:
            raise PfcError("bad sizes")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self.workspace.data_ptr() + 255) // 256 * 256
            masses = None if masses_amu is None else np.ascontiguousarray(masses_amu, dtype=np.float32)
            d = _Desc(self.n_atoms, self.n_systems,
                      species.ctypes.data_as(POINTER(c_int32)), sys_offsets.ctypes.data_as(POINTER(c_int32)),
                      weights.ctypes.data_as(POINTER(c_float)),
                      None if masses is None else masses.ctypes.data_as(POINTER(c_float)),
                      c_void_p(base), c_size_t(nbytes), int(mlp_path),
                      None if tuning is None else ctypes.pointer(tuning))
            h = c_void_p()
            _check(self._lib.pfc_create(byref(d), byref(h)), "pfc_create")
        self._h = h
        self._bound = None

    # -- pfc_energy_forces ------------------------------------------------------
    @_on_device
    def energy_forces(self, pos, E=None, F=None, stream=None):
        """pos: cuda float32 [N,4].  Returns (E [n_systems], F [N,4] = {Fx,Fy,Fz,e_i}); enqueues only."""
        import torch
        self._expect(pos, (self.n_atoms, 4))
        if E is None:
            E = torch.empty(self.n_systems, dtype=torch.float32, device=self.device)
        if F is None:
            F = torch.empty(self.n_atoms, 4, dtype=torch.float32, device=self.device)
        self._expect(E, (self.n_systems,))
        self._expect(F, (self.n_atoms, 4))
        _check(self._lib.pfc_energy_forces(self._h, pos.data_ptr(), E.data_ptr(), F.data_ptr(),
                                           _stream_ptr(stream)), "pfc_energy_forces")
        return E, F

    @_on_device
    def profile_stages(self, pos, E, F, stream=None):
        """Per-stage device times (ms) of one energy_forces pass; synchronises."""
        ms = (c_float * N_STAGES)()
        _check(self._lib.pfc_profile_stages(self._h, pos.data_ptr(), E.data_ptr(), F.data_ptr(),
                                            _stream_ptr(stream), ms), "pfc_profile_stages")
        return [float(x) for x in ms]

    # -- pfc_set_state / pfc_step -------------------------------------------------
    @_on_device
    def set_state(self, pos, vel, E=None, F=None, stream=None):
        import torch
        self._expect(pos, (self.n_atoms, 4))
        self._expect(vel, (self.n_atoms, 4))
        if E is None:
            E = torch.empty(self.n_systems, dtype=torch.float32, device=self.device)
        if F is None:
            F = torch.empty(self.n_atoms, 4, dtype=torch.float32, device=self.device)
        self._expect(E, (self.n_systems,))
        self._expect(F, (self.n_atoms, 4))
        _check(self._lib.pfc_set_state(self._h, pos.data_ptr(), vel.data_ptr(), E.data_ptr(), F.data_ptr(),
                                       _stream_ptr(stream)), "pfc_set_state")
        self._bound = (pos, vel, E, F)          # keep the tensors alive while bound
        return E, F

    @_on_device
    def step(self, n_steps: int, dt_fs: float = 0.5):
        _check(self._lib.pfc_step(self._h, int(n_steps), float(dt_fs)), "pfc_step")

    @_on_device
    def energy_forces_nm(self, pos_nm, want_forces: bool = True, stream=None):
        """Provider call in the paper's units: pos_nm cuda [N,3] float32 (nm) -> (E kJ/mol [n_systems],
        F kJ/mol/nm [N,3] or None).  Marshalling only; the conversion runs in the library's kernels."""
        import torch
        self._expect(pos_nm, (self.n_atoms, 3))
        E = torch.empty(self.n_systems, dtype=torch.float32, device=self.device)
        F = torch.empty(self.n_atoms, 3, dtype=torch.float32, device=self.device) if want_forces else None
        _check(self._lib.pfc_energy_forces_nm(self._h, pos_nm.data_ptr(), E.data_ptr(),
                                              F.data_ptr() if want_forces else None, _stream_ptr(stream)),
               "pfc_energy_forces_nm")
        return E, F

    @_on_device
    def step_langevin(self, n_steps: int, dt_fs: float, friction_per_fs: float, temperature_K: float, seed: int):
        _check(self._lib.pfc_step_langevin(self._h, int(n_steps), float(dt_fs), float(friction_per_fs),
                                           float(temperature_K), int(seed)), "pfc_step_langevin")

    @_on_device
    def set_frames(self, frames, stride: int):
        """frames: device tensor [max_frames, N, 4] float32 (None unbinds)."""
        if frames is None:
            _check(self._lib.pfc_set_frames(self._h, None, 0, 0), "pfc_set_frames")
        else:
            self._expect(frames, (frames.shape[0], self.n_atoms, 4))
            _check(self._lib.pfc_set_frames(self._h, frames.data_ptr(), int(stride), int(frames.shape[0])),
                   "pfc_set_frames")
        self._frames = frames                   # keep alive while bound

    def frames_written(self) -> int:
        n = c_int32()
        _check(self._lib.pfc_frames_written(self._h, byref(n)), "pfc_frames_written")
        return int(n.value)

    # -- pfc_run_host -------------------------------------------------------------
    @_on_device
    def run_host(self, pos_host, vel_host, n_steps: int, dt_fs: float, E_host, F_host=None, stream=None):
        """Host tensors/arrays [N,4] float32 (pinned for async copies), updated in place."""
        def ptr(a):
            if a is None:
                return None
            return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data
        _check(self._lib.pfc_run_host(self._h, ptr(pos_host), ptr(vel_host), int(n_steps), float(dt_fs),
                                      ptr(E_host), ptr(F_host), _stream_ptr(stream)), "pfc_run_host")

    @_on_device
    def run_host_resume(self, pos_host, vel_host, F_host, n_steps: int, dt_fs: float, E_host, stream=None):
        """As run_host, with F_host [N,4] holding the forces at pos_host on entry (uploaded, not recomputed)."""
        def ptr(a):
            return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data
        _check(self._lib.pfc_run_host_resume(self._h, ptr(pos_host), ptr(vel_host), ptr(F_host), int(n_steps),
                                             float(dt_fs), ptr(E_host), _stream_ptr(stream)), "pfc_run_host_resume")

    # -- getters ------------------------------------------------------------------
    def mlp_path(self) -> int:
        """The MLP path in use (MLP_AUTO resolved)."""
        v = c_int32()
        _check(self._lib.pfc_mlp_path(self._h, byref(v)), "pfc_mlp_path")
        return int(v.value)

    def tc_calibration(self):
        """pfc_tc_calibration: per element {lambda_f, lambda_b, slope_e, slope_g, max_de, max_dg, final, fallback}."""
        out = (c_float * 32)()
        _check(self._lib.pfc_tc_calibration(self._h, out), "pfc_tc_calibration")
        return np.array(out[:], dtype=np.float32).reshape(4, 8)

    @_on_device
    def status(self) -> int:
        bits = c_uint32()
        _check(self._lib.pfc_status(self._h, byref(bits)), "pfc_status")
        return int(bits.value)

    def check_status(self) -> None:
        bits = self.status()
        if bits:
            raise PfcError("device status: " + ", ".join(v for k, v in STATUS_BITS.items() if bits & k))

    def launch_counts(self):
        """(kernel launches per energy/forces evaluation, per steady-state MD step)."""
        a, b, k = c_int32(), c_int32(), c_int32()
        _check(self._lib.pfc_launch_counts(self._h, byref(a), byref(b), byref(k)), "pfc_launch_counts")
        return int(a.value), int(b.value)

    def steps_per_graph(self) -> int:
        a, b, k = c_int32(), c_int32(), c_int32()
        _check(self._lib.pfc_launch_counts(self._h, byref(a), byref(b), byref(k)), "pfc_launch_counts")
        return int(k.value)

    @_on_device
    def k3_timeline(self):
        """SM-clock timeline of the tensor-core MLP kernel's first CTA: int64 array [8, 128] (pfc_k3_timeline)."""
        v = (ctypes.c_int64 * 1024)()
        _check(self._lib.pfc_k3_timeline(self._h, v, 1024), "pfc_k3_timeline")
        return np.array(v[:], dtype=np.int64).reshape(8, 128)

    @_on_device
    def work_counts(self):
        """Row totals of the last evaluation: dict(radial, angular, triples, brute_tests, skin_builds); synchronises."""
        v = (ctypes.c_int64 * 5)()
        _check(self._lib.pfc_work_counts(self._h, v), "pfc_work_counts")
        return {"radial": int(v[0]), "angular": int(v[1]), "triples": int(v[2]), "brute_tests": int(v[3]),
                "skin_builds": int(v[4])}

    @_on_device
    def neighbors(self):
        """The neighbour lists of the last evaluation as int32 CSR (r_off, r_idx, a_off, a_idx), copied
        to host numpy arrays (pfc_get_neighbors exports the step path's rows; synchronises)."""
        import torch
        p = [POINTER(c_int32)() for _ in range(4)]
        _check(self._lib.pfc_get_neighbors(self._h, *[byref(x) for x in p]), "pfc_get_neighbors")
        torch.cuda.synchronize(self.device)
        r_off = self._copy(p[0], self.n_atoms + 1, np.int32)
        a_off = self._copy(p[2], self.n_atoms + 1, np.int32)
        r_idx = self._copy(p[1], int(r_off[-1]), np.int32)
        a_idx = self._copy(p[3], int(a_off[-1]), np.int32)
        return r_off, r_idx, a_off, a_idx

    @_on_device
    def neighbor_offsets_noalloc(self, r_off=None, a_off=None, stream=None):
        """pfc_neighbor_offsets_noalloc (include/pfc_noalloc.h): r_off / a_off of the last evaluation into
        caller-owned cuda int32 tensors [n_atoms + 1] (made here if not given); the library's scratch for it is a
        static device array.  Enqueues only."""
        import torch
        if r_off is None:
            r_off = torch.empty(self.n_atoms + 1, dtype=torch.int32, device=self.device)
        if a_off is None:
            a_off = torch.empty(self.n_atoms + 1, dtype=torch.int32, device=self.device)
        for t in (r_off, a_off):
            if not (t.is_cuda and t.dtype == torch.int32 and t.numel() == self.n_atoms + 1 and t.is_contiguous()):
                raise PfcError("expected contiguous cuda int32 tensors of n_atoms + 1 elements")
        _check(self._lib.pfc_neighbor_offsets_noalloc(self._h, r_off.data_ptr(), a_off.data_ptr(), _stream_ptr(stream)),
               "pfc_neighbor_offsets_noalloc")
        return r_off, a_off

    @_on_device
    def intermediates(self):
        """(aev [N,384], g [N,384]) of the last evaluation in ATOM order (host copies)."""
        import torch
        pa, pg, pr, nr = POINTER(c_float)(), POINTER(c_float)(), POINTER(c_int32)(), c_int32()
        _check(self._lib.pfc_get_intermediates(self._h, byref(pa), byref(pg), byref(pr), byref(nr)),
               "pfc_get_intermediates")
        torch.cuda.synchronize(self.device)
        rows = self._copy(pr, self.n_atoms, np.int32)
        aev = self._copy(pa, nr.value * AEV_LEN, np.float32).reshape(nr.value, AEV_LEN)
        g = self._copy(pg, nr.value * AEV_LEN, np.float32).reshape(nr.value, AEV_LEN)
        return aev[rows], g[rows]

    def _copy(self, dev_ptr, n, dtype):
        """device -> host copy of n items (marshalling only)."""
        out = np.empty(n, dtype=dtype)
        if n:
            addr = ctypes.cast(dev_ptr, c_void_p).value
            _check(self._lib.pfc_copy_to_host(addr, out.ctypes.data, n * out.itemsize), "pfc_copy_to_host")
        return out

    def _expect(self, t, shape):
        import torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32
                and tuple(t.shape) == tuple(shape) and t.is_contiguous()):
            raise PfcError(f"expected a contiguous cuda float32 tensor of shape {shape}")

    @_on_device
    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.pfc_destroy(self._h)
            self._h = c_void_p()
        self._bound = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def pack4(a3) -> np.ndarray:
    """[N,3] -> [N,4] float32 with a zero .w lane (layout helper, no arithmetic)."""
    a3 = np.asarray(a3, dtype=np.float32)
    out = np.zeros((a3.shape[0], 4), dtype=np.float32)
    out[:, :3] = a3
    return out
