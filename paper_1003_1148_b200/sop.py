"""ctypes binding of include/sop.h.  Argument marshalling only."""
from __future__ import annotations

import ctypes as C
import math
import os

import numpy as np

from . import _build

_lib = None

STATUS = {0: "SOP_OK", -1: "SOP_E_ARG", -2: "SOP_E_CUDA", -3: "SOP_E_LIST_OVERFLOW", -4: "SOP_E_FENE",
          -5: "SOP_E_NONFINITE"}

NOALLOC_SCRATCH_BYTES = 1 << 20      # SOP_NOALLOC_SCRATCH_BYTES of include/sop.h

SYMBOLS = ["sop_query_workspace", "sop_create", "sop_destroy", "sop_run", "sop_sync", "sop_get_coords",
           "sop_set_coords", "sop_get_energies", "sop_get_observables", "sop_get_forces", "sop_get_lists", "sop_get_step", "sop_set_step",
           "sop_device_coords", "sop_get_config", "sop_set_profiling", "sop_get_profile", "sop_last_error",
           "sop_set_observable_stride", "sop_get_observable_series", "sop_replica_exchange", "sop_get_temperatures",
           "sop_energies_noalloc", "sop_plan_slices"]


class _Topology(C.Structure):
    _fields_ = [("n_beads", C.c_int32),
                ("n_bonds", C.c_int32), ("bonds", C.c_void_p),
                ("n_native", C.c_int32), ("native", C.c_void_p),
                ("native_eps", C.c_void_p)]


class _Params(C.Structure):
    _fields_ = [("k_fene", C.c_float), ("R0", C.c_float), ("eps_native", C.c_float),
                ("eps_rep", C.c_float), ("sigma", C.c_float),
                ("R_nb", C.c_float), ("R_pl", C.c_float),
                ("nb_interval", C.c_int32), ("pl_interval", C.c_int32),
                ("cap_nb", C.c_int32), ("cap_pl", C.c_int32),
                ("dt_over_zeta", C.c_float), ("kT", C.c_float),
                ("kT_per_traj", C.c_void_p), ("integrator", C.c_int32),
                ("seed", C.c_uint64),
                ("traj_offset", C.c_int32),
                ("n_fixed", C.c_int32), ("fixed", C.c_void_p),
                ("n_pulled", C.c_int32), ("pulled", C.c_void_p),
                ("pull_k", C.c_float), ("pull_v", C.c_float), ("pull_dir", C.c_float * 3),
                ("tip_on", C.c_int32), ("tip_R", C.c_float), ("tip_eps", C.c_float), ("tip_sigma", C.c_float),
                ("tip_c0", C.c_float * 3), ("tip_dir", C.c_float * 3), ("tip_v", C.c_float),
                ("lanes_per_bead", C.c_int32), ("block_size", C.c_int32), ("compensated", C.c_int32),
                ("pair_atomics", C.c_int32), ("mode", C.c_int32), ("reorder", C.c_int32), ("chunk_beads", C.c_int32), ("resident_variant", C.c_int32),
                ("obs_stride", C.c_int32), ("obs_capacity", C.c_int32), ("rng", C.c_int32),
                ("stream", C.c_void_p)]


def library_path() -> str:
    return _build.LIB


def lib():
    """Load libsop.so (building it with nvcc if it is missing or older than its sources).  No fallback."""
    global _lib
    if _lib is None:
        try:
            path = _build.build()
            L = C.CDLL(path)
        except Exception as e:  # noqa: BLE001
            raise ImportError(f"the CUDA library {_build.LIB} is missing and could not be built: {e}. "
                              "This package has no CPU fallback.") from e
        vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
        L.sop_query_workspace.argtypes = [C.POINTER(_Topology), vp, C.POINTER(_Params), i32, C.POINTER(C.c_size_t)]
        L.sop_create.argtypes = [C.POINTER(_Topology), vp, C.POINTER(_Params), i32, vp, C.c_size_t, C.POINTER(vp)]
        L.sop_destroy.argtypes = [vp]; L.sop_destroy.restype = None
        L.sop_run.argtypes = [vp, i64]
        L.sop_sync.argtypes = [vp]
        L.sop_get_coords.argtypes = [vp, vp]
        L.sop_set_coords.argtypes = [vp, vp]
        L.sop_get_energies.argtypes = [vp, vp]
        L.sop_energies_noalloc.argtypes = [vp, vp]
        L.sop_get_forces.argtypes = [vp, vp]
        L.sop_get_observables.argtypes = [vp, vp]
        L.sop_set_observable_stride.argtypes = [vp, i32]
        L.sop_replica_exchange.argtypes = [vp, i32, C.c_uint64, vp]
        L.sop_get_temperatures.argtypes = [vp, vp]
        L.sop_get_observable_series.argtypes = [vp, vp, vp, i32, C.POINTER(i32)]
        L.sop_get_lists.argtypes = [vp, i32, i32, vp, vp, C.POINTER(i32), C.POINTER(i64)]
        L.sop_get_step.argtypes = [vp, C.POINTER(i64)]
        L.sop_set_step.argtypes = [vp, i64]
        L.sop_device_coords.argtypes = [vp, C.POINTER(vp), vp]
        L.sop_get_config.argtypes = [vp, vp]
        L.sop_plan_slices.argtypes = [i32, i32, i32, i32]; L.sop_plan_slices.restype = i32
        L.sop_set_profiling.argtypes = [vp, i32]
        L.sop_get_profile.argtypes = [vp, vp]
        L.sop_last_error.argtypes = [vp]; L.sop_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def exported_symbols():
    """Names declared in include/sop.h that the loaded library exports (no compute call is made)."""
    L = lib()
    return [s for s in SYMBOLS if hasattr(L, s)]


class SopError(RuntimeError):
    def __init__(self, code, where, msg=""):
        super().__init__(f"{where}: {STATUS.get(code, code)} {msg}")
        self.code = code


def _marshal(xyz, bonds, native, params, native_eps, overrides):
    p = dict(params)
    p.update(overrides)
    keep = {}
    keep["xyz"] = np.ascontiguousarray(xyz, np.float32).reshape(-1, 3)
    keep["bonds"] = np.ascontiguousarray(bonds, np.int32).reshape(-1, 2)
    keep["native"] = np.ascontiguousarray(native, np.int32).reshape(-1, 2)
    keep["eps"] = None if native_eps is None else np.ascontiguousarray(native_eps, np.float32)
    keep["fixed"] = np.ascontiguousarray(p.get("fixed", []), np.int32)
    keep["pulled"] = np.ascontiguousarray(p.get("pulled", []), np.int32)
    keep["kT_t"] = None if p.get("kT_per_traj") is None else np.ascontiguousarray(p["kT_per_traj"], np.float32)
    tp = _Topology(len(keep["xyz"]), len(keep["bonds"]), keep["bonds"].ctypes.data, len(keep["native"]),
                   keep["native"].ctypes.data, None if keep["eps"] is None else keep["eps"].ctypes.data)
    pp = _Params()
    for name in ("k_fene", "R0", "eps_native", "eps_rep", "sigma", "R_nb", "dt_over_zeta", "kT"):
        setattr(pp, name, float(p[name]))
    pp.R_pl = math.inf if math.isinf(p["R_pl"]) else float(p["R_pl"])
    pp.nb_interval = int(p["nb_interval"]); pp.pl_interval = int(p["pl_interval"])
    pp.cap_nb = int(p.get("cap_nb", 0)); pp.cap_pl = int(p.get("cap_pl", 0))
    pp.seed = int(p["seed"]); pp.traj_offset = int(p.get("traj_offset", 0))
    pp.n_fixed = len(keep["fixed"]); pp.fixed = keep["fixed"].ctypes.data
    pp.n_pulled = len(keep["pulled"]); pp.pulled = keep["pulled"].ctypes.data
    pp.kT_per_traj = None if keep["kT_t"] is None else keep["kT_t"].ctypes.data
    pp.integrator = int(p.get("integrator", 0))
    pp.pull_k = float(p.get("pull_k", 0.0)); pp.pull_v = float(p.get("pull_v", 0.0))
    pp.pull_dir = (C.c_float * 3)(*[float(v) for v in p.get("pull_dir", [0, 0, 1])])
    pp.tip_on = int(p.get("tip_on", 0))
    pp.tip_R = float(p.get("tip_R", 0.0)); pp.tip_eps = float(p.get("tip_eps", 0.0)); pp.tip_sigma = float(p.get("tip_sigma", 0.0))
    pp.tip_c0 = (C.c_float * 3)(*[float(v) for v in p.get("tip_c0", [0, 0, 0])])
    pp.tip_dir = (C.c_float * 3)(*[float(v) for v in p.get("tip_dir", [0, 0, -1])])
    pp.tip_v = float(p.get("tip_v", 0.0))
    pp.lanes_per_bead = int(p.get("lanes_per_bead", 0)); pp.block_size = int(p.get("block_size", 0))
    pp.pair_atomics = int(p.get("pair_atomics", 0))
    pp.compensated = int(p.get("compensated", 0)); pp.mode = int(p.get("mode", 0)); pp.reorder = int(p.get("reorder", 0))
    pp.chunk_beads = int(p.get("chunk_beads", 0)); pp.rng = int(p.get("rng", 0))
    pp.resident_variant = int(p.get("resident_variant", 0))
    pp.obs_stride = int(p.get("obs_stride", 0)); pp.obs_capacity = int(p.get("obs_capacity", 0))
    return tp, pp, keep


class Sop:
    """One simulation handle.  `params` is a plain dict (see workloads.generators.BASE_PARAMS); keyword overrides
    (lanes_per_bead, block_size, mode, reorder, chunk_beads, compensated, cap_nb, cap_pl, traj_offset, ...) are merged in."""

    def __init__(self, xyz, bonds, native, params, n_traj=1, native_eps=None, device=None, **overrides):
        import torch
        L = lib()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1003_1148_b200 needs a CUDA device; there is no CPU fallback")
        self._h = None
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        tp, pp, self._keep = _marshal(xyz, bonds, native, params, native_eps, overrides)
        self.N = tp.n_beads; self.T = int(n_traj)
        self._keep_obs_capacity = pp.obs_capacity
        with torch.cuda.device(self.device):
            self._stream = torch.cuda.current_stream()
            pp.stream = self._stream.cuda_stream
            nbytes = C.c_size_t()
            rc = L.sop_query_workspace(C.byref(tp), self._keep["xyz"].ctypes.data, C.byref(pp), self.T, C.byref(nbytes))
            if rc:
                raise SopError(rc, "sop_query_workspace", (L.sop_last_error(None) or b"").decode())
            self.workspace_bytes = nbytes.value
            self._ws = torch.empty(nbytes.value + 256, dtype=torch.uint8, device=self.device)
            base = (self._ws.data_ptr() + 255) // 256 * 256
            h = C.c_void_p()
            rc = L.sop_create(C.byref(tp), self._keep["xyz"].ctypes.data, C.byref(pp), self.T, base, nbytes.value, C.byref(h))
            if rc:
                raise SopError(rc, "sop_create", (L.sop_last_error(None) or b"").decode())
            self._h = h

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None):
            lib().sop_destroy(self._h)
            self._h = None
            self._ws = None

    __del__ = close

    def _chk(self, rc, where):
        if rc:
            raise SopError(rc, where, (lib().sop_last_error(self._h) or b"").decode())

    # -- the four calls of the north star
    def run(self, n_steps):
        self._chk(lib().sop_run(self._h, int(n_steps)), "sop_run")

    def sync(self):
        self._chk(lib().sop_sync(self._h), "sop_sync")

    def get_coords(self, out=None):
        out = np.empty((self.T, self.N, 3), np.float32) if out is None else out
        self._chk(lib().sop_get_coords(self._h, out.ctypes.data), "sop_get_coords")
        return out

    def get_energies(self):
        out = np.empty((self.T, 6), np.float64)
        self._chk(lib().sop_get_energies(self._h, out.ctypes.data), "sop_get_energies")
        return out

    def energies_noalloc(self, d_out):
        """sop_energies_noalloc: the six energies into the caller's DEVICE tensor [T][6] float64; nothing is allocated, nothing
        copied to the host, no synchronisation (the result is valid after sync()).  Scratch: a static device array of
        NOALLOC_SCRATCH_BYTES shared by every call on the device."""
        if not (d_out.is_cuda and d_out.is_contiguous() and d_out.dtype.itemsize == 8 and d_out.numel() >= self.T * 6):
            raise ValueError("d_out must be a contiguous CUDA float64 tensor of at least T * 6 elements")
        self._chk(lib().sop_energies_noalloc(self._h, d_out.data_ptr()), "sop_energies_noalloc")
        return d_out

    # -- hooks
    def get_observables(self):
        """[T][4] float64: Rg, end-to-end distance, cantilever force, tip force (reduced on the device)."""
        out = np.zeros((self.T, 4), np.float64)
        self._chk(lib().sop_get_observables(self._h, out.ctypes.data), "sop_get_observables")
        return out

    def replica_exchange(self, parity, sweep):
        """one sweep of temperature swaps between trajectories (t, t+1), t = parity mod 2 -> accepted[T // 2]"""
        acc = np.zeros(max(1, self.T // 2), np.int32)
        self._chk(lib().sop_replica_exchange(self._h, int(parity), int(sweep), acc.ctypes.data), "sop_replica_exchange")
        return acc

    def get_temperatures(self):
        out = np.zeros(self.T, np.float32)
        self._chk(lib().sop_get_temperatures(self._h, out.ctypes.data), "sop_get_temperatures")
        return out

    def set_observable_stride(self, stride):
        self._chk(lib().sop_set_observable_stride(self._h, int(stride)), "sop_set_observable_stride")

    def get_observable_series(self, max_samples=1 << 20):
        """-> (steps[n], series[n][T][10]): Rg, X, cantilever force, tip force, V_fene, V_nat, V_rep, V_pull, V_tip, V_total
        of the samples recorded inside run() every obs_stride steps (the last `obs_capacity` of them at most)."""
        cap = max(1, min(int(max_samples), int(self._keep_obs_capacity)))
        out = np.zeros((cap, self.T, 10), np.float64); steps = np.zeros(cap, np.int64); n = C.c_int32()
        self._chk(lib().sop_get_observable_series(self._h, out.ctypes.data, steps.ctypes.data, cap, C.byref(n)), "sop_get_observable_series")
        return steps[:n.value].copy(), out[:n.value].copy()

    def set_coords(self, xyz):
        x = np.ascontiguousarray(xyz, np.float32).reshape(self.T, self.N, 3)
        self._chk(lib().sop_set_coords(self._h, x.ctypes.data), "sop_set_coords")

    def get_forces(self):
        out = np.empty((self.T, self.N, 3), np.float32)
        self._chk(lib().sop_get_forces(self._h, out.ctypes.data), "sop_get_forces")
        return out

    def get_lists(self, level, traj=0, counts_only=False):
        cap = C.c_int32(); at = C.c_int64()
        self._chk(lib().sop_get_lists(self._h, traj, level, None, None, C.byref(cap), C.byref(at)), "sop_get_lists")
        cnt = np.empty(self.N, np.int32)
        idx = None if counts_only else np.empty((self.N, cap.value), np.int32)
        self._chk(lib().sop_get_lists(self._h, traj, level, cnt.ctypes.data, None if idx is None else idx.ctypes.data,
                                      C.byref(cap), C.byref(at)), "sop_get_lists")
        return cnt, idx, at.value

    @property
    def step(self):
        s = C.c_int64(); self._chk(lib().sop_get_step(self._h, C.byref(s)), "sop_get_step"); return s.value

    @step.setter
    def step(self, v):
        self._chk(lib().sop_set_step(self._h, int(v)), "sop_set_step")

    def config(self):
        out = np.zeros(12, np.int32)
        self._chk(lib().sop_get_config(self._h, out.ctypes.data), "sop_get_config")
        names = ["lanes_per_bead", "block_size", "compensated", "mode", "reorder", "cap_nb", "cap_pl"]
        d = {k: int(v) for k, v in zip(names, out[:7])}
        d["launches"] = int(np.uint32(out[7])) | (int(np.uint32(out[8])) << 32)
        d["resident_variant"] = int(out[9])
        d["slice_len"] = int(out[10])
        return d

    def set_profiling(self, on=True):
        self._chk(lib().sop_set_profiling(self._h, 1 if on else 0), "sop_set_profiling")

    def get_profile(self):
        """-> dict of ms / span counts per kernel kind since the last call (synchronises)."""
        out = np.zeros(8, np.float64)
        self._chk(lib().sop_get_profile(self._h, out.ctypes.data), "sop_get_profile")
        return {"step_ms": out[0], "filter_ms": out[1], "l1_ms": out[2], "step_spans": int(out[3]),
                "filter_spans": int(out[4]), "l1_spans": int(out[5]), "langevin_steps": int(out[6])}

    def device_coords(self):
        """Zero-copy torch view [T][N][4] of the current layer (internal bead order) and the permutation."""
        import torch
        p = C.c_void_p(); perm = np.empty(self.N, np.int32)
        self._chk(lib().sop_device_coords(self._h, C.byref(p), perm.ctypes.data), "sop_device_coords")
        off = p.value - self._ws.data_ptr()
        view = self._ws[off: off + self.T * self.N * 16].view(torch.float32).view(self.T, self.N, 4)
        return view, perm


def from_workload(w, n_traj=None, **overrides):
    return Sop(w.xyz, w.bonds, w.native, w.params, n_traj=w.n_traj if n_traj is None else n_traj, **overrides)


# module-level names mirroring the C ABI
def sop_create(xyz, bonds, native, params, n_traj=1, **kw): return Sop(xyz, bonds, native, params, n_traj, **kw)
def sop_run(h, n_steps): return h.run(n_steps)
def sop_sync(h): return h.sync()
def sop_get_coords(h): return h.get_coords()
def sop_set_coords(h, xyz): return h.set_coords(xyz)
def sop_get_energies(h): return h.get_energies()
def sop_energies_noalloc(h, d_out): return h.energies_noalloc(d_out)
def sop_get_forces(h): return h.get_forces()
def sop_get_observables(h): return h.get_observables()
def sop_replica_exchange(h, parity, sweep): return h.replica_exchange(parity, sweep)
def sop_get_temperatures(h): return h.get_temperatures()
def sop_set_observable_stride(h, stride): return h.set_observable_stride(stride)
def sop_get_observable_series(h, max_samples=1 << 20): return h.get_observable_series(max_samples)
def sop_get_lists(h, level, traj=0): return h.get_lists(level, traj)
def sop_get_step(h): return h.step
def sop_set_step(h, v): h.step = v
def sop_destroy(h): return h.close()
