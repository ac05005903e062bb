"""ctypes binding of the fp64 oracle (oracle/sopo.c).  TEST INFRASTRUCTURE -- see oracle/sopo.h.

Argument marshalling only.  Every fp32 input of the product (coordinates, parameters) is rounded to fp32 and
promoted to double here, so that the oracle and the CUDA path see the same parameter values (R0)."""
from __future__ import annotations

import ctypes as C
import math

import numpy as np

from . import build as _build

_lib = None


class _Topology(C.Structure):
    _fields_ = [("n_beads", C.c_int32),
                ("n_bonds", C.c_int32), ("bonds", C.c_void_p),
                ("n_native", C.c_int32), ("native", C.c_void_p),
                ("native_eps", C.c_void_p)]


class _Params(C.Structure):
    _fields_ = [("k_fene", C.c_double), ("R0", C.c_double), ("eps_native", C.c_double),
                ("eps_rep", C.c_double), ("sigma", C.c_double),
                ("R_nb", C.c_double), ("R_pl", C.c_double),
                ("nb_interval", C.c_int32), ("pl_interval", C.c_int32),
                ("dt_over_zeta", C.c_double), ("kT", C.c_double),
                ("seed", C.c_uint64),
                ("traj_offset", C.c_int32),
                ("n_fixed", C.c_int32), ("fixed", C.c_void_p),
                ("n_pulled", C.c_int32), ("pulled", C.c_void_p),
                ("pull_k", C.c_double), ("pull_v", C.c_double), ("pull_dir", C.c_double * 3),
                ("tip_on", C.c_int32), ("tip_R", C.c_double), ("tip_eps", C.c_double), ("tip_sigma", C.c_double),
                ("tip_c0", C.c_double * 3), ("tip_dir", C.c_double * 3), ("tip_v", C.c_double),
                ("list_builder", C.c_int32), ("rng", C.c_int32), ("integrator", C.c_int32), ("kT_per_traj", C.c_void_p)]


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.sopo_create.argtypes = [C.POINTER(_Topology), C.c_void_p, C.POINTER(_Params), C.c_int32, C.POINTER(C.c_void_p)]
        L.sopo_destroy.argtypes = [C.c_void_p]
        L.sopo_destroy.restype = None
        L.sopo_run.argtypes = [C.c_void_p, C.c_int64]
        L.sopo_get_coords.argtypes = [C.c_void_p, C.c_void_p]
        L.sopo_set_coords.argtypes = [C.c_void_p, C.c_void_p]
        L.sopo_get_step.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
        L.sopo_set_step.argtypes = [C.c_void_p, C.c_int64]
        L.sopo_get_energies.argtypes = [C.c_void_p, C.c_void_p]
        L.sopo_get_forces.argtypes = [C.c_void_p, C.c_void_p]
        L.sopo_get_observables.argtypes = [C.c_void_p, C.c_void_p]
        L.sopo_taus_step.argtypes = [C.c_void_p]
        L.sopo_taus_step.restype = C.c_uint32
        L.sopo_taus_seed.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_void_p]
        L.sopo_taus_seed.restype = None
        L.sopo_get_lists.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(C.c_int64)]
        L.sopo_max_row.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.POINTER(C.c_int32)]
        L.sopo_build_lists.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_int32]
        L.sopo_filter.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_int32]
        L.sopo_eval_frozen.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
        L.sopo_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.sopo_philox4x32_10.restype = None
        L.sopo_normals.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint64, C.c_void_p]
        L.sopo_normals.restype = None
        L.sopo_normals_batch.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint64, C.c_void_p]
        L.sopo_normals_batch.restype = None
        L.sopo_pred.argtypes = [C.c_void_p, C.c_void_p, C.c_double]
        L.sopo_replica_exchange.argtypes = [C.c_void_p, C.c_int32, C.c_uint64, C.c_void_p]
        L.sopo_get_temperatures.argtypes = [C.c_void_p, C.c_void_p]
        L.sopo_rex_probability.argtypes = [C.c_double] * 4
        L.sopo_rex_probability.restype = C.c_double
        L.sopo_rex_accept.argtypes = [C.c_double] * 5
        _lib = L
    return _lib


class OracleError(RuntimeError):
    def __init__(self, code, where):
        super().__init__(f"oracle {where}: status {code}")
        self.code = code


def f32(v) -> float:
    """Round to fp32, promote to double."""
    return float(np.float32(v))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, np.uint32); k = np.asarray(key, np.uint32); o = np.zeros(4, np.uint32)
    lib().sopo_philox4x32_10(c.ctypes.data, k.ctypes.data, o.ctypes.data)
    return o


def normals(seed, bead, traj, step):
    g = np.zeros(3)
    lib().sopo_normals(int(seed), int(bead), int(traj), int(step), g.ctypes.data)
    return g


def normals_batch(seed, bead0, n_beads, traj, step):
    g = np.zeros((int(n_beads), 3))
    lib().sopo_normals_batch(int(seed), int(bead0), int(n_beads), int(traj), int(step), g.ctypes.data)
    return g


def pred(a, b, R):
    a = np.asarray(a, np.float64); b = np.asarray(b, np.float64)
    return bool(lib().sopo_pred(a.ctypes.data, b.ctypes.data, float(R)))


def num_threads():
    return int(lib().sopo_num_threads())


class Oracle:
    """One oracle simulation.  `params` is the plain dict produced by workloads.generators."""

    def __init__(self, xyz, bonds, native, params, n_traj=1, native_eps=None, list_builder=0, traj_offset=0):
        L = lib()
        self.N = int(len(xyz)); self.T = int(n_traj)
        self._xyz = np.ascontiguousarray(xyz, np.float32)
        self._bonds = np.ascontiguousarray(bonds, np.int32).reshape(-1, 2)
        self._native = np.ascontiguousarray(native, np.int32).reshape(-1, 2)
        self._eps = None if native_eps is None else np.ascontiguousarray([f32(e) for e in native_eps], np.float64)
        tp = _Topology(self.N, len(self._bonds), self._bonds.ctypes.data, len(self._native),
                       self._native.ctypes.data, None if self._eps is None else self._eps.ctypes.data)
        p = dict(params)
        self._fixed = np.ascontiguousarray(p.get("fixed", []), np.int32)
        self._pulled = np.ascontiguousarray(p.get("pulled", []), np.int32)
        pp = _Params()
        for name in ("k_fene", "R0", "eps_native", "eps_rep", "sigma", "R_nb", "dt_over_zeta", "kT"):
            setattr(pp, name, f32(p[name]))
        pp.R_pl = math.inf if math.isinf(p["R_pl"]) else f32(p["R_pl"])
        pp.nb_interval = int(p["nb_interval"]); pp.pl_interval = int(p["pl_interval"])
        pp.seed = int(p["seed"]); pp.traj_offset = int(traj_offset)
        pp.n_fixed = len(self._fixed); pp.fixed = self._fixed.ctypes.data
        pp.n_pulled = len(self._pulled); pp.pulled = self._pulled.ctypes.data
        pp.pull_k = f32(p.get("pull_k", 0.0)); pp.pull_v = f32(p.get("pull_v", 0.0))
        pp.pull_dir = (C.c_double * 3)(*[f32(v) for v in p.get("pull_dir", [0, 0, 1])])
        pp.tip_on = int(p.get("tip_on", 0))
        pp.tip_R = f32(p.get("tip_R", 0.0)); pp.tip_eps = f32(p.get("tip_eps", 0.0)); pp.tip_sigma = f32(p.get("tip_sigma", 0.0))
        pp.tip_c0 = (C.c_double * 3)(*[f32(v) for v in p.get("tip_c0", [0, 0, 0])])
        pp.tip_dir = (C.c_double * 3)(*[f32(v) for v in p.get("tip_dir", [0, 0, -1])])
        pp.tip_v = f32(p.get("tip_v", 0.0))
        pp.list_builder = int(list_builder)
        pp.rng = int(p.get("rng", 0))
        pp.integrator = int(p.get("integrator", 0))
        self._kT_t = None if p.get("kT_per_traj") is None else np.ascontiguousarray([f32(v) for v in p["kT_per_traj"]], np.float64)
        pp.kT_per_traj = None if self._kT_t is None else self._kT_t.ctypes.data
        self._h = C.c_void_p()
        rc = L.sopo_create(C.byref(tp), self._xyz.ctypes.data, C.byref(pp), self.T, C.byref(self._h))
        if rc:
            self._h = None
            raise OracleError(rc, "create")

    def close(self):
        if getattr(self, "_h", None):
            lib().sopo_destroy(self._h); self._h = None

    __del__ = close

    def _chk(self, rc, where):
        if rc:
            raise OracleError(rc, where)

    def run(self, n_steps):
        self._chk(lib().sopo_run(self._h, int(n_steps)), "run")

    def get_coords(self):
        out = np.zeros((self.T, self.N, 3), np.float64)
        self._chk(lib().sopo_get_coords(self._h, out.ctypes.data), "get_coords")
        return out

    def set_coords(self, xyz):
        x = np.ascontiguousarray(xyz, np.float64).reshape(self.T, self.N, 3)
        self._chk(lib().sopo_set_coords(self._h, x.ctypes.data), "set_coords")

    @property
    def step(self):
        s = C.c_int64(); lib().sopo_get_step(self._h, C.byref(s)); return s.value

    @step.setter
    def step(self, v):
        self._chk(lib().sopo_set_step(self._h, int(v)), "set_step")

    def get_energies(self):
        out = np.zeros((self.T, 6), np.float64)
        self._chk(lib().sopo_get_energies(self._h, out.ctypes.data), "get_energies")
        return out

    def get_observables(self):
        """[T][4]: Rg, end-to-end distance X, cantilever force, tip force."""
        out = np.zeros((self.T, 4), np.float64)
        self._chk(lib().sopo_get_observables(self._h, out.ctypes.data), "get_observables")
        return out

    def replica_exchange(self, parity, sweep):
        """one sweep of temperature swaps between runs (t, t+1), t = parity mod 2 -> accepted[T // 2] (pairs tried)"""
        acc = np.zeros(max(1, self.T // 2), np.int32)
        self._chk(lib().sopo_replica_exchange(self._h, int(parity), int(sweep), acc.ctypes.data), "replica_exchange")
        return acc

    def get_temperatures(self):
        out = np.zeros(self.T, np.float64)
        self._chk(lib().sopo_get_temperatures(self._h, out.ctypes.data), "get_temperatures")
        return out

    def get_forces(self):
        out = np.zeros((self.T, self.N, 3), np.float64)
        self._chk(lib().sopo_get_forces(self._h, out.ctypes.data), "get_forces")
        return out

    def max_row(self, level, traj=0):
        m = C.c_int32(); self._chk(lib().sopo_max_row(self._h, traj, level, C.byref(m)), "max_row"); return m.value

    def get_lists(self, level, traj=0):
        """-> (row_cnt[N], idx[N][cap], built_at_step); rows ascending in j."""
        cap = max(1, self.max_row(level, traj))
        cnt = np.zeros(self.N, np.int32); idx = np.full((self.N, cap), -1, np.int32); at = C.c_int64()
        self._chk(lib().sopo_get_lists(self._h, traj, level, cnt.ctypes.data, idx.ctypes.data, cap, C.byref(at)), "get_lists")
        return cnt, idx, at.value

    def build_lists(self, xyz, level, builder=0, cap=None):
        x = np.ascontiguousarray(xyz, np.float64).reshape(self.N, 3)
        cap = int(cap) if cap else self.N
        while True:
            cnt = np.zeros(self.N, np.int32); idx = np.full((self.N, cap), -1, np.int32)
            rc = lib().sopo_build_lists(self._h, x.ctypes.data, level, builder, cnt.ctypes.data, idx.ctypes.data, cap)
            if rc == -3 and cap < self.N:
                cap = min(self.N, cap * 2); continue
            self._chk(rc, "build_lists")
            m = max(1, int(cnt.max()) if self.N else 1)
            return cnt, np.ascontiguousarray(idx[:, :m])

    def filter(self, xyz, l1_cnt, l1_idx):
        x = np.ascontiguousarray(xyz, np.float64).reshape(self.N, 3)
        l1_cnt = np.ascontiguousarray(l1_cnt, np.int32); l1_idx = np.ascontiguousarray(l1_idx, np.int32)
        cap1 = l1_idx.shape[1]
        cnt = np.zeros(self.N, np.int32); idx = np.full((self.N, cap1), -1, np.int32)
        self._chk(lib().sopo_filter(self._h, x.ctypes.data, l1_cnt.ctypes.data, l1_idx.ctypes.data, cap1,
                                    cnt.ctypes.data, idx.ctypes.data, cap1), "filter")
        return cnt, idx

    def eval_frozen(self, xyz, step=0, traj=0, want_forces=True):
        x = np.ascontiguousarray(xyz, np.float64).reshape(self.N, 3)
        e = np.zeros(6); f = np.zeros((self.N, 3)) if want_forces else None
        rc = lib().sopo_eval_frozen(self._h, traj, x.ctypes.data, int(step), e.ctypes.data,
                                    None if f is None else f.ctypes.data)
        self._chk(rc, "eval_frozen")
        return e, f


def from_workload(w, n_traj=None, **kw):
    return Oracle(w.xyz, w.bonds, w.native, w.params, n_traj=w.n_traj if n_traj is None else n_traj, **kw)


def rex_probability(E_i, E_j, kT_i, kT_j):
    return float(lib().sopo_rex_probability(float(E_i), float(E_j), float(kT_i), float(kT_j)))


def rex_accept(E_i, E_j, kT_i, kT_j, u):
    return bool(lib().sopo_rex_accept(float(E_i), float(E_j), float(kT_i), float(kT_j), float(u)))


def taus_step(y):
    """One Hybrid Taus draw (Alg. 6): y = 4 uint32 words of state, advanced in place; returns the 32-bit output."""
    return int(lib().sopo_taus_step(y.ctypes.data))


def taus_seed(seed, bead, traj):
    y = np.zeros(4, np.uint32)
    lib().sopo_taus_seed(int(seed), int(bead), int(traj), y.ctypes.data)
    return y
