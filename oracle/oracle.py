"""ctypes wrapper of the fp64 CPU oracle (oracle/fredopt_oracle.cpp) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fredopt_oracle.cpp")
_LIB = os.path.join(_HERE, "libfredopt_oracle.so")
_LIB_OMP = os.path.join(_HERE, "libfredopt_oracle_omp.so")      # timing build: same source, -fopenmp

OPT_ETA, OPT_REDUCTIONS, OPT_ACCEPT_CHECK, OPT_MAX_TRIALS, OPT_RESET = 0, 1, 2, 3, 4
OPT_BLOCK_SEQUENTIAL, OPT_NORMALIZE_GRAD, OPT_ONE_SIDED_COST = 7, 8, 9
VB_DOSE_LO, VB_DOSE_HI, VB_DL_LO, VB_DL_HI, VB_LETD_MAX, VB_DOSE_REF, VB_DL_REF = range(7)


def build(force: bool = False, omp: bool = False) -> str:
    """Compile the oracle with plain g++ -O2 (no fast-math); omp=True: the timing build of the same source with -fopenmp (row
    loops on all host cores)."""
    lib = _LIB_OMP if omp else _LIB
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off"] + (["-fopenmp"] if omp else []) +
                              ["-o", lib, _SRC])
    return lib


_libs = {}


def _load(omp: bool = False):
    if omp not in _libs:
        lib = C.CDLL(build(omp=omp))
        vp, i64, i32, f32, f64 = C.c_void_p, C.c_int64, C.c_int32, C.c_float, C.c_double
        lib.oracle_create.restype = vp
        lib.oracle_create.argtypes = [i64, i64, vp, vp, vp, vp, vp, vp, vp, vp, i32]
        lib.oracle_destroy.argtypes = [vp]
        lib.oracle_set_x.argtypes = [vp, vp]
        lib.oracle_set_x64.argtypes = [vp, vp]
        lib.oracle_get_x.argtypes = [vp, vp]
        lib.oracle_set_option.argtypes = [vp, i32, f64]
        lib.oracle_set_voxel_bounds.restype = i32
        lib.oracle_set_voxel_bounds.argtypes = [vp, i32, vp]
        lib.oracle_dose_let.argtypes = [vp, vp, vp, vp, vp]
        lib.oracle_dose_let_rows.argtypes = [vp, vp, vp, i64, vp, vp, vp]
        lib.oracle_transpose.argtypes = [vp, vp, vp, i32, vp, vp]
        lib.oracle_cost.restype = f64
        lib.oracle_cost.argtypes = [vp, vp]
        lib.oracle_grad.argtypes = [vp, vp, vp]
        lib.oracle_proximity.argtypes = [vp, vp, vp, vp]
        lib.oracle_iterate.restype = i32
        lib.oracle_iterate.argtypes = [vp, i32, f32, f32, f32]
        lib.oracle_stats.argtypes = [vp, vp, vp]
        lib.oracle_get_state.argtypes = [vp, vp, vp]
        lib.oracle_set_state.argtypes = [vp, vp, vp]
        lib.oracle_sweep_stats.argtypes = [vp, vp, vp]
        lib.oracle_structure_stats.argtypes = [vp, vp, i32, i32, vp, vp]
        lib.oracle_volume_histogram.argtypes = [vp, vp, i32, i32, i32, f64, vp]
        lib.oracle_percentile_value.restype = f64
        lib.oracle_percentile_value.argtypes = [vp, vp, i32, i32, f64]
        lib.oracle_norms.argtypes = [vp, vp, vp, vp]
        lib.oracle_what.argtypes = [vp, vp]
        lib.oracle_sequential_sweep.argtypes = [vp, f32]
        _libs[omp] = lib
    return _libs[omp]


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Oracle:
    """fp64 CPU restatement of the hot path.  Inputs are numpy arrays (fp32 values, int32 cols, int64 ptrs)."""

    def __init__(self, D, L, labels, bounds, omp=False):
        lib = _load(omp)
        rpD, ciD, vD = D
        rpL, ciL, vL = L
        self.V = len(rpD) - 1
        self.n_struct = int(np.asarray(bounds).shape[0])
        self._keep = [np.ascontiguousarray(rpD, np.int64), np.ascontiguousarray(ciD, np.int32),
                      np.ascontiguousarray(vD, np.float32), np.ascontiguousarray(rpL, np.int64),
                      np.ascontiguousarray(ciL, np.int32), np.ascontiguousarray(vL, np.float32),
                      np.ascontiguousarray(labels, np.int32), np.ascontiguousarray(bounds, np.float32)]
        self._lib = lib

    @classmethod
    def create(cls, V, S, D, L, labels, bounds, omp=False):
        """omp=True: the OpenMP timing build (threads = OMP_NUM_THREADS / all host cores)."""
        self = cls(D, L, labels, bounds, omp=omp)
        self.V, self.S = int(V), int(S)
        k = self._keep
        assert len(k[0]) == V + 1 and len(k[3]) == V + 1 and len(k[6]) == V
        self._h = self._lib.oracle_create(V, S, _p(k[0]), _p(k[1]), _p(k[2]), _p(k[3]), _p(k[4]), _p(k[5]),
                                          _p(k[6]), _p(k[7]), self.n_struct)
        self._keep = None   # the oracle copied everything
        return self

    def __del__(self):
        h = getattr(self, "_h", None)
        if h:
            self._lib.oracle_destroy(h)
            self._h = None

    # ---- state
    def set_x(self, x):
        x = np.ascontiguousarray(x)
        if x.dtype == np.float32:
            self._lib.oracle_set_x(self._h, _p(x))
        else:
            x = np.ascontiguousarray(x, np.float64)
            self._lib.oracle_set_x64(self._h, _p(x))

    def get_x(self):
        x = np.empty(self.S, np.float64)
        self._lib.oracle_get_x(self._h, _p(x))
        return x

    def set_option(self, key, value):
        self._lib.oracle_set_option(self._h, key, float(value))

    def set_voxel_bounds(self, field, values):
        """values: V floats (NaN = the structure's scalar) or None (remove the array)."""
        v = None if values is None else np.ascontiguousarray(values, np.float32)
        if self._lib.oracle_set_voxel_bounds(self._h, int(field), _p(v)) != 0:
            raise ValueError("per-voxel bounds: infinite value or lo > hi on a voxel")

    # ---- the calls of the boundary
    def dose_let(self, x=None):
        d = np.empty(self.V, np.float64); l = np.empty(self.V, np.float64); t = np.empty(self.V, np.float64)
        xx = None if x is None else np.ascontiguousarray(x, np.float64)
        self._lib.oracle_dose_let(self._h, _p(xx), _p(d), _p(l), _p(t))
        return d, l, t

    def dose_let_rows(self, rows, x=None):
        rows = np.ascontiguousarray(rows, np.int64)
        n = len(rows)
        d = np.empty(n, np.float64); l = np.empty(n, np.float64); t = np.empty(n, np.float64)
        xx = None if x is None else np.ascontiguousarray(x, np.float64)
        self._lib.oracle_dose_let_rows(self._h, _p(xx), _p(rows), n, _p(d), _p(l), _p(t))
        return d, l, t

    def transpose(self, u, v, active_only=False):
        uu = None if u is None else np.ascontiguousarray(u, np.float64)
        vv = None if v is None else np.ascontiguousarray(v, np.float64)
        out = np.empty(self.S, np.float64); oa = np.empty(self.S, np.float64)
        self._lib.oracle_transpose(self._h, _p(uu), _p(vv), int(active_only), _p(out), _p(oa))
        return out, oa

    def cost(self, x=None):
        xx = None if x is None else np.ascontiguousarray(x, np.float64)
        return float(self._lib.oracle_cost(self._h, _p(xx)))

    def grad(self, x=None):
        xx = None if x is None else np.ascontiguousarray(x, np.float64)
        g = np.empty(self.S, np.float64)
        self._lib.oracle_grad(self._h, _p(xx), _p(g))
        return g

    def proximity(self, x=None):
        xx = None if x is None else np.ascontiguousarray(x, np.float64)
        pr = C.c_double(0.0); nv = C.c_int64(0)
        self._lib.oracle_proximity(self._h, _p(xx), C.byref(pr), C.byref(nv))
        return pr.value, nv.value

    def iterate(self, n_iter, lam, beta0, a):
        if self._lib.oracle_iterate(self._h, int(n_iter), float(lam), float(beta0), float(a)) != 0:
            raise ValueError("beta0 / a differ from the pair latched by the first superiorized call (reset first)")

    def stats(self):
        o = np.zeros(5, np.int64); d = np.zeros(3, np.float64)
        self._lib.oracle_stats(self._h, _p(o), _p(d))
        return dict(k=int(o[0]), s=int(o[1]), trials=int(o[2]), n_sets=int(o[3]), n_zero_norm_sets=int(o[4]),
                    last_beta=float(d[0]), W=float(d[1]), beta_next=float(d[2]))

    def get_state(self):
        i = np.zeros(4, np.int64); d = np.zeros(5, np.float64)
        self._lib.oracle_get_state(self._h, _p(i), _p(d))
        return i, d

    def set_state(self, state):
        i, d = state
        self._lib.oracle_set_state(self._h, _p(np.ascontiguousarray(i, np.int64)), _p(np.ascontiguousarray(d, np.float64)))

    def sweep_stats(self):
        """(proximity, violated sets) met by the last block-sequential sweep at visit time."""
        pr = C.c_double(0.0); nv = C.c_int64(0)
        self._lib.oracle_sweep_stats(self._h, C.byref(pr), C.byref(nv))
        return pr.value, nv.value

    # ---- evaluation quantities (DVH / LVH / cDLVH, cDL30, Table 1)
    def structure_stats(self, quantity, label, x=None):
        xx = None if x is None else np.ascontiguousarray(x, np.float64)
        o = np.zeros(3, np.float64); n = C.c_int64(0)
        self._lib.oracle_structure_stats(self._h, _p(xx), int(quantity), int(label), _p(o), C.byref(n))
        return float(o[0]), float(o[1]), float(o[2]), n.value

    def volume_histogram(self, quantity, label, n_bins, vmax, x=None):
        xx = None if x is None else np.ascontiguousarray(x, np.float64)
        hst = np.zeros(n_bins, np.float64)
        self._lib.oracle_volume_histogram(self._h, _p(xx), int(quantity), int(label), int(n_bins), float(vmax), _p(hst))
        return hst

    def percentile_value(self, quantity, label, fraction, x=None):
        xx = None if x is None else np.ascontiguousarray(x, np.float64)
        return float(self._lib.oracle_percentile_value(self._h, _p(xx), int(quantity), int(label), float(fraction)))

    def norms(self):
        a = np.empty(self.V, np.float64); b = np.empty(self.V, np.float64); c = np.empty(self.V, np.float64)
        self._lib.oracle_norms(self._h, _p(a), _p(b), _p(c))
        return a, b, c

    def what(self):
        w = np.empty(self.n_struct, np.float64)
        self._lib.oracle_what(self._h, _p(w))
        return w

    def sequential_sweep(self, lam):
        self._lib.oracle_sequential_sweep(self._h, float(lam))


def from_plan(plan, omp=False) -> "Oracle":
    """Oracle over a plangen.Plan (tensors are copied to host numpy)."""
    rp, ci, vd, vl, lab = plan.to_numpy()
    return Oracle.create(plan.n_rows, plan.n_cols, (rp, ci, vd), (rp, ci, vl), lab, plan.bounds, omp=omp)


def omp_threads(n: int = 0) -> int:
    """Threads the OpenMP timing build runs with (n >= 1: set them first)."""
    lib = _load(True)
    lib.oracle_threads.restype = C.c_int32
    lib.oracle_set_threads.argtypes = [C.c_int32]
    if n >= 1:
        lib.oracle_set_threads(int(n))
    return int(lib.oracle_threads())
