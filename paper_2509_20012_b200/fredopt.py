"""Thin ctypes binding onto the C-ABI library (include/fredopt.h): argument marshalling only.

Every step of the hot path runs inside libfredopt.so (hand-written CUDA for sm_100a).  There is no CPU
fallback: importing this module raises if the library is missing or fails to load, and every call raises
`FredoptError` on a non-zero return code.  Array arguments may be torch tensors (CPU or CUDA), numpy arrays
or None; only their data pointers cross the boundary.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfredopt.so")

OK, INVALID_ARG, OUT_OF_MEMORY, CUDA_ERROR, UNSUPPORTED_ARCH, UNSUPPORTED = 0, -1, -2, -3, -4, -5
OPT_ETA, OPT_REDUCTIONS, OPT_ACCEPT_CHECK, OPT_MAX_TRIALS, OPT_RESET, OPT_USE_GRAPH, OPT_TIME_PASSES, \
    OPT_BLOCK_SEQUENTIAL, OPT_NORMALIZE_GRAD, OPT_ONE_SIDED_COST, OPT_USE_PDL, OPT_WORK_QUEUE, OPT_SKIP_SATISFIED = range(13)
ROWS_ALL, ROWS_ACTIVE = 0, 1
VB_DOSE_LO, VB_DOSE_HI, VB_DL_LO, VB_DL_HI, VB_LETD_MAX, VB_DOSE_REF, VB_DL_REF = range(7)
PASS_NAMES = ("forward_x", "transpose_g", "forward_g", "select", "residual", "transpose_b")
N_PASSES = len(PASS_NAMES)

# every symbol include/fredopt.h declares (tests check the library exports exactly these)
SYMBOLS = (
    "fredopt_create", "fredopt_create_ex", "fredopt_destroy", "fredopt_set_weights", "fredopt_get_weights", "fredopt_get_weights_f64",
    "fredopt_set_weights_f64", "fredopt_get_state", "fredopt_set_state", "fredopt_shard_range", "fredopt_set_reduce",
    "fredopt_set_voxel_bounds", "fredopt_dose_let", "fredopt_iterate", "fredopt_iterate_host", "fredopt_proximity", "fredopt_set_option", "fredopt_get_stats",
    "fredopt_spmv_forward", "fredopt_spmv_transpose", "fredopt_get_pass_times", "fredopt_get_pass_bytes",
    "fredopt_get_pass_bytes_timed",
    "fredopt_launch_count", "fredopt_stream_read", "fredopt_strerror", "fredopt_last_cuda_error",
    "fredopt_structure_stats", "fredopt_volume_histogram", "fredopt_percentile_value",
    "fredopt_no_alloc_setup", "fredopt_volume_histogram_no_alloc",
)


class FredoptError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = _lib.fredopt_strerror(code).decode()
        cuda = _lib.fredopt_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} ({code})" + (f" [{cuda}]" if cuda and code == CUDA_ERROR else ""))


class _Csr(C.Structure):
    _fields_ = [("n_rows", C.c_int64), ("n_cols", C.c_int64), ("nnz", C.c_int64),
                ("row_ptr", C.c_void_p), ("col_idx", C.c_void_p), ("values", C.c_void_p)]


class _Bounds(C.Structure):
    _fields_ = [(n, C.c_float) for n in ("weight", "dose_lo", "dose_hi", "dl_lo", "dl_hi", "letd_max",
                                         "dose_ref", "dl_ref")]


class _CreateOptions(C.Structure):
    _fields_ = [("struct_size", C.c_int32), ("index_width", C.c_int32), ("block_rows", C.c_int32), ("shard_rank", C.c_int32),
                ("shard_world", C.c_int32), ("value_bits", C.c_int32)]


REDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p)   # fredopt_reduce_fn


class State(C.Structure):
    """fredopt_state: plain data, e.g. bytes(state) / State.from_buffer_copy(b) for a checkpoint file."""
    _fields_ = [("k", C.c_int64), ("s", C.c_int64), ("trials", C.c_int64), ("beta_next", C.c_double), ("eta_pow", C.c_double),
                ("last_beta", C.c_double), ("beta0", C.c_float), ("a", C.c_float), ("latched", C.c_int32), ("reserved", C.c_int32)]


class Stats(C.Structure):
    _fields_ = [(n, C.c_int64) for n in ("k", "s", "trials", "n_violated", "n_sets", "n_zero_norm_sets",
                                         "n_active_rows", "nnz", "nnz_active", "alg_bytes_iter", "block_rows", "entries_active")] + \
               [(n, C.c_double) for n in ("last_beta", "phi", "prox", "weight_sum")]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


def _load():
    if not os.path.exists(LIB_PATH):
        # a fresh checkout has no built library (it is git-ignored): compile it in-tree with nvcc, or fail loudly
        try:
            from . import build as _build
            _build.build_library()
        except Exception as e:
            raise ImportError(f"{LIB_PATH} is missing and could not be built ({e}); build it with "
                              "`python -m paper_2509_20012_b200.build` (there is no CPU fallback)") from e
    lib = C.CDLL(LIB_PATH)
    vp, i64, i32, f32, f64 = C.c_void_p, C.c_int64, C.c_int32, C.c_float, C.c_double
    lib.fredopt_create.argtypes = [C.POINTER(_Csr), C.POINTER(_Csr), vp, C.POINTER(_Bounds), i32, vp, C.POINTER(vp)]
    lib.fredopt_create_ex.argtypes = [C.POINTER(_Csr), C.POINTER(_Csr), vp, C.POINTER(_Bounds), i32, vp, C.POINTER(_CreateOptions),
                                      C.POINTER(vp)]
    lib.fredopt_destroy.argtypes = [vp]
    lib.fredopt_destroy.restype = None
    lib.fredopt_set_weights.argtypes = [vp, vp]
    lib.fredopt_get_weights.argtypes = [vp, vp]
    lib.fredopt_get_weights_f64.argtypes = [vp, vp]
    lib.fredopt_set_weights_f64.argtypes = [vp, vp]
    lib.fredopt_shard_range.argtypes = [vp, vp, i64, i32, i32, C.POINTER(i64), C.POINTER(i64)]
    lib.fredopt_set_reduce.argtypes = [vp, REDUCE_FN, vp]
    lib.fredopt_get_state.argtypes = [vp, C.POINTER(State)]
    lib.fredopt_set_state.argtypes = [vp, C.POINTER(State)]
    lib.fredopt_set_voxel_bounds.argtypes = [vp, i32, vp]
    lib.fredopt_dose_let.argtypes = [vp, vp, vp, vp]
    lib.fredopt_iterate.argtypes = [vp, i32, f32, f32, f32]
    lib.fredopt_iterate_host.argtypes = [vp, i32, f32, f32, f32, vp, vp, C.POINTER(Stats)]
    lib.fredopt_proximity.argtypes = [vp, vp, C.POINTER(f64), C.POINTER(i64)]
    lib.fredopt_set_option.argtypes = [vp, i32, f64]
    lib.fredopt_get_stats.argtypes = [vp, C.POINTER(Stats)]
    lib.fredopt_spmv_forward.argtypes = [vp, i32, vp, vp, vp]
    lib.fredopt_spmv_transpose.argtypes = [vp, i32, vp, vp, vp]
    lib.fredopt_structure_stats.argtypes = [vp, vp, i32, i32, C.POINTER(f64), C.POINTER(f64), C.POINTER(f64), C.POINTER(i64)]
    lib.fredopt_volume_histogram.argtypes = [vp, vp, i32, i32, i32, f64, vp]
    lib.fredopt_percentile_value.argtypes = [vp, vp, i32, i32, f64, C.POINTER(f64)]
    lib.fredopt_no_alloc_setup.argtypes = []
    lib.fredopt_volume_histogram_no_alloc.argtypes = [vp, vp, i64, i32, i32, f64, vp, vp, vp]
    lib.fredopt_get_pass_times.argtypes = [vp, C.POINTER(f64), C.POINTER(i64)]
    lib.fredopt_get_pass_bytes.argtypes = [vp, C.POINTER(i64)]
    lib.fredopt_get_pass_bytes_timed.argtypes = [vp, C.POINTER(i64)]
    lib.fredopt_launch_count.argtypes = [vp]
    lib.fredopt_launch_count.restype = i64
    lib.fredopt_stream_read.argtypes = [vp, vp, i64, i32]
    lib.fredopt_strerror.argtypes = [C.c_int]
    lib.fredopt_strerror.restype = C.c_char_p
    lib.fredopt_last_cuda_error.argtypes = []
    lib.fredopt_last_cuda_error.restype = C.c_char_p
    return lib


_lib = _load()


def _ptr(a, dtype=None, n=None):
    """Data pointer of a torch tensor / numpy array (contiguous, of the stated dtype and length), or None."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        if not a.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be contiguous")
        if dtype is not None and a.dtype != np.dtype(dtype):
            raise TypeError(f"expected {dtype}, got {a.dtype}")
        if n is not None and a.size != n:
            raise ValueError(f"expected {n} elements, got {a.size}")
        return a.ctypes.data
    # torch tensor
    if not a.is_contiguous():
        raise ValueError("tensor must be contiguous")
    if dtype is not None and str(a.dtype).split(".")[-1] != np.dtype(dtype).name:
        raise TypeError(f"expected {dtype}, got {a.dtype}")
    if n is not None and a.numel() != n:
        raise ValueError(f"expected {n} elements, got {a.numel()}")
    return a.data_ptr()


def _check(rc, where):
    if rc != OK:
        raise FredoptError(rc, where)


class Plan:
    """One plan = one GPU, one stream.  Mirrors the C calls one to one."""

    def __init__(self, n_rows, n_cols, D, L, voxel_labels, bounds, stream=None, **create_options):
        """D, L: (row_ptr int64, col_idx int32, values float32) triples; bounds: float32 [n_struct, 8] rows of
        (weight, dose_lo, dose_hi, dl_lo, dl_hi, letd_max, dose_ref, dl_ref), NaN = absent;
        stream: a raw cudaStream_t integer (e.g. torch.cuda.current_stream().cuda_stream) or None;
        create_options: fields of fredopt_create_options (index_width=...): fredopt_create_ex is called when given."""
        self._h = None
        self.n_rows, self.n_cols = int(n_rows), int(n_cols)

        def csr(M):
            rp, ci, vv = M
            nnz = int(ci.size if isinstance(ci, np.ndarray) else ci.numel())
            return _Csr(self.n_rows, self.n_cols, nnz, _ptr(rp, np.int64, self.n_rows + 1), _ptr(ci, np.int32),
                        _ptr(vv, np.float32, nnz))

        cD, cL = csr(D), csr(L)
        b = np.ascontiguousarray(np.asarray(bounds, dtype=np.float32).reshape(-1, 8))
        n_struct = b.shape[0]
        barr = (_Bounds * max(n_struct, 1))()
        for s in range(n_struct):
            barr[s] = _Bounds(*[float(t) for t in b[s]])
        h = C.c_void_p()
        if create_options:
            opt = _CreateOptions(struct_size=C.sizeof(_CreateOptions), **{k: int(v) for k, v in create_options.items()})
            rc = _lib.fredopt_create_ex(C.byref(cD), C.byref(cL), _ptr(voxel_labels, np.int32, self.n_rows), barr, n_struct,
                                        C.c_void_p(stream or 0), C.byref(opt), C.byref(h))
        else:
            rc = _lib.fredopt_create(C.byref(cD), C.byref(cL), _ptr(voxel_labels, np.int32, self.n_rows), barr, n_struct,
                                     C.c_void_p(stream or 0), C.byref(h))
        _check(rc, "fredopt_create")
        self._h = h

    def destroy(self):
        if self._h:
            _lib.fredopt_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # ---- state
    def set_weights(self, x):
        _check(_lib.fredopt_set_weights(self._h, _ptr(x, np.float32, self.n_cols)), "fredopt_set_weights")

    def get_weights(self, out):
        _check(_lib.fredopt_get_weights(self._h, _ptr(out, np.float32, self.n_cols)), "fredopt_get_weights")
        return out

    def set_weights_f64(self, x):
        _check(_lib.fredopt_set_weights_f64(self._h, _ptr(x, np.float64, self.n_cols)), "fredopt_set_weights_f64")

    def get_state(self):
        st = State()
        _check(_lib.fredopt_get_state(self._h, C.byref(st)), "fredopt_get_state")
        return st

    def set_state(self, st):
        _check(_lib.fredopt_set_state(self._h, C.byref(st)), "fredopt_set_state")

    def get_weights_f64(self, out):
        _check(_lib.fredopt_get_weights_f64(self._h, _ptr(out, np.float64, self.n_cols)), "fredopt_get_weights_f64")
        return out

    def set_voxel_bounds(self, field, values):
        """values: n_rows float32 (NaN = the structure's scalar), host or device, or None (remove the array)."""
        _check(_lib.fredopt_set_voxel_bounds(self._h, int(field), _ptr(values, np.float32, self.n_rows)), "fredopt_set_voxel_bounds")

    # ---- the four calls of north_star
    def dose_let(self, x, dose, letd):
        _check(_lib.fredopt_dose_let(self._h, _ptr(x, np.float32, self.n_cols), _ptr(dose, np.float32, self.n_rows),
                                     _ptr(letd, np.float32, self.n_rows)), "fredopt_dose_let")

    def iterate(self, n_iter, lam, beta0, a):
        _check(_lib.fredopt_iterate(self._h, int(n_iter), float(lam), float(beta0), float(a)), "fredopt_iterate")

    def iterate_host(self, n_iter, lam, beta0, a, x_in=None, x_out=None, stats=True):
        """set_weights(x_in), iterate, get_weights(x_out), stats as one call with one synchronisation; returns the stats or None."""
        s = Stats() if stats else None
        _check(_lib.fredopt_iterate_host(self._h, int(n_iter), float(lam), float(beta0), float(a), _ptr(x_in, np.float32, self.n_cols),
                                         _ptr(x_out, np.float32, self.n_cols), C.byref(s) if stats else None), "fredopt_iterate_host")
        return s.as_dict() if stats else None

    def proximity(self, x=None):
        p, n = C.c_double(0.0), C.c_int64(0)
        _check(_lib.fredopt_proximity(self._h, _ptr(x, np.float32, self.n_cols), C.byref(p), C.byref(n)),
               "fredopt_proximity")
        return p.value, n.value

    # ---- evaluation quantities (DVH / LVH / cDLVH, cDL30, Table 1)
    def structure_stats(self, quantity, label, x=None):
        mn, mean, mx, n = C.c_double(0.0), C.c_double(0.0), C.c_double(0.0), C.c_int64(0)
        _check(_lib.fredopt_structure_stats(self._h, _ptr(x, np.float32, self.n_cols), int(quantity), int(label), C.byref(mn),
                                            C.byref(mean), C.byref(mx), C.byref(n)), "fredopt_structure_stats")
        return mn.value, mean.value, mx.value, n.value

    def volume_histogram(self, quantity, label, n_bins, vmax, hist, x=None):
        _check(_lib.fredopt_volume_histogram(self._h, _ptr(x, np.float32, self.n_cols), int(quantity), int(label), int(n_bins),
                                             float(vmax), _ptr(hist, np.float32, n_bins)), "fredopt_volume_histogram")
        return hist

    def percentile_value(self, quantity, label, fraction, x=None):
        v = C.c_double(0.0)
        _check(_lib.fredopt_percentile_value(self._h, _ptr(x, np.float32, self.n_cols), int(quantity), int(label),
                                             float(fraction), C.byref(v)), "fredopt_percentile_value")
        return v.value

    def set_reduce(self, fn):
        """fn(device_pointer: int, n: int, cuda_stream: int) -> None must sum the n doubles at device_pointer over all ranks in
        place, ordered on cuda_stream (sharded plans; fredopt_set_reduce).  Exceptions are reported as a failed reduction."""
        def tramp(_ctx, buf, n, stream):
            try:
                fn(int(buf), int(n), int(stream or 0))
                return 0
            except Exception:                                    # never let an exception cross the C boundary
                import traceback
                traceback.print_exc()
                return 1
        self._reduce_cb = REDUCE_FN(tramp)                         # keep the callback object alive as long as the plan
        _check(_lib.fredopt_set_reduce(self._h, self._reduce_cb, None), "fredopt_set_reduce")

    # ---- options, stats
    def set_option(self, key, value):
        _check(_lib.fredopt_set_option(self._h, int(key), float(value)), "fredopt_set_option")

    def stats(self):
        s = Stats()
        _check(_lib.fredopt_get_stats(self._h, C.byref(s)), "fredopt_get_stats")
        return s.as_dict()

    # ---- per-pass exports
    def spmv_forward(self, rows, x, d, l):
        _check(_lib.fredopt_spmv_forward(self._h, int(rows), _ptr(x, np.float32, self.n_cols),
                                         _ptr(d, np.float32, self.n_rows), _ptr(l, np.float32, self.n_rows)),
               "fredopt_spmv_forward")

    def spmv_transpose(self, rows, u, v, out):
        _check(_lib.fredopt_spmv_transpose(self._h, int(rows), _ptr(u, np.float32, self.n_rows),
                                           _ptr(v, np.float32, self.n_rows), _ptr(out, np.float32, self.n_cols)),
               "fredopt_spmv_transpose")

    def pass_times(self):
        ms = (C.c_double * N_PASSES)()
        n = (C.c_int64 * N_PASSES)()
        _check(_lib.fredopt_get_pass_times(self._h, ms, n), "fredopt_get_pass_times")
        return {PASS_NAMES[i]: (ms[i], n[i]) for i in range(N_PASSES)}

    def pass_bytes(self):
        b = (C.c_int64 * N_PASSES)()
        _check(_lib.fredopt_get_pass_bytes(self._h, b), "fredopt_get_pass_bytes")
        return {PASS_NAMES[i]: b[i] for i in range(N_PASSES)}

    def pass_bytes_timed(self):
        b = (C.c_int64 * N_PASSES)()
        _check(_lib.fredopt_get_pass_bytes_timed(self._h, b), "fredopt_get_pass_bytes_timed")
        return {PASS_NAMES[i]: b[i] for i in range(N_PASSES)}

    def launch_count(self):
        return int(_lib.fredopt_launch_count(self._h))

    def stream_read(self, device_buf, nbytes, reps=1):
        _check(_lib.fredopt_stream_read(self._h, _ptr(device_buf), int(nbytes), int(reps)), "fredopt_stream_read")


NO_ALLOC_MAX_BINS = 4096      # FREDOPT_NO_ALLOC_MAX_BINS


def no_alloc_setup():
    """Look up the fixed scratch of volume_histogram_no_alloc on the current device (before a stream capture begins)."""
    _check(_lib.fredopt_no_alloc_setup(), "fredopt_no_alloc_setup")


def volume_histogram_no_alloc(values, labels, label, n_bins, vmax, hist, n_in_structure=None, stream=None):
    """fredopt_volume_histogram_no_alloc: DEVICE tensors only (values float32 [n], labels int32 [n] or None, hist float32
    [n_bins], n_in_structure int64 [1] or None); asynchronous on `stream` (a cudaStream_t as int; None = default stream)."""
    n = values.numel()
    if hist.numel() < n_bins:
        raise ValueError(f"hist holds {hist.numel()} floats, n_bins = {n_bins}")
    rc = _lib.fredopt_volume_histogram_no_alloc(_ptr(values, np.float32, n), _ptr(labels, np.int32, n), n, int(label), int(n_bins),
                                                float(vmax), _ptr(hist, np.float32), _ptr(n_in_structure, np.int64, 1), stream)
    if rc != OK:
        raise FredoptError(rc, "fredopt_volume_histogram_no_alloc [" + _lib.fredopt_last_cuda_error().decode() + "]")
    return hist


def shard_range(row_ptr, voxel_labels, rank, world):
    """fredopt_shard_range on host numpy arrays: the voxel range [begin, end) of shard `rank` of `world` (pure host code)."""
    rp = np.ascontiguousarray(row_ptr, np.int64); lab = np.ascontiguousarray(voxel_labels, np.int32)
    b, e = C.c_int64(0), C.c_int64(0)
    _check(_lib.fredopt_shard_range(rp.ctypes.data, lab.ctypes.data, len(lab), int(rank), int(world), C.byref(b), C.byref(e)),
           "fredopt_shard_range")
    return b.value, e.value


class DeviceDoubles:
    """A view of n doubles of device memory for torch.as_tensor(view, device="cuda") (CUDA array interface, zero copy): how a
    reduction callback hands the library's buffer to torch.distributed."""

    def __init__(self, ptr, n):
        self.__cuda_array_interface__ = {"shape": (int(n),), "typestr": "<f8", "data": (int(ptr), False), "version": 3}


def from_plan(plan, stream=None, **create_options) -> Plan:
    """Plan over a plangen.Plan; tensors are passed where they live (host or device)."""
    return Plan(plan.n_rows, plan.n_cols, (plan.row_ptr, plan.col_idx, plan.val_D),
                (plan.row_ptr, plan.col_idx, plan.val_L), plan.labels, plan.bounds, stream=stream, **create_options)
