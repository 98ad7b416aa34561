"""Thin ctypes binding over libspmv_b200.so (include/spmv_b200.h): argument marshalling
only -- every step of the path runs in the library's CUDA kernels.  PyTorch is used for
device memory and streams, nothing else.  There is no fallback: if the shared library is
missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libspmv_b200.so")
_lib = None

SPMV_OK = 0
STATUS_NAMES = ["SPMV_OK", "SPMV_ERR_INVALID_ARG", "SPMV_ERR_INVALID_MATRIX", "SPMV_ERR_UNSUPPORTED",
                "SPMV_ERR_ALLOC", "SPMV_ERR_CUDA", "SPMV_ERR_VERIFY_FAILED", "SPMV_ERR_INTERNAL"]

EXPORTS = ["spmv_create", "spmv_tune", "spmv_apply", "spmv_apply_host", "spmv_apply_host_batch", "spmv_apply_batch",
           "spmv_tune_batch", "spmv_select", "spmv_list_variants", "spmv_get_info",
           "spmv_format_download", "spmv_destroy", "spmv_measure_ceiling", "spmv_update_values", "spmv_cg", "spmv_jacobi", "spmv_status_string",
           "spmv_last_error", "spmv_version", "spmv_clear_cache", "spmv_graph_create", "spmv_graph_launch",
           "spmv_graph_destroy", "spmv_partition_rows", "spmv_external_columns", "spmv_gather", "spmv_scatter",
           "spmv_apply_rows", "spmv_merge_apply_noalloc", "spmv_merge_noalloc_max_path"]


class SpmvError(RuntimeError):
    def __init__(self, status: int, where: str, text: str = ""):
        self.status = status
        name = STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else str(status)
        super().__init__(f"{where}: {name}" + (f" ({text})" if text else ""))


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class Allocator(C.Structure):
    _fields_ = [("alloc", ALLOC_FN), ("free", FREE_FN), ("ctx", C.c_void_p)]


class Info(C.Structure):
    _fields_ = [("rows", C.c_int64), ("cols", C.c_int64), ("nnz", C.c_int64),
                ("min_row_len", C.c_int32), ("max_row_len", C.c_int32),
                ("mean_row_len", C.c_double), ("var_row_len", C.c_double),
                ("len_hist", C.c_int64 * 32), ("bandwidth", C.c_int64),
                ("cols_sorted", C.c_int32), ("block3_full", C.c_int32), ("n_blocks3", C.c_int64),
                ("sig_row_ptr", C.c_uint64), ("sig_col_idx", C.c_uint64),
                ("tuned", C.c_int32), ("sm_count", C.c_int32), ("l2_bytes", C.c_int64),
                ("format_bytes", C.c_int64), ("owned_bytes", C.c_int64),
                ("variant", C.c_char * 128), ("device_name", C.c_char * 64)]


class TuneOpts(C.Structure):
    _fields_ = [("has_scalars", C.c_int32), ("alpha", C.c_double), ("beta", C.c_double),
                ("d_x_probe", C.c_void_p), ("d_y0_probe", C.c_void_p),
                ("d_y_ref", C.c_void_p), ("d_scale", C.c_void_p),
                ("tolerance", C.c_double), ("warmup", C.c_int32), ("reps", C.c_int32),
                ("min_batch_ms", C.c_double), ("time_budget_s", C.c_double),
                ("variant_filter", C.c_char_p), ("n_carveouts", C.c_int32), ("carveouts", C.c_int32 * 8),
                ("use_cache", C.c_int32), ("cache_path", C.c_char_p), ("fault_inject", C.c_char_p),
                ("seed", C.c_uint64), ("flush_l2", C.c_int32), ("search", C.c_int32), ("stream", C.c_void_p)]


class CgOpts(C.Structure):
    _fields_ = [("tol", C.c_double), ("max_iters", C.c_int32), ("check_every", C.c_int32), ("no_graph", C.c_int32),
                ("no_fused", C.c_int32), ("no_fused_dot", C.c_int32), ("tune_loop", C.c_int32)]


class CgResult(C.Structure):
    _fields_ = [("iters", C.c_int32), ("converged", C.c_int32), ("breakdown", C.c_int32),
                ("iterations_launched", C.c_int32), ("graph_replays", C.c_int32), ("fused", C.c_int32),
                ("fused_dot", C.c_int32), ("kernels_per_iteration", C.c_int32), ("loop_variant", C.c_char * 128),
                ("rel_residual", C.c_double), ("device_seconds", C.c_double), ("wall_seconds", C.c_double)]


class JacobiOpts(C.Structure):
    _fields_ = [("omega", C.c_double), ("tol", C.c_double), ("max_iters", C.c_int32), ("check_every", C.c_int32),
                ("no_graph", C.c_int32), ("no_fused", C.c_int32)]


class JacobiResult(C.Structure):
    _fields_ = [("iters", C.c_int32), ("converged", C.c_int32), ("zero_diagonal", C.c_int32),
                ("iterations_launched", C.c_int32), ("graph_replays", C.c_int32), ("kernels_per_iteration", C.c_int32),
                ("fused_step", C.c_int32), ("rel_residual", C.c_double), ("device_seconds", C.c_double), ("wall_seconds", C.c_double)]


class TuneReport(C.Structure):
    _fields_ = [("winner", C.c_char * 128), ("winner_us", C.c_double), ("default_us", C.c_double),
                ("n_enumerated", C.c_int32), ("n_pruned_structural", C.c_int32),
                ("n_pruned_slow", C.c_int32), ("n_rejected", C.c_int32), ("n_timed", C.c_int32),
                ("tune_seconds", C.c_double), ("cache_hit", C.c_int32),
                ("runner_up", C.c_char * 128), ("runner_up_us", C.c_double),
                ("log_buf", C.c_void_p), ("log_cap", C.c_size_t), ("log_len", C.c_size_t)]


def lib():
    """Loads libspmv_b200.so; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1309_1894_b200.build` "
                           "(there is no CPU or PyTorch fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i64, i32, dbl = C.c_void_p, C.c_int64, C.c_int32, C.c_double
    L.spmv_create.argtypes = [C.POINTER(vp), i64, i64, i64, vp, vp, vp, C.POINTER(Allocator), vp]
    L.spmv_tune.argtypes = [vp, C.POINTER(TuneOpts), C.POINTER(TuneReport)]
    L.spmv_apply.argtypes = [vp, dbl, vp, dbl, vp, vp]
    L.spmv_apply_host.argtypes = [vp, dbl, vp, dbl, vp, vp]
    L.spmv_apply_host_batch.argtypes = [i32, C.POINTER(vp), C.POINTER(dbl), C.POINTER(vp), C.POINTER(dbl), C.POINTER(vp), vp]
    L.spmv_apply_batch.argtypes = [i32, C.POINTER(vp), C.POINTER(dbl), C.POINTER(vp), C.POINTER(dbl),
                                   C.POINTER(vp), C.POINTER(vp), i32]
    L.spmv_tune_batch.argtypes = [i32, C.POINTER(vp), C.POINTER(dbl), C.POINTER(vp), C.POINTER(dbl),
                                  C.POINTER(vp), C.POINTER(vp), i32, C.POINTER(i32), C.POINTER(dbl)]
    L.spmv_select.argtypes = [vp, C.c_char_p, vp]
    L.spmv_list_variants.argtypes = [vp, C.c_char_p, C.c_size_t, C.POINTER(C.c_size_t)]
    L.spmv_get_info.argtypes = [vp, C.POINTER(Info)]
    L.spmv_format_download.argtypes = [vp, C.c_char_p, vp, C.c_size_t, C.POINTER(C.c_size_t), vp]
    L.spmv_destroy.argtypes = [vp]
    L.spmv_measure_ceiling.argtypes = [i32, C.c_size_t, i32, vp, C.POINTER(dbl)]
    L.spmv_update_values.argtypes = [vp, vp, C.POINTER(i32), vp]
    L.spmv_cg.argtypes = [vp, vp, vp, C.POINTER(CgOpts), C.POINTER(CgResult), vp]
    L.spmv_jacobi.argtypes = [vp, vp, vp, C.POINTER(JacobiOpts), C.POINTER(JacobiResult), vp]
    L.spmv_graph_create.argtypes = [vp, dbl, vp, dbl, vp, i32, C.POINTER(vp)]
    L.spmv_graph_launch.argtypes = [vp, vp]
    L.spmv_graph_destroy.argtypes = [vp]
    L.spmv_partition_rows.argtypes = [i64, vp, i32, i64, vp]
    L.spmv_external_columns.argtypes = [vp, i64, i64, vp, i64, C.POINTER(i64), C.POINTER(i64), C.POINTER(i64), vp]
    L.spmv_gather.argtypes = [i64, vp, vp, vp, vp]
    L.spmv_scatter.argtypes = [i64, vp, vp, vp, vp]
    L.spmv_apply_rows.argtypes = [vp, dbl, vp, dbl, vp, i64, i64, C.POINTER(i64), vp]
    L.spmv_merge_apply_noalloc.argtypes = [i64, i64, i64, vp, vp, vp, dbl, vp, dbl, vp, vp]
    L.spmv_merge_apply_noalloc.restype = C.c_int
    L.spmv_merge_noalloc_max_path.argtypes = []
    L.spmv_merge_noalloc_max_path.restype = i64
    for n in ("spmv_create", "spmv_tune", "spmv_apply", "spmv_apply_host", "spmv_apply_host_batch", "spmv_apply_batch",
              "spmv_tune_batch", "spmv_select", "spmv_list_variants", "spmv_get_info",
              "spmv_format_download", "spmv_destroy", "spmv_measure_ceiling", "spmv_update_values", "spmv_cg", "spmv_jacobi",
              "spmv_graph_create", "spmv_graph_launch", "spmv_graph_destroy", "spmv_partition_rows",
              "spmv_external_columns", "spmv_gather", "spmv_scatter", "spmv_apply_rows"):
        getattr(L, n).restype = C.c_int
    L.spmv_status_string.argtypes = [C.c_int]
    L.spmv_status_string.restype = C.c_char_p
    L.spmv_last_error.restype = C.c_char_p
    L.spmv_version.restype = C.c_char_p
    L.spmv_clear_cache.restype = None
    _lib = L
    return L


def _check(st: int, where: str):
    if st != SPMV_OK:
        raise SpmvError(st, where, lib().spmv_last_error().decode(errors="replace"))


def _stream_ptr(stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


_fast = False


def _fast_apply():
    """paper_1309_1894_b200/_spmvfast (built by build.py next to the library), or None: then ctypes marshals."""
    global _fast
    if _fast is False:
        try:
            lib()                                   # libspmv_b200.so first: _spmvfast links against it
            from . import _spmvfast
            _fast = _spmvfast.apply
        except Exception:
            _fast = None
    return _fast


def _getraw(device_index):
    """cudaStream_t of torch's current stream as an int (the fast private accessor when torch has it)."""
    import torch
    try:
        return torch._C._cuda_getCurrentRawStream(device_index)
    except AttributeError:
        return torch.cuda.current_stream(device_index).cuda_stream


def _dptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


# torch caching allocator behind the spmv_allocator_t callbacks (device memory plumbing only)
def _torch_allocator():
    import torch

    def _alloc(nbytes, stream, ctx):
        try:
            return torch.cuda.caching_allocator_alloc(int(nbytes), stream=int(stream or 0))
        except Exception:
            return 0

    def _free(ptr, ctx):
        torch.cuda.caching_allocator_delete(int(ptr))

    a = Allocator(ALLOC_FN(_alloc), FREE_FN(_free), None)
    return a


class SpMV:
    """Handle wrapper.  row_ptr/col_idx (int32) and val (float64) are CUDA torch tensors that
    this object keeps alive (the C handle borrows them)."""

    def __init__(self, rows, cols, row_ptr, col_idx, val, *, use_torch_allocator=True, stream=None, allocator=None):
        import torch
        assert row_ptr.is_cuda and row_ptr.dtype == torch.int32 and row_ptr.is_contiguous()
        assert col_idx.dtype == torch.int32 and val.dtype == torch.float64
        assert col_idx.is_contiguous() and val.is_contiguous()
        self._keep = (row_ptr, col_idx, val)
        # allocator: a ready-made Allocator struct (spmv_allocator_t callbacks; the tests pass a failing one)
        self._alloc = allocator if allocator is not None else (_torch_allocator() if use_torch_allocator else None)
        self.rows, self.cols, self.nnz = int(rows), int(cols), int(val.numel())
        h = C.c_void_p(0)
        st = lib().spmv_create(C.byref(h), self.rows, self.cols, self.nnz, _dptr(row_ptr),
                               _dptr(col_idx) if self.nnz else C.c_void_p(col_idx.data_ptr() or 0),
                               _dptr(val) if self.nnz else C.c_void_p(val.data_ptr() or 0),
                               C.byref(self._alloc) if self._alloc is not None else None, _stream_ptr(stream))
        _check(st, "spmv_create")
        self.h = h
        self._hv = h.value
        self._apply = lib().spmv_apply
        self._fast = _fast_apply()
        self._dev = row_ptr.device.index

    @classmethod
    def from_csr(cls, A, device="cuda:0", **kw):
        """A: workloads.CSR (numpy).  Copies the arrays to the device."""
        import torch
        rp = torch.from_numpy(np.ascontiguousarray(A.row_ptr, dtype=np.int32)).to(device)
        ci = torch.from_numpy(np.ascontiguousarray(A.col_idx, dtype=np.int32)).to(device)
        va = torch.from_numpy(np.ascontiguousarray(A.val, dtype=np.float64)).to(device)
        return cls(A.rows, A.cols, rp, ci, va, **kw)

    def close(self):
        if getattr(self, "h", None) is not None and self.h.value:
            _check(lib().spmv_destroy(self.h), "spmv_destroy")
            self.h = C.c_void_p(0)
            self._hv = 0

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def info(self) -> Info:
        out = Info()
        _check(lib().spmv_get_info(self.h, C.byref(out)), "spmv_get_info")
        return out

    @property
    def variant(self) -> str:
        return self.info().variant.decode()

    def select(self, desc: str, stream=None):
        _check(lib().spmv_select(self.h, desc.encode(), _stream_ptr(stream)), f"spmv_select({desc})")

    def variants(self) -> list[str]:
        n = C.c_size_t(0)
        _check(lib().spmv_list_variants(self.h, None, 0, C.byref(n)), "spmv_list_variants")
        buf = C.create_string_buffer(n.value + 1)
        _check(lib().spmv_list_variants(self.h, buf, n.value + 1, C.byref(n)), "spmv_list_variants")
        return [l for l in buf.value.decode().split("\n") if l]

    def apply(self, alpha, x, beta, y, stream=None):
        """y = alpha*A*x + beta*y on the device, asynchronous on the (current) stream.
        Kept lean: for small matrices the call overhead is what a user sees (a ctypes call costs ~0.7 us,
        the CUDA launch ~2 us; spmv_graph_create amortises both over k applies)."""
        if x.numel() != self.cols or y.numel() != self.rows or not (x.is_cuda and y.is_cuda):
            raise ValueError("spmv_apply: x must hold cols and y rows CUDA float64 entries")
        s = _getraw(self._dev) if stream is None else stream.cuda_stream
        if self._fast is not None:              # CPython fast-call entry (csrc/pyfast.c): same C function, ~0.7 us less
            st = self._fast(self._hv, float(alpha), x.data_ptr(), float(beta), y.data_ptr(), s)
        else:
            st = self._apply(self.h, alpha, x.data_ptr(), beta, y.data_ptr(), s)
        if st != SPMV_OK:
            _check(st, "spmv_apply")
        return y

    def update_values(self, val, stream=None) -> bool:
        """New values on the same pattern (CUDA float64 tensor, kept alive here).  Returns True if the
        selected variant no longer applied and the handle fell back to another one."""
        assert val.is_cuda and val.is_contiguous() and val.numel() == self.nnz
        fb = C.c_int32(0)
        _check(lib().spmv_update_values(self.h, _dptr(val), C.byref(fb), _stream_ptr(stream)), "spmv_update_values")
        self._keep = (self._keep[0], self._keep[1], val)
        return bool(fb.value)

    def cg(self, b, x, *, tol=1e-10, max_iters=1000, check_every=8, no_graph=False, no_fused=False,
           no_fused_dot=False, tune_loop=False, stream=None) -> dict:
        """Conjugate gradients with the selected variant (spmv_cg).  x: initial guess in, solution out."""
        assert b.is_cuda and x.is_cuda and b.numel() == self.rows and x.numel() == self.rows
        o = CgOpts(float(tol), int(max_iters) if max_iters > 0 else -1, int(check_every), int(bool(no_graph)),
                   int(bool(no_fused)), int(bool(no_fused_dot)), int(bool(tune_loop)))
        r = CgResult()
        _check(lib().spmv_cg(self.h, _dptr(b), _dptr(x), C.byref(o), C.byref(r), _stream_ptr(stream)), "spmv_cg")
        out = {k: getattr(r, k) for k, _ in CgResult._fields_}
        out["loop_variant"] = out["loop_variant"].decode()
        return out

    def jacobi(self, b, x, *, omega=1.0, tol=1e-10, max_iters=1000, check_every=8, no_graph=False, no_fused=False,
               stream=None) -> dict:
        """Weighted Jacobi with the selected variant (spmv_jacobi).  x: initial guess in, iterate out."""
        assert b.is_cuda and x.is_cuda and b.numel() == self.rows and x.numel() == self.rows
        o = JacobiOpts(float(omega), float(tol), int(max_iters) if max_iters > 0 else -1, int(check_every),
                       int(bool(no_graph)), int(bool(no_fused)))
        r = JacobiResult()
        _check(lib().spmv_jacobi(self.h, _dptr(b), _dptr(x), C.byref(o), C.byref(r), _stream_ptr(stream)), "spmv_jacobi")
        return {k: getattr(r, k) for k, _ in JacobiResult._fields_}

    def apply_rows(self, alpha, x, beta, y, row_begin: int, row_end: int, stream=None):
        """spmv_apply restricted to rows [row_begin, row_end); x, y are the whole vectors."""
        al = C.c_int64(0)
        _check(lib().spmv_apply_rows(self.h, float(alpha), _dptr(x), float(beta), _dptr(y), int(row_begin), int(row_end),
                                     C.byref(al), _stream_ptr(stream)), "spmv_apply_rows")
        return y

    def range_align(self) -> int:
        """Row alignment of the selected variant's row-range form (0: it has none)."""
        al = C.c_int64(0)
        _check(lib().spmv_apply_rows(self.h, 1.0, None, 0.0, None, 0, 0, C.byref(al), None), "spmv_apply_rows")
        return int(al.value)

    def external_columns(self, own_lo: int, own_hi: int):
        """(sorted int32 array of the columns referenced outside [own_lo, own_hi), (interior_lo, interior_hi))."""
        n, a, b = C.c_int64(0), C.c_int64(0), C.c_int64(0)
        _check(lib().spmv_external_columns(self.h, int(own_lo), int(own_hi), None, 0, C.byref(n), C.byref(a), C.byref(b),
                                           _stream_ptr()), "spmv_external_columns")
        out = np.empty(n.value, dtype=np.int32)
        if n.value:
            _check(lib().spmv_external_columns(self.h, int(own_lo), int(own_hi), C.c_void_p(out.ctypes.data), n.value,
                                               C.byref(n), C.byref(a), C.byref(b), _stream_ptr()), "spmv_external_columns")
        return out, (int(a.value), int(b.value))

    def graph(self, alpha, x, beta, y, k: int) -> "Graph":
        """k back-to-back applies captured into one CUDA graph (spmv_graph_create); x, y are baked in."""
        assert x.is_cuda and y.is_cuda and x.numel() == self.cols and y.numel() == self.rows
        g = C.c_void_p(0)
        _check(lib().spmv_graph_create(self.h, float(alpha), _dptr(x), float(beta), _dptr(y), int(k), C.byref(g)),
               "spmv_graph_create")
        return Graph(g, k, (x, y, self))

    def apply_host(self, alpha, x_host, beta, y_host, stream=None):
        """Host-buffer form: x_host/y_host are CPU tensors or numpy arrays (pinned is faster)."""
        xp = x_host.data_ptr() if hasattr(x_host, "data_ptr") else x_host.ctypes.data
        yp = y_host.data_ptr() if hasattr(y_host, "data_ptr") else y_host.ctypes.data
        _check(lib().spmv_apply_host(self.h, float(alpha), C.c_void_p(xp), float(beta), C.c_void_p(yp),
                                     _stream_ptr(stream)), "spmv_apply_host")
        return y_host

    def tune(self, *, alpha=1.0, beta=0.0, x=None, y0=None, y_ref=None, scale=None, tolerance=0.0,
             warmup=0, reps=0, min_batch_ms=0.0, time_budget_s=0.0, variant_filter=None,
             carveouts=None, use_cache=0, cache_path=None, fault_inject=None, seed=0, flush_l2=False,
             stream=None, log_bytes=1 << 20, search=0) -> dict:
        o = TuneOpts()
        o.has_scalars, o.alpha, o.beta = 1, float(alpha), float(beta)
        o.d_x_probe, o.d_y0_probe = _dptr(x), _dptr(y0)
        o.d_y_ref, o.d_scale = _dptr(y_ref), _dptr(scale)
        o.tolerance, o.warmup, o.reps = float(tolerance), int(warmup), int(reps)
        o.min_batch_ms, o.time_budget_s = float(min_batch_ms), float(time_budget_s)
        o.variant_filter = variant_filter.encode() if variant_filter else None
        if carveouts:
            o.n_carveouts = len(carveouts)
            for i, c in enumerate(carveouts[:8]):
                o.carveouts[i] = int(c)
        o.use_cache = int(use_cache)
        o.cache_path = cache_path.encode() if cache_path else None
        o.fault_inject = fault_inject.encode() if fault_inject else None
        o.seed, o.flush_l2, o.stream = int(seed), int(bool(flush_l2)), _stream_ptr(stream)
        o.search = int(search)
        rep = TuneReport()
        logbuf = C.create_string_buffer(log_bytes) if log_bytes else None
        if logbuf is not None:
            rep.log_buf, rep.log_cap = C.cast(logbuf, C.c_void_p), log_bytes
        st = lib().spmv_tune(self.h, C.byref(o), C.byref(rep))
        log = logbuf.value.decode() if logbuf is not None else ""
        out = {"status": st, "winner": rep.winner.decode(), "winner_us": rep.winner_us,
               "default_us": rep.default_us, "n_enumerated": rep.n_enumerated,
               "n_pruned_structural": rep.n_pruned_structural, "n_pruned_slow": rep.n_pruned_slow,
               "n_rejected": rep.n_rejected, "n_timed": rep.n_timed, "tune_seconds": rep.tune_seconds,
               "cache_hit": bool(rep.cache_hit), "runner_up": rep.runner_up.decode(),
               "runner_up_us": rep.runner_up_us,
               "log": [l.split() for l in log.split("\n") if l]}
        if st != SPMV_OK:
            err = SpmvError(st, "spmv_tune", lib().spmv_last_error().decode(errors="replace"))
            err.report = out
            raise err
        return out

    def download(self, name: str, dtype) -> np.ndarray:
        n = C.c_size_t(0)
        _check(lib().spmv_format_download(self.h, name.encode(), None, 0, C.byref(n), _stream_ptr()),
               f"spmv_format_download({name})")
        out = np.empty(n.value // np.dtype(dtype).itemsize, dtype=dtype)
        if n.value:
            _check(lib().spmv_format_download(self.h, name.encode(), C.c_void_p(out.ctypes.data), n.value,
                                              C.byref(n), _stream_ptr()), f"spmv_format_download({name})")
        return out


class Graph:
    """spmv_graph_t wrapper; keeps the vectors and the handle it was captured from alive."""

    def __init__(self, g, k, keep):
        self.g, self.k, self._keep = g, k, keep

    def launch(self, stream=None):
        _check(lib().spmv_graph_launch(self.g, _stream_ptr(stream)), "spmv_graph_launch")

    def close(self):
        if self.g is not None and self.g.value:
            _check(lib().spmv_graph_destroy(self.g), "spmv_graph_destroy")
            self.g = C.c_void_p(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def apply_batch(handles, alphas, xs, betas, ys, streams):
    """spmv_apply_batch: handle i on streams[i % len(streams)]; no synchronisation."""
    n = len(handles)
    vp, dbl = C.c_void_p, C.c_double
    hs = (vp * n)(*[h.h for h in handles])
    al = (dbl * n)(*[float(a) for a in alphas])
    be = (dbl * n)(*[float(b) for b in betas])
    dx = (vp * n)(*[x.data_ptr() for x in xs])
    dy = (vp * n)(*[y.data_ptr() for y in ys])
    ss = (vp * len(streams))(*[s.cuda_stream for s in streams])
    _check(lib().spmv_apply_batch(n, hs, al, dx, be, dy, ss, len(streams)), "spmv_apply_batch")


def apply_host_batch(handles, alphas, xs_host, betas, ys_host, stream=None):
    """spmv_apply_host_batch: host-vector applies of n different handles, enqueued together, one synchronise."""
    n = len(handles)
    ptr = lambda a: a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data
    hs = (C.c_void_p * n)(*[h.h for h in handles])
    al = (C.c_double * n)(*[float(a) for a in alphas])
    be = (C.c_double * n)(*[float(b) for b in betas])
    xp = (C.c_void_p * n)(*[ptr(x) for x in xs_host])
    yp = (C.c_void_p * n)(*[ptr(y) for y in ys_host])
    _check(lib().spmv_apply_host_batch(n, hs, al, xp, be, yp, _stream_ptr(stream)), "spmv_apply_host_batch")


def tune_batch(handles, alphas, xs, betas, ys, streams):
    """spmv_tune_batch: returns (best stream count, {count: microseconds per batch})."""
    n = len(handles)
    vp, dbl = C.c_void_p, C.c_double
    hs = (vp * n)(*[h.h for h in handles])
    al = (dbl * n)(*[float(a) for a in alphas])
    be = (dbl * n)(*[float(b) for b in betas])
    dx = (vp * n)(*[x.data_ptr() for x in xs])
    dy = (vp * n)(*[y.data_ptr() for y in ys])
    ss = (vp * len(streams))(*[s.cuda_stream for s in streams])
    best = C.c_int32(0)
    us = (dbl * 8)()
    _check(lib().spmv_tune_batch(n, hs, al, dx, be, dy, ss, len(streams), C.byref(best), us), "spmv_tune_batch")
    counts, c, i = {}, 1, 0
    while c <= len(streams):
        counts[c] = us[i]
        c *= 2
        i += 1
    return best.value, counts


def partition_rows(row_ptr: np.ndarray, nparts: int, align: int = 1) -> np.ndarray:
    """spmv_partition_rows: nnz-balanced contiguous row blocks; returns int64 bounds [nparts + 1]."""
    rp = np.ascontiguousarray(row_ptr, dtype=np.int32)
    out = np.zeros(nparts + 1, dtype=np.int64)
    _check(lib().spmv_partition_rows(rp.size - 1, C.c_void_p(rp.ctypes.data), int(nparts), int(align),
                                     C.c_void_p(out.ctypes.data)), "spmv_partition_rows")
    return out


def gather(idx, src, dst, stream=None):
    """dst[i] = src[idx[i]] (CUDA tensors; idx int32): the library's pack kernel."""
    assert idx.is_cuda and src.is_cuda and dst.is_cuda and dst.numel() >= idx.numel()
    _check(lib().spmv_gather(idx.numel(), _dptr(idx), _dptr(src), _dptr(dst), _stream_ptr(stream)), "spmv_gather")


def scatter(idx, src, dst, stream=None):
    """dst[idx[i]] = src[i] (CUDA tensors; idx int32): the library's unpack kernel."""
    assert idx.is_cuda and src.is_cuda and dst.is_cuda and src.numel() >= idx.numel()
    _check(lib().spmv_scatter(idx.numel(), _dptr(idx), _dptr(src), _dptr(dst), _stream_ptr(stream)), "spmv_scatter")


def merge_apply_noalloc(rows, cols, row_ptr, col_idx, val, alpha, x, beta, y, stream=None):
    """spmv_merge_apply_noalloc: y = alpha*A*x + beta*y by the merge-path kernels, straight from CSR arrays that are
    already CUDA tensors (row_ptr / col_idx int32, val / x / y float64), for callers that must not allocate device
    memory where they need the product -- their memory pool owns the whole GPU, or they sit in a loop that cannot
    take the device-wide stall of cudaMalloc / cudaFree.  This wrapper allocates nothing either: it passes pointers.
    The kernels' scratch is a fixed array inside the library, shared by every call on the GPU: calls that may
    overlap (two streams, two threads) must be ordered by the caller.  rows + nnz <= merge_noalloc_max_path().
    Make the first call on each device during set-up (it resolves the array's device address)."""
    nnz = int(val.numel())
    for t in (row_ptr, col_idx, val, x, y):
        assert t.is_cuda and t.is_contiguous()
    assert row_ptr.numel() == rows + 1 and col_idx.numel() == nnz and x.numel() >= cols and y.numel() >= rows
    _check(lib().spmv_merge_apply_noalloc(int(rows), int(cols), nnz, _dptr(row_ptr), _dptr(col_idx), _dptr(val),
                                          float(alpha), _dptr(x), float(beta), _dptr(y), _stream_ptr(stream)),
           "spmv_merge_apply_noalloc")


def merge_noalloc_max_path() -> int:
    """Largest rows + nnz spmv_merge_apply_noalloc accepts (what its built-in scratch array can serve)."""
    return int(lib().spmv_merge_noalloc_max_path())


def measure_ceiling(kind: int, nbytes: int = 1 << 30, reps: int = 10) -> float:
    out = C.c_double(0.0)
    _check(lib().spmv_measure_ceiling(kind, nbytes, reps, _stream_ptr(), C.byref(out)), "spmv_measure_ceiling")
    return out.value


def clear_cache():
    lib().spmv_clear_cache()


def version() -> str:
    return lib().spmv_version().decode()
