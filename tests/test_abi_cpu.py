"""CPU-side checks of the boundary: the shared library builds, loads and exports every symbol
include/spmv_b200.h declares; error paths that need no GPU return codes, never abort."""
import ctypes
import os
import re

import pytest

from paper_1309_1894_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    build.build()
    return binding.lib()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "spmv_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(spmv_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(L):
    names = _declared_symbols()
    assert len(names) >= 16
    for n in names:
        assert hasattr(L, n), n
    assert sorted(binding.EXPORTS) == names


def test_status_strings_and_version(L):
    assert L.spmv_status_string(0) == b"SPMV_OK"
    assert L.spmv_status_string(6) == b"SPMV_ERR_VERIFY_FAILED"
    assert L.spmv_status_string(99) == b"SPMV_ERR_UNKNOWN"
    assert binding.version() == "0.1.0"


def test_null_and_bad_arguments_return_codes(L):
    h = ctypes.c_void_p(0)
    # NULL out pointer / negative sizes / NULL row_ptr
    assert L.spmv_create(None, 1, 1, 0, ctypes.c_void_p(8), None, None, None, None) == 1
    assert L.spmv_create(ctypes.byref(h), -1, 1, 0, ctypes.c_void_p(8), None, None, None, None) == 1
    assert L.spmv_create(ctypes.byref(h), 1, 1, 0, None, None, None, None, None) == 1
    assert L.spmv_create(ctypes.byref(h), 1, 1, 5, ctypes.c_void_p(8), None, None, None, None) == 1
    # over the int32 limits
    assert L.spmv_create(ctypes.byref(h), 1 << 31, 1, 0, ctypes.c_void_p(8), None, None, None, None) == 3
    assert h.value is None
    # NULL / never-created handles
    assert L.spmv_destroy(None) == 1
    assert L.spmv_destroy(ctypes.c_void_p(0x1234)) == 1
    assert L.spmv_apply(None, 1.0, None, 0.0, None, None) == 1
    assert L.spmv_tune(None, None, None) == 1
    assert L.spmv_select(None, b"default", None) == 1
    assert L.spmv_get_info(None, None) == 1
    L.spmv_clear_cache()
    # round-2 entry points: graphs, row ranges, sharding helpers
    g = ctypes.c_void_p(0)
    assert L.spmv_graph_create(None, 1.0, None, 0.0, None, 4, ctypes.byref(g)) == 1 and not g.value
    assert L.spmv_graph_launch(None, None) == 1 and L.spmv_graph_destroy(None) == 1
    assert L.spmv_apply_rows(None, 1.0, None, 0.0, None, 0, 0, None, None) == 1
    assert L.spmv_apply_host(None, 1.0, None, 0.0, None, None) == 1
    assert L.spmv_apply_host_batch(2, None, None, None, None, None, None) == 1 and L.spmv_apply_host_batch(-1, None, None, None, None, None, None) == 1
    assert L.spmv_gather(-1, None, None, None, None) == 1 and L.spmv_gather(0, None, None, None, None) == 0
    assert L.spmv_scatter(3, None, None, None, None) == 1
    assert L.spmv_external_columns(None, 0, 0, None, 0, None, None, None, None) == 1
    assert L.spmv_partition_rows(4, None, 2, 1, None) == 1
    assert L.spmv_cg(None, None, None, None, None, None) == 1
    assert L.spmv_jacobi(None, None, None, None, None, None) == 1


def test_struct_sizes_match_header():
    # guards the ctypes mirrors against drift from include/spmv_b200.h (x86-64 layout)
    assert ctypes.sizeof(binding.Info) == 3 * 8 + 2 * 4 + 2 * 8 + 32 * 8 + 8 + 2 * 4 + 8 + 2 * 8 + 2 * 4 + 3 * 8 + 128 + 64
    assert ctypes.sizeof(binding.Allocator) == 24
    # spmv_cg_opts_t: double + 6 int32; spmv_cg_result_t: 8 int32 + char[128] + 3 doubles
    assert ctypes.sizeof(binding.CgOpts) == 8 + 6 * 4
    assert ctypes.sizeof(binding.CgResult) == 8 * 4 + 128 + 3 * 8
    assert binding.CgResult.rel_residual.offset == 160 and binding.CgResult.loop_variant.offset == 32
    # spmv_jacobi_opts_t: 2 doubles + 4 int32; spmv_jacobi_result_t: 7 int32 (+ 4 padding) + 3 doubles
    assert ctypes.sizeof(binding.JacobiOpts) == 2 * 8 + 4 * 4
    assert ctypes.sizeof(binding.JacobiResult) == 7 * 4 + 4 + 3 * 8 and binding.JacobiResult.rel_residual.offset == 32
    # spmv_tune_report_t: the log buffer triple closes the struct
    assert binding.TuneReport.log_len.offset + 8 == ctypes.sizeof(binding.TuneReport)


def test_sizes_over_the_int32_limits_are_unsupported(L):
    """Limits (include/spmv_b200.h): rows, cols, nnz <= 2^31-1 -> SPMV_ERR_UNSUPPORTED, checked before any
    device work (so it can be asserted without a GPU); negative sizes -> INVALID_ARG."""
    import ctypes as C
    h = C.c_void_p(0)
    dummy = (C.c_int32 * 4)()
    big = 1 << 31
    for rows, cols, nnz in ((big, 10, 10), (10, big, 10), (10, 10, big)):
        st = L.spmv_create(C.byref(h), C.c_int64(rows), C.c_int64(cols), C.c_int64(nnz), dummy, dummy, dummy, None, None)
        assert st == 3 and not h.value
    st = L.spmv_create(C.byref(h), C.c_int64(-1), C.c_int64(10), C.c_int64(10), dummy, dummy, dummy, None, None)
    assert st == 1 and not h.value
