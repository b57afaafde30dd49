"""Host-side checks of the C-ABI library: it loads, exports every symbol include/rbmf.h declares, validates its
arguments and reports call-order errors.  No compute calls: none of this needs a GPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "rbmf.h")


def _declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rbmf_[a-z0-9_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib(built_library):
    return ctypes.CDLL(built_library)


@pytest.fixture(scope="module")
def binding(built_library):
    from paper_2110_13115_b200 import rbmf
    return rbmf


def test_header_symbols_are_exported(lib):
    names = _declared_symbols()
    assert len(names) >= 18 and "rbmf_filter" in names and "rbmf_plan_create" in names
    for name in names:
        assert hasattr(lib, name), "librbmf.so does not export %s" % name


def test_binding_covers_the_header(binding):
    assert sorted(binding.SIGNATURES) == _declared_symbols()


def test_struct_sizes_match_header(binding):
    assert binding.TRIGGER_DTYPE.itemsize == 16 and binding.CANDIDATE_DTYPE.itemsize == 16


def _create(b, N=4096, fs=1024.0, f_low=30.0, k=16, T=64):
    h = ctypes.c_void_p()
    st = b.rbmf_plan_create(ctypes.byref(h), N, fs, f_low, k, T)
    return st, h


def test_plan_create_validates_arguments(binding):
    b = binding
    st, h = _create(b)
    assert st == b.RBMF_OK and h.value
    assert b.rbmf_plan_destroy(h) == b.RBMF_OK
    for N in (1 << 21, 1 << 24):      # valid by the contract (up to 2^24), not built: two FFT passes of <= 1024
        st, h = _create(b, N=N)
        assert st == b.RBMF_ERR_UNSUPPORTED and not h.value
    for kw in (dict(N=4095), dict(N=512), dict(N=1 << 25), dict(k=20), dict(k=8), dict(k=2048), dict(T=0),
               dict(f_low=0.0), dict(f_low=600.0), dict(fs=-1.0)):
        st, h = _create(b, **kw)
        assert st == b.RBMF_ERR_ARG and not h.value, kw
    assert b.rbmf_plan_create(None, 4096, 1024.0, 30.0, 16, 64) == b.RBMF_ERR_ARG


def test_window_capacity_and_workspace_size(binding):
    b = binding
    st, h = _create(b)
    nbytes = ctypes.c_size_t()
    assert b.rbmf_workspace_bytes(h, ctypes.byref(nbytes)) == b.RBMF_OK
    default_bytes = nbytes.value
    # beta (N k 8) + the re-laid-out basis (N/2 k 8) alone are 1.5 N k 8 bytes
    assert default_bytes > 1.5 * 4096 * 16 * 8
    for w in (0, 3, 64):             # not a power of two in [1, 32]
        assert b.rbmf_plan_set_window(h, w) == b.RBMF_ERR_ARG
    st2, h2 = _create(b, N=1024)
    assert b.rbmf_plan_set_window(h2, 16) == b.RBMF_ERR_ARG      # N/w = 64 < 128 bins (one GEMM tile)
    assert b.rbmf_plan_set_window(h2, 8) == b.RBMF_OK
    b.rbmf_plan_destroy(h2)
    assert b.rbmf_plan_set_window(h, 4) == b.RBMF_OK
    assert b.rbmf_plan_set_capacity(h, 0, 10) == b.RBMF_ERR_ARG
    assert b.rbmf_plan_set_capacity(h, 1000, 1000) == b.RBMF_OK
    assert b.rbmf_workspace_bytes(h, ctypes.byref(nbytes)) == b.RBMF_OK
    assert nbytes.value < default_bytes          # smaller lists
    n = ctypes.c_int32()
    assert b.rbmf_launches_per_filter(h, ctypes.byref(n)) == b.RBMF_OK and n.value == 7   # screen mode (default): prep, FFT, bin norms, GEMM, stage 2 = alloc + scatter + score
    assert b.rbmf_plan_set_window(h, 1) == b.RBMF_OK
    assert b.rbmf_launches_per_filter(h, ctypes.byref(n)) == b.RBMF_OK and n.value == 7
    assert b.rbmf_plan_set_gemm_impl(h, 7) == b.RBMF_ERR_ARG
    assert b.rbmf_plan_set_gemm_impl(h, 1) == b.RBMF_ERR_ARG     # the fp32 check kernel is not a product mode
    assert b.rbmf_plan_set_gemm_impl(h, b.RBMF_GEMM_TCGEN05) == b.RBMF_OK
    assert b.rbmf_launches_per_filter(h, ctypes.byref(n)) == b.RBMF_OK and n.value == 6
    assert b.rbmf_diag_set(h, b.RBMF_DIAG_STAGE2_PER_CANDIDATE, 1) == b.RBMF_OK
    assert b.rbmf_launches_per_filter(h, ctypes.byref(n)) == b.RBMF_OK and n.value == 4
    assert b.rbmf_diag_set(h, b.RBMF_DIAG_STAGE2_PER_CANDIDATE, 0) == b.RBMF_OK
    assert b.rbmf_plan_set_batch(h, 0) == b.RBMF_ERR_ARG
    assert b.rbmf_plan_set_batch(h, 1 << 20) == b.RBMF_ERR_ARG     # batch * N must fit a 31-bit sample index
    before = ctypes.c_size_t()
    assert b.rbmf_workspace_bytes(h, ctypes.byref(before)) == b.RBMF_OK
    assert b.rbmf_plan_set_batch(h, 4) == b.RBMF_OK
    assert b.rbmf_workspace_bytes(h, ctypes.byref(nbytes)) == b.RBMF_OK and nbytes.value > before.value
    assert b.rbmf_plan_set_gemm_impl(h, b.RBMF_GEMM_SCREEN) == b.RBMF_OK
    assert b.rbmf_diag_set(h, 99, 1) == b.RBMF_ERR_ARG
    # scheduling overrides (formerly environment variables read inside rbmf_filter_batch): validated, 0 = automatic
    assert b.rbmf_diag_set(h, b.RBMF_DIAG_FFT_CHUNK_MAJOR, 1) == b.RBMF_OK
    assert b.rbmf_diag_set(h, b.RBMF_DIAG_FFT_CHUNK_MAJOR, 0) == b.RBMF_OK
    for opt, bad in ((b.RBMF_DIAG_FFT_LOOKAHEAD, (-1, 257)), (b.RBMF_DIAG_GEMM_GROUP, (-1,))):
        for v in bad:
            assert b.rbmf_diag_set(h, opt, v) == b.RBMF_ERR_ARG
        assert b.rbmf_diag_set(h, opt, 3) == b.RBMF_OK
        assert b.rbmf_diag_set(h, opt, 0) == b.RBMF_OK
    assert b.rbmf_diag_set(h, b.RBMF_DIAG_STAGE1_FP32_CHECK, 1) == b.RBMF_OK
    assert b.rbmf_launches_per_filter(h, ctypes.byref(n)) == b.RBMF_OK and n.value == 6
    assert b.rbmf_diag_set(h, b.RBMF_DIAG_STAGE1_FP32_CHECK, 0) == b.RBMF_OK
    assert b.rbmf_get_screened_count(h, ctypes.byref(ctypes.c_int64())) == b.RBMF_ERR_STATE
    ms = (ctypes.c_float * 4)()
    assert b.rbmf_get_stage_ms_history(h, 64, ms) == b.RBMF_ERR_ARG       # the plan keeps 64 timed calls: 0..63
    assert b.rbmf_get_stage_ms_history(h, -1, ms) == b.RBMF_ERR_ARG
    assert b.rbmf_get_stage_ms_history(h, 0, None) == b.RBMF_ERR_ARG
    assert b.rbmf_get_stage_ms_history(h, 0, ms) == b.RBMF_ERR_STATE      # nothing filtered yet
    b.rbmf_plan_destroy(h)


def test_call_order_errors_without_workspace(binding):
    b = binding
    st, h = _create(b)
    dummy = ctypes.c_void_p(1024)
    assert b.rbmf_set_basis(h, dummy) == b.RBMF_ERR_STATE
    assert b.rbmf_set_coeffs(h, dummy, None) == b.RBMF_ERR_STATE
    assert b.rbmf_filter(h, dummy, 5.0, 6.0, dummy, dummy) == b.RBMF_ERR_STATE
    assert b.rbmf_filter(h, dummy, -1.0, 6.0, dummy, dummy) == b.RBMF_ERR_ARG
    assert b.rbmf_filter(h, None, 5.0, 6.0, dummy, dummy) == b.RBMF_ERR_ARG
    assert b.rbmf_get_counts(h, None, None) == b.RBMF_ERR_STATE
    # misaligned / too small workspace is rejected before any CUDA call
    assert b.rbmf_plan_set_workspace(h, ctypes.c_void_p(1000), 1 << 40) == b.RBMF_ERR_ARG
    assert b.rbmf_plan_set_workspace(h, ctypes.c_void_p(1024), 16) == b.RBMF_ERR_ARG
    b.rbmf_plan_destroy(h)


def test_status_strings(binding):
    b = binding
    seen = set()
    for code in (0, -1, -2, -3, -4, -5):
        s = b.rbmf_status_string(code)
        assert s and s not in seen
        seen.add(s)
    assert b.rbmf_status_string(-99) == b"unknown status"


def test_product_path_does_not_import_the_oracle():
    """The oracle is test infrastructure: nothing under the package may import it (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2110_13115_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2110_13115_b200" not in text and "from paper_2110_13115_b200" not in text, f


def test_new_entry_points_validate_arguments_without_a_gpu(binding):
    """rbmf_filter_batch / rbmf_prepare_strain / template routes / bank sets: argument and call-order errors are
    reported before any CUDA call."""
    b = binding
    st, h = _create(b)
    dummy = ctypes.c_void_p(1024)
    assert b.rbmf_filter_batch(h, dummy, 0, 5.0, 6.0, dummy, dummy) == b.RBMF_ERR_ARG          # thresholds / state first
    assert b.rbmf_filter_batch(h, dummy, 1, 5.0, 6.0, dummy, dummy) == b.RBMF_ERR_STATE
    assert b.rbmf_filter_batch_host(h, dummy, 1, 5.0, 6.0, dummy, 10, ctypes.byref(ctypes.c_int64())) == b.RBMF_ERR_STATE
    assert b.rbmf_prepare_strain(h, dummy, None, 1, dummy) == b.RBMF_ERR_STATE
    assert b.rbmf_prepare_strain(h, None, None, 1, dummy) == b.RBMF_ERR_ARG
    assert b.rbmf_plan_enable_template_routes(h, 1028) == b.RBMF_ERR_ARG
    assert b.rbmf_plan_set_window(h, 4) == b.RBMF_OK
    assert b.rbmf_plan_enable_template_routes(h, 0) == b.RBMF_OK
    before, after = ctypes.c_size_t(), ctypes.c_size_t()
    assert b.rbmf_workspace_bytes(h, ctypes.byref(before)) == b.RBMF_OK
    assert b.rbmf_plan_enable_template_routes(h, 64) == b.RBMF_OK
    assert b.rbmf_workspace_bytes(h, ctypes.byref(after)) == b.RBMF_OK and after.value > before.value
    # bank sets: NULL / empty / plans that are not set up
    bs = ctypes.c_void_p()
    arr = (ctypes.c_void_p * 1)(h)
    assert b.rbmf_bankset_create(None, arr, 1) == b.RBMF_ERR_ARG
    assert b.rbmf_bankset_create(ctypes.byref(bs), arr, 0) == b.RBMF_ERR_ARG and not bs.value
    assert b.rbmf_bankset_create(ctypes.byref(bs), arr, 1) == b.RBMF_ERR_STATE and not bs.value
    assert b.rbmf_bankset_filter(None, dummy, 5.0, 6.0, dummy, 10, dummy, None) == b.RBMF_ERR_ARG
    assert b.rbmf_bankset_get_counts(None, None, None, None) == b.RBMF_ERR_ARG
    assert b.rbmf_bankset_destroy(None) == b.RBMF_ERR_ARG
    b.rbmf_plan_destroy(h)
