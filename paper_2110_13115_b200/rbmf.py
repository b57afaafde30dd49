"""Thin ctypes binding of librbmf.so (include/rbmf.h): argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels.  torch is used for device memory and streams.
Importing this module raises ImportError when the library has not been built -- there is no fallback of any kind.
The module-level functions carry the C names (rbmf_plan_create, rbmf_set_basis, rbmf_set_coeffs, rbmf_filter, ...);
`Plan` is a small convenience wrapper that owns the workspace tensor.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_PKG_DIR = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG_DIR, "librbmf.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(
        "librbmf.so is not built (%s missing). Build it with `python -m paper_2110_13115_b200.build` "
        "or `python -c 'import __graft_entry__ as g; g.build()'`. There is no CPU fallback." % LIB_PATH)

_lib = ctypes.CDLL(LIB_PATH)

RBMF_OK, RBMF_ERR_ARG, RBMF_ERR_STATE, RBMF_ERR_CUDA, RBMF_ERR_OVERFLOW, RBMF_ERR_UNSUPPORTED = 0, -1, -2, -3, -4, -5
RBMF_GEMM_TCGEN05, RBMF_GEMM_SCREEN = 0, 2
RBMF_STAGE1_BASIS, RBMF_STAGE1_TEMPLATES = 0, 1
RBMF_DIAG_STAGE1_FP32_CHECK, RBMF_DIAG_SINGLE_CTA_SCREEN, RBMF_DIAG_STAGE2_PER_CANDIDATE = 1, 2, 3
RBMF_DIAG_FFT_CHUNK_MAJOR, RBMF_DIAG_FFT_LOOKAHEAD, RBMF_DIAG_GEMM_GROUP = 4, 5, 6

TRIGGER_DTYPE = np.dtype([("template", np.int32), ("time", np.int32), ("re", np.float32), ("im", np.float32)])
CANDIDATE_DTYPE = np.dtype([("template", np.int32), ("bin", np.int32), ("re", np.float32), ("im", np.float32)])

# name -> (restype, argtypes); this table is also what tests/test_abi.py checks against include/rbmf.h
_vp, _i32, _i64, _f32, _f64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_float, ctypes.c_double
_pi32, _pi64, _psz = ctypes.POINTER(_i32), ctypes.POINTER(_i64), ctypes.POINTER(ctypes.c_size_t)
SIGNATURES = {
    "rbmf_plan_create": (_i32, [ctypes.POINTER(_vp), _i64, _f64, _f64, _i32, _i32]),
    "rbmf_plan_set_window": (_i32, [_vp, _i32]),
    "rbmf_plan_set_capacity": (_i32, [_vp, _i64, _i64]),
    "rbmf_plan_set_batch": (_i32, [_vp, _i32]),
    "rbmf_plan_set_gemm_impl": (_i32, [_vp, _i32]),
    "rbmf_workspace_bytes": (_i32, [_vp, _psz]),
    "rbmf_plan_set_workspace": (_i32, [_vp, _vp, ctypes.c_size_t]),
    "rbmf_set_stream": (_i32, [_vp, _vp]),
    "rbmf_set_basis": (_i32, [_vp, _vp]),
    "rbmf_set_coeffs": (_i32, [_vp, _vp, _vp]),
    "rbmf_filter": (_i32, [_vp, _vp, _f32, _f32, _vp, _vp]),
    "rbmf_prepare_strain": (_i32, [_vp, _vp, _vp, _i32, _vp]),
    "rbmf_prepare_strain_static": (_i32, [_vp, _vp, _i64, _i32, _vp, _vp, _pi32]),
    "rbmf_prepare_strain_static_limits": (_i32, [_pi64, _psz]),
    "rbmf_prepare_basis_workspace_bytes": (_i32, [_i32, _i32, _psz]),
    "rbmf_prepare_basis": (_i32, [_vp, _i32, _i64, _f64, _f64, _i32, _i32, ctypes.c_uint64, _vp, ctypes.c_size_t, _vp, _vp,
                                  _vp]),
    "rbmf_prepare_coeffs": (_i32, [_vp, _i32, _vp, _i32, _i64, _f64, _f64, _vp, _vp, _vp]),
    "rbmf_bankset_create": (_i32, [ctypes.POINTER(_vp), ctypes.POINTER(_vp), _i32]),
    "rbmf_bankset_filter": (_i32, [_vp, _vp, _f32, _f32, _vp, _i64, _vp, _vp]),
    "rbmf_bankset_get_counts": (_i32, [_vp, _pi64, _pi64, _pi64]),
    "rbmf_bankset_destroy": (_i32, [_vp]),
    "rbmf_plan_enable_template_routes": (_i32, [_vp, _i32]),
    "rbmf_set_templates": (_i32, [_vp, _vp, _vp]),
    "rbmf_plan_set_stage1_route": (_i32, [_vp, _i32]),
    "rbmf_filter_flat": (_i32, [_vp, _vp, _f32, _vp, _vp]),
    "rbmf_filter_batch": (_i32, [_vp, _vp, _i32, _f32, _f32, _vp, _vp]),
    "rbmf_filter_host": (_i32, [_vp, _vp, _f32, _f32, _vp, _i64, _pi64]),
    "rbmf_filter_batch_host": (_i32, [_vp, _vp, _i32, _f32, _f32, _vp, _i64, _pi64]),
    "rbmf_get_counts": (_i32, [_vp, _pi64, _pi64]),
    "rbmf_get_screened_count": (_i32, [_vp, _pi64]),
    "rbmf_get_candidates": (_i32, [_vp, _vp, _i64, _pi64]),
    "rbmf_get_internal": (_i32, [_vp, _i32, ctypes.POINTER(_vp), _psz]),
    "rbmf_plan_set_timing": (_i32, [_vp, _i32]),
    "rbmf_get_stage_ms": (_i32, [_vp, ctypes.POINTER(_f32)]),
    "rbmf_get_stage_ms_history": (_i32, [_vp, _i32, ctypes.POINTER(_f32)]),
    "rbmf_launches_per_filter": (_i32, [_vp, _pi32]),
    "rbmf_plan_destroy": (_i32, [_vp]),
    "rbmf_status_string": (ctypes.c_char_p, [_i32]),
    "rbmf_last_cuda_error": (_i32, [_vp]),
    "rbmf_diag_set": (_i32, [_vp, _i32, _i32]),
}
for _name, (_res, _args) in SIGNATURES.items():
    _fn = getattr(_lib, _name)          # AttributeError here = library does not export what rbmf.h declares
    _fn.restype, _fn.argtypes = _res, _args
    globals()[_name] = _fn


class RbmfError(RuntimeError):
    def __init__(self, status, where, cuda=0):
        self.status = status
        msg = _lib.rbmf_status_string(status).decode()
        super().__init__("%s: %s (status %d, cuda error %d)" % (where, msg, status, cuda))


def _ptr(t):
    """Device (or host) address of a torch tensor / numpy array; None -> NULL."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def prepare_strain_static(x_dev, inv_asd_dev=None, out=None, stream=None):
    """rbmf_prepare_strain_static: time series -> whitened spectrum without a plan and without a workspace.

    For code that may not (or cannot) allocate GPU memory for the library -- a whitening stage with no plan of its
    own, a callback inside somebody else's pipeline that only gets its input and output buffers, a process whose
    memory pool already owns the whole card -- the scratch of the transform is a fixed 12 MiB array inside librbmf.so.
    x_dev: contiguous float32 CUDA tensor (n_segments, N), N a power of two in [2^10, 2^20], n_segments * N <= 2^20
    (RbmfError with RBMF_ERR_UNSUPPORTED beyond that: split the batch); inv_asd_dev: (N/2+1,) float32 or None;
    out: a preallocated (n_segments, N/2+1) complex64 CUDA tensor (allocated with torch when None -- pass it if the
    point is to allocate nothing); stream: a torch stream (default: torch's current one).  Asynchronous.  Same values,
    bit for bit, as Plan.prepare_strain.  All calls on a device share the one array: keep them on one stream or order
    them with events, and make the first call on each device before any stream capture."""
    import torch
    if x_dev.dtype != torch.float32 or x_dev.dim() != 2 or not x_dev.is_cuda or not x_dev.is_contiguous():
        raise ValueError("x must be a contiguous float32 CUDA tensor of shape (n_segments, N)")
    nb, N = int(x_dev.shape[0]), int(x_dev.shape[1])
    if inv_asd_dev is not None and (inv_asd_dev.dtype != torch.float32 or inv_asd_dev.numel() != N // 2 + 1
                                    or inv_asd_dev.device != x_dev.device or not inv_asd_dev.is_contiguous()):
        raise ValueError("inv_asd must be a contiguous float32 CUDA tensor with N/2+1 entries on x's device")
    if out is None:
        out = torch.empty((nb, N // 2 + 1), dtype=torch.complex64, device=x_dev.device)
    elif out.dtype != torch.complex64 or tuple(out.shape) != (nb, N // 2 + 1) or out.device != x_dev.device \
            or not out.is_contiguous():
        raise ValueError("out must be a contiguous complex64 CUDA tensor of shape (n_segments, N/2+1) on x's device")
    with torch.cuda.device(x_dev.device):
        cur = torch.cuda.current_stream()
        st = stream if stream is not None else cur
        if st != cur:
            st.wait_stream(cur)      # tensors the caller has just produced on the current stream
        err = _i32(0)
        status = _lib.rbmf_prepare_strain_static(_ptr(x_dev), _ptr(inv_asd_dev), N, nb, _ptr(out), st.cuda_stream,
                                                 ctypes.byref(err))
    if status != RBMF_OK:
        raise RbmfError(status, "rbmf_prepare_strain_static", err.value)
    return out


class Plan:
    """Owns an rbmf_plan and its workspace tensor.  All tensors handed in must live on the plan's CUDA device.

    Stream discipline: the library enqueues on the plan's stream only.  Every copy this wrapper makes (host -> device
    staging of inputs, device -> host read-back of results) is issued on that same stream, and a tensor the caller
    produced on another stream is ordered before its first use here (`_order_after_current`), so a `Plan(stream=s)`
    works whether or not the caller has made `s` torch's current stream."""

    def __init__(self, N, fs, f_low, k, T, w=8, max_candidates=1 << 22, max_triggers=1 << 22, device="cuda:0",
                 stream=None, max_batch=1, template_slab=0):
        import torch
        self._torch = torch
        self.N, self.fs, self.f_low, self.k, self.T, self.w = int(N), float(fs), float(f_low), int(k), int(T), int(w)
        self.max_candidates, self.max_triggers = int(max_candidates), int(max_triggers)
        self.max_batch = int(max_batch)
        self.device = torch.device(device)
        self._h = _vp()
        self.stream = None
        self._fp32_check = False
        self._check(_lib.rbmf_plan_create(ctypes.byref(self._h), self.N, self.fs, self.f_low, self.k, self.T),
                    "rbmf_plan_create")
        self._check(_lib.rbmf_plan_set_window(self._h, self.w), "rbmf_plan_set_window")
        self._check(_lib.rbmf_plan_set_capacity(self._h, self.max_candidates, self.max_triggers),
                    "rbmf_plan_set_capacity")
        self._check(_lib.rbmf_plan_set_batch(self._h, self.max_batch), "rbmf_plan_set_batch")
        if template_slab:
            self._check(_lib.rbmf_plan_enable_template_routes(self._h, int(template_slab)),
                        "rbmf_plan_enable_template_routes")
        nbytes = ctypes.c_size_t()
        self._check(_lib.rbmf_workspace_bytes(self._h, ctypes.byref(nbytes)), "rbmf_workspace_bytes")
        self.workspace_bytes = nbytes.value
        with torch.cuda.device(self.device):
            self._ws = torch.empty(self.workspace_bytes + 1024, dtype=torch.uint8, device=self.device)
            base = (self._ws.data_ptr() + 1023) // 1024 * 1024
            self.set_stream(stream)
            with torch.cuda.stream(self.stream):
                self._check(_lib.rbmf_plan_set_workspace(self._h, base, self.workspace_bytes),
                            "rbmf_plan_set_workspace")
                self._out = torch.empty(self.max_triggers * 4, dtype=torch.int32, device=self.device)
                self._n_out = torch.zeros(1, dtype=torch.int64, device=self.device)
        self._keep = []
        self.gemm_impl = RBMF_GEMM_SCREEN      # the library's default (include/rbmf.h)

    # -- helpers -----------------------------------------------------------------------------
    def _check(self, status, where, allow=()):
        if status != RBMF_OK and status not in allow:
            cuda = _lib.rbmf_last_cuda_error(self._h) if self._h else 0
            raise RbmfError(status, where, cuda)
        return status

    def set_stream(self, stream=None):
        """Enqueue on `stream` from now on (default: torch's current stream).  Work already enqueued on the previous
        stream (table initialisation, set_basis / set_coeffs, an earlier filter) is ordered before the new one."""
        torch = self._torch
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        old = self.stream
        if old is not None and old.cuda_stream != stream.cuda_stream:
            ev = torch.cuda.Event()
            ev.record(old)
            stream.wait_event(ev)
        self.stream = stream
        self._check(_lib.rbmf_set_stream(self._h, _vp(stream.cuda_stream)), "rbmf_set_stream")

    def _order_after_current(self):
        """Make the plan's stream wait for what torch's current stream has enqueued so far (the producer of a tensor
        the caller hands in), unless they are the same stream."""
        cur = self._torch.cuda.current_stream(self.device)
        if cur.cuda_stream != self.stream.cuda_stream:
            self.stream.wait_stream(cur)

    def _dev(self, x, dtype):
        """`x` as a contiguous tensor on the plan's device; the copy, if one is needed, runs on the plan's stream."""
        torch = self._torch
        t = torch.as_tensor(x)
        if t.dtype != dtype:
            raise TypeError("expected %s, got %s" % (dtype, t.dtype))
        self._order_after_current()
        with torch.cuda.stream(self.stream):
            t = t.to(self.device).contiguous()
            t.record_stream(self.stream)
        return t

    # -- ABI calls ---------------------------------------------------------------------------
    def set_gemm_impl(self, impl):
        self._check(_lib.rbmf_plan_set_gemm_impl(self._h, int(impl)), "rbmf_plan_set_gemm_impl")
        self.gemm_impl = int(impl)

    def diag_set(self, option, value):
        """Test-only switches (include/rbmf.h, diagnostics section)."""
        self._check(_lib.rbmf_diag_set(self._h, int(option), int(value)), "rbmf_diag_set")
        if int(option) == RBMF_DIAG_STAGE1_FP32_CHECK:
            self._fp32_check = bool(value)

    def set_timing(self, enabled=True):
        self._check(_lib.rbmf_plan_set_timing(self._h, 1 if enabled else 0), "rbmf_plan_set_timing")

    def set_basis(self, basis):
        torch = self._torch
        b = self._dev(basis, torch.complex64)
        if tuple(b.shape) != (self.k, self.N // 2 + 1):
            raise ValueError("basis must be k x (N/2+1)")
        with torch.cuda.device(self.device):
            self._check(_lib.rbmf_set_basis(self._h, _ptr(b)), "rbmf_set_basis")
        self.stream.synchronize()      # the library has copied; `b` may go away

    def set_coeffs(self, coeffs, sigma=None):
        torch = self._torch
        c = self._dev(coeffs, torch.complex64)
        if tuple(c.shape) != (self.T, self.k):
            raise ValueError("coeffs must be T x k")
        s = None if sigma is None else self._dev(sigma, torch.float32)
        if s is not None and tuple(s.shape) != (self.T,):
            raise ValueError("sigma must have T entries")
        with torch.cuda.device(self.device):
            self._check(_lib.rbmf_set_coeffs(self._h, _ptr(c), _ptr(s)), "rbmf_set_coeffs")
        self.stream.synchronize()

    def filter_async(self, strain_dev, thr1, thr2):
        """Enqueue rbmf_filter on the plan's stream; strain_dev is a complex64 CUDA tensor of N/2+1 bins."""
        torch = self._torch
        if strain_dev.dtype != torch.complex64 or strain_dev.numel() != self.N // 2 + 1 or not strain_dev.is_cuda:
            raise ValueError("strain must be a complex64 CUDA tensor with N/2+1 entries")
        self._order_after_current()
        with torch.cuda.device(self.device):
            self._check(_lib.rbmf_filter(self._h, _ptr(strain_dev), float(thr1), float(thr2), _ptr(self._out),
                                         _ptr(self._n_out)), "rbmf_filter")

    def set_templates(self, templates_dev, sigma=None):
        """rbmf_set_templates: a (T, N/2+1) complex64 CUDA tensor, RETAINED (kept alive by this object), + sigma."""
        torch = self._torch
        if (templates_dev.dtype != torch.complex64 or tuple(templates_dev.shape) != (self.T, self.N // 2 + 1)
                or not templates_dev.is_cuda or not templates_dev.is_contiguous()):
            raise ValueError("templates must be a contiguous complex64 CUDA tensor of shape (T, N/2+1)")
        s = None if sigma is None else self._dev(sigma, torch.float32)
        self._order_after_current()
        with torch.cuda.device(self.device):
            self._check(_lib.rbmf_set_templates(self._h, _ptr(templates_dev), _ptr(s)), "rbmf_set_templates")
        self.stream.synchronize()
        self._templates = templates_dev

    def set_stage1_route(self, route):
        self._check(_lib.rbmf_plan_set_stage1_route(self._h, int(route)), "rbmf_plan_set_stage1_route")

    def filter_flat(self, strain, thr, allow_overflow=False):
        """rbmf_filter_flat: the flat template method; returns triggers sorted by (template, time)."""
        torch = self._torch
        s = self._dev(strain, torch.complex64)
        with torch.cuda.device(self.device):
            self._check(_lib.rbmf_filter_flat(self._h, _ptr(s), float(thr), _ptr(self._out), _ptr(self._n_out)),
                        "rbmf_filter_flat")
        return self.triggers(allow_overflow)

    def prepare_strain(self, x_dev, inv_asd_dev=None):
        """rbmf_prepare_strain: (n_segments, N) float32 CUDA time series [+ (N/2+1,) float32 whitening array] ->
        (n_segments, N/2+1) complex64 CUDA tensor, the input of filter_batch_async."""
        torch = self._torch
        if x_dev.dtype != torch.float32 or x_dev.dim() != 2 or x_dev.shape[1] != self.N or not x_dev.is_cuda \
                or not x_dev.is_contiguous():
            raise ValueError("x must be a contiguous float32 CUDA tensor of shape (n_segments, N)")
        if inv_asd_dev is not None and (inv_asd_dev.dtype != torch.float32 or inv_asd_dev.numel() != self.N // 2 + 1
                                        or not inv_asd_dev.is_cuda or not inv_asd_dev.is_contiguous()):
            raise ValueError("inv_asd must be a contiguous float32 CUDA tensor with N/2+1 entries")
        self._order_after_current()
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            out = torch.empty((x_dev.shape[0], self.N // 2 + 1), dtype=torch.complex64, device=self.device)
            self._check(_lib.rbmf_prepare_strain(self._h, _ptr(x_dev), _ptr(inv_asd_dev), int(x_dev.shape[0]),
                                                 _ptr(out)), "rbmf_prepare_strain")
        return out

    def filter_batch_async(self, strain_dev, thr1, thr2):
        """Enqueue rbmf_filter_batch; strain_dev is a complex64 CUDA tensor of shape (n_segments, N/2+1)."""
        torch = self._torch
        if (strain_dev.dtype != torch.complex64 or strain_dev.dim() != 2 or strain_dev.shape[1] != self.N // 2 + 1
                or not strain_dev.is_cuda or not strain_dev.is_contiguous()):
            raise ValueError("strain must be a contiguous complex64 CUDA tensor of shape (n_segments, N/2+1)")
        self._order_after_current()
        with torch.cuda.device(self.device):
            self._check(_lib.rbmf_filter_batch(self._h, _ptr(strain_dev), int(strain_dev.shape[0]), float(thr1),
                                               float(thr2), _ptr(self._out), _ptr(self._n_out)), "rbmf_filter_batch")

    def filter_batch(self, strains, thr1, thr2, allow_overflow=False):
        """Filter a batch; returns the triggers sorted by (template, time) with time = segment * N + n."""
        s = self._dev(strains, self._torch.complex64)
        self.filter_batch_async(s, thr1, thr2)
        return self.triggers(allow_overflow)

    def filter_batch_host(self, strains_host, thr1, thr2, out_host=None):
        """rbmf_filter_batch_host: host strains (n_segments, N/2+1) in, host triggers out (unsorted)."""
        torch = self._torch
        if out_host is None:
            out_host = np.empty(self.max_triggers, dtype=TRIGGER_DTYPE)
        n = _i64()
        with torch.cuda.device(self.device):
            st = _lib.rbmf_filter_batch_host(self._h, _ptr(strains_host), int(strains_host.shape[0]), float(thr1),
                                             float(thr2), _ptr(out_host), len(out_host), ctypes.byref(n))
        self._check(st, "rbmf_filter_batch_host", allow=(RBMF_ERR_OVERFLOW,))
        return out_host[: min(n.value, len(out_host))], n.value

    def counts(self, allow_overflow=False):
        nc, nt = _i64(), _i64()
        st = self._check(_lib.rbmf_get_counts(self._h, ctypes.byref(nc), ctypes.byref(nt)), "rbmf_get_counts",
                         allow=(RBMF_ERR_OVERFLOW,) if allow_overflow else ())
        return nc.value, nt.value, st

    def triggers(self, allow_overflow=False):
        """Synchronise and return the trigger list of the last filter call, sorted by (template, time)."""
        nc, nt, _ = self.counts(allow_overflow)
        n = min(nt, self.max_triggers)
        with self._torch.cuda.stream(self.stream):
            raw = self._out[: 4 * n].cpu().numpy()
        trig = raw.view(TRIGGER_DTYPE).copy() if n else np.empty(0, dtype=TRIGGER_DTYPE)
        return np.sort(trig, order=("template", "time"))

    def triggers_device(self, allow_overflow=False):
        """The trigger list of the last filter call as an (n, 4) int32 CUDA tensor (columns: template, time, and the
        bit patterns of re, im), unsorted, without a device -> host copy: for callers that select on the device."""
        nc, nt, _ = self.counts(allow_overflow)
        n = min(nt, self.max_triggers)
        return self._out[: 4 * n].view(n, 4)

    def candidates_device(self):
        """The first-stage candidate list of the last filter call as an (n, 4) int32 CUDA tensor (template, bin, bits
        of avg_re, avg_im)."""
        nc, _, _ = self.counts(allow_overflow=True)
        n = min(nc, self.max_candidates)
        p, nb = _vp(), ctypes.c_size_t()
        self._check(_lib.rbmf_get_internal(self._h, 6, ctypes.byref(p), ctypes.byref(nb)), "rbmf_get_internal")
        off = p.value - self._ws.data_ptr()
        return self._ws[off: off + 16 * n].view(self._torch.int32).view(n, 4)

    def filter(self, strain, thr1, thr2, allow_overflow=False):
        torch = self._torch
        s = self._dev(strain, torch.complex64)
        self.filter_async(s, thr1, thr2)
        return self.triggers(allow_overflow)

    def filter_host(self, strain_host, thr1, thr2, out_host=None):
        """rbmf_filter_host: host strain in, host triggers out (unsorted); returns (array view, total found)."""
        torch = self._torch
        if out_host is None:
            out_host = np.empty(self.max_triggers, dtype=TRIGGER_DTYPE)
        n = _i64()
        with torch.cuda.device(self.device):
            st = _lib.rbmf_filter_host(self._h, _ptr(strain_host), float(thr1), float(thr2), _ptr(out_host),
                                       len(out_host), ctypes.byref(n))
        self._check(st, "rbmf_filter_host", allow=(RBMF_ERR_OVERFLOW,))
        return out_host[: min(n.value, len(out_host))], n.value

    def screened_count(self):
        n = _i64()
        self._check(_lib.rbmf_get_screened_count(self._h, ctypes.byref(n)), "rbmf_get_screened_count")
        return n.value

    def candidates(self):
        nc, _, _ = self.counts(allow_overflow=True)
        n = min(nc, self.max_candidates)
        out = np.empty(max(n, 1), dtype=CANDIDATE_DTYPE)
        tot = _i64()
        self._check(_lib.rbmf_get_candidates(self._h, _ptr(out), n, ctypes.byref(tot)), "rbmf_get_candidates",
                    allow=(RBMF_ERR_OVERFLOW,))
        return np.sort(out[:n], order=("template", "bin"))

    def internal(self, which, segment=0):
        """Copy of an internal array: 'beta' -> (N, k) complex64; 'beta_avg' -> (N/w, k) complex64 (bf16 hi + lo, or
        the single fp16 plane in RBMF_GEMM_SCREEN mode), of segment `segment` of the last batch."""
        torch = self._torch
        self.stream.synchronize()

        def view(idx):
            p, nb = _vp(), ctypes.c_size_t()
            self._check(_lib.rbmf_get_internal(self._h, idx, ctypes.byref(p), ctypes.byref(nb)), "rbmf_get_internal")
            off = p.value - self._ws.data_ptr()
            return self._ws[off: off + nb.value]

        C = 4   # columns per chunk of the library's chunk-blocked layouts (include/rbmf.h, rbmf_get_internal)
        screen = self.gemm_impl == RBMF_GEMM_SCREEN and not self._fp32_check
        if which == "screened":      # the stage-1 list as kernel 2 wrote it (raw fp16-product values in screen mode)
            n = min(self.screened_count(), self.max_candidates)
            with torch.cuda.stream(self.stream):
                raw = view(3)[: 16 * n].cpu().numpy()
            return raw.view(CANDIDATE_DTYPE).copy()
        if which in ("bin_norm", "tnorm_blk"):
            with torch.cuda.stream(self.stream):
                return view(4 if which == "bin_norm" else 5).view(torch.float32).cpu().numpy()
        if which == "beta":
            with torch.cuda.stream(self.stream):
                v = view(0).view(torch.float32).view(self.max_batch, self.k // C, self.N, C, 2)[segment]   # [chunk][n][C]
                return torch.view_as_complex(
                    v.permute(1, 0, 2, 3).reshape(self.N, self.k, 2).contiguous()).cpu().numpy()
        if which == "beta_avg":
            M, nkb, Mp = self.N // self.w, (self.k + 31) // 32, self.max_batch * (self.N // self.w)
            if screen:                                   # one fp16 plane
                hi = view(1).view(torch.float16).to(torch.float32)
                lo = torch.zeros_like(hi)
            else:
                hi = view(1).view(torch.bfloat16).to(torch.float32)
                lo = view(2).view(torch.bfloat16).to(torch.float32)
            v = (hi + lo).view(nkb, Mp, 32, 2)[:, segment * M:(segment + 1) * M]                        # [kb][bin][32]
            v = v.permute(1, 0, 2, 3).reshape(M, nkb * 32, 2)[:, : self.k]
            return torch.view_as_complex(v.contiguous()).cpu().numpy()
        raise KeyError(which)

    def stage_ms(self):
        ms = (_f32 * 4)()
        self._check(_lib.rbmf_get_stage_ms(self._h, ms), "rbmf_get_stage_ms")
        return {"fft": ms[0], "gemm": ms[1], "stage2": ms[2], "total": ms[3]}

    def stage_ms_history(self, n_calls):
        """Per-stage times of the last `n_calls` (<= 64) timed calls, oldest first, read after the fact: the calls
        themselves can be enqueued back to back without a host synchronisation in between."""
        out = []
        for back in range(int(n_calls) - 1, -1, -1):
            ms = (_f32 * 4)()
            self._check(_lib.rbmf_get_stage_ms_history(self._h, back, ms), "rbmf_get_stage_ms_history")
            out.append({"fft": ms[0], "gemm": ms[1], "stage2": ms[2], "total": ms[3]})
        return out

    def launches_per_filter(self):
        n = _i32()
        self._check(_lib.rbmf_launches_per_filter(self._h, ctypes.byref(n)), "rbmf_launches_per_filter")
        return n.value

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            try:
                self._torch.cuda.synchronize(self.device)
            except Exception:
                pass
            _lib.rbmf_plan_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class BankSet:
    """rbmf_bankset_*: several fully set-up `Plan`s (sub-banks with their own k, T, w; same N, fs, f_low) filtered
    against one strain into one trigger list; template ids are offset by the sizes of the sub-banks before."""

    def __init__(self, plans, max_triggers=1 << 22, stream=None):
        import torch
        self._torch = torch
        self.plans = list(plans)
        self.device = self.plans[0].device
        self.max_triggers = int(max_triggers)
        self.stream = stream if stream is not None else self.plans[0].stream
        self._h = _vp()
        arr = (_vp * len(self.plans))(*[p._h for p in self.plans])
        with torch.cuda.device(self.device):
            st = _lib.rbmf_bankset_create(ctypes.byref(self._h), arr, len(self.plans))
        if st != RBMF_OK:
            raise RbmfError(st, "rbmf_bankset_create")
        with torch.cuda.stream(self.stream):
            self._out = torch.empty(self.max_triggers * 4, dtype=torch.int32, device=self.device)
            self._n_out = torch.zeros(1, dtype=torch.int64, device=self.device)

    def filter_async(self, strain_dev, thr1, thr2):
        # the strain may have been produced on torch's current stream: order the set's stream after it, as
        # Plan._order_after_current does (the library orders the sub-banks after the set's stream and the plans' own)
        cur = self._torch.cuda.current_stream(self.device)
        if cur.cuda_stream != self.stream.cuda_stream:
            self.stream.wait_stream(cur)
        with self._torch.cuda.device(self.device):
            st = _lib.rbmf_bankset_filter(self._h, _ptr(strain_dev), float(thr1), float(thr2), _ptr(self._out),
                                          self.max_triggers, _ptr(self._n_out), _vp(self.stream.cuda_stream))
        if st != RBMF_OK:
            raise RbmfError(st, "rbmf_bankset_filter")

    def counts(self):
        n = len(self.plans)
        nc, nt, tot = (_i64 * n)(), (_i64 * n)(), _i64()
        with self._torch.cuda.device(self.device):
            st = _lib.rbmf_bankset_get_counts(self._h, nc, nt, ctypes.byref(tot))
        if st not in (RBMF_OK, RBMF_ERR_OVERFLOW):
            raise RbmfError(st, "rbmf_bankset_get_counts")
        return list(nc), list(nt), tot.value, st

    def filter(self, strain, thr1, thr2):
        torch = self._torch
        with torch.cuda.stream(self.stream):
            s = torch.as_tensor(strain).to(self.device)
        self.filter_async(s, thr1, thr2)
        _, _, tot, _ = self.counts()
        n = min(tot, self.max_triggers)
        with torch.cuda.stream(self.stream):
            raw = self._out[: 4 * n].cpu().numpy()
        trig = raw.view(TRIGGER_DTYPE).copy() if n else np.empty(0, dtype=TRIGGER_DTYPE)
        return np.sort(trig, order=("template", "time"))

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._torch.cuda.synchronize(self.device)
            _lib.rbmf_bankset_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def prepare_basis(templates_dev, N, fs, f_low, k, iterations=12, seed=1, stream=None):
    """rbmf_prepare_basis + rbmf_prepare_coeffs on a (S, N/2+1) complex64 CUDA tensor of templates: returns
    (basis (k, N/2+1) complex64, eigenvalue estimates (k,) float32) as CUDA tensors."""
    import torch
    if (templates_dev.dtype != torch.complex64 or templates_dev.dim() != 2 or templates_dev.shape[1] != N // 2 + 1
            or not templates_dev.is_cuda or not templates_dev.is_contiguous()):
        raise ValueError("templates must be a contiguous complex64 CUDA tensor of shape (S, N/2+1)")
    S = int(templates_dev.shape[0])
    st = stream if stream is not None else torch.cuda.current_stream(templates_dev.device)
    nbytes = ctypes.c_size_t()
    rc = _lib.rbmf_prepare_basis_workspace_bytes(S, int(k), ctypes.byref(nbytes))
    if rc != RBMF_OK:
        raise RbmfError(rc, "rbmf_prepare_basis_workspace_bytes")
    with torch.cuda.device(templates_dev.device), torch.cuda.stream(st):
        ws = torch.empty(nbytes.value + 16, dtype=torch.uint8, device=templates_dev.device)
        base = (ws.data_ptr() + 15) // 16 * 16
        basis = torch.empty((int(k), N // 2 + 1), dtype=torch.complex64, device=templates_dev.device)
        eig = torch.empty(int(k), dtype=torch.float32, device=templates_dev.device)
        rc = _lib.rbmf_prepare_basis(_ptr(templates_dev), S, int(N), float(fs), float(f_low), int(k), int(iterations),
                                     int(seed), _vp(base), nbytes.value, _ptr(basis), _ptr(eig), _vp(st.cuda_stream))
        if rc != RBMF_OK:
            raise RbmfError(rc, "rbmf_prepare_basis")
        st.synchronize()
    return basis, eig


def prepare_coeffs(templates_dev, basis_dev, N, fs, f_low, stream=None):
    """rbmf_prepare_coeffs: (T, N/2+1) templates and (k, N/2+1) basis -> (coeffs (T, k) complex64, sigma (T,) float32)."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream(templates_dev.device)
    T, k = int(templates_dev.shape[0]), int(basis_dev.shape[0])
    with torch.cuda.device(templates_dev.device), torch.cuda.stream(st):
        coeffs = torch.empty((T, k), dtype=torch.complex64, device=templates_dev.device)
        sigma = torch.empty(T, dtype=torch.float32, device=templates_dev.device)
        rc = _lib.rbmf_prepare_coeffs(_ptr(templates_dev), T, _ptr(basis_dev), k, int(N), float(fs), float(f_low),
                                      _ptr(coeffs), _ptr(sigma), _vp(st.cuda_stream))
        if rc != RBMF_OK:
            raise RbmfError(rc, "rbmf_prepare_coeffs")
        st.synchronize()
    return coeffs, sigma
