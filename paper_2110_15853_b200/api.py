"""ctypes binding of include/ttdft.h -- argument marshalling only (same names as the C calls)."""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_char_p, c_double, c_int32, c_int64, c_size_t, c_uint32, c_void_p

_PKG = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_PKG, "libttdft.so")

CHECK_SORTED, CHECK_SYMMETRY, FORCE_GENERIC, NO_I8, OWNED_ROWS_ONLY, PACKED = 1, 2, 4, 8, 16, 32
MATH_AUTO, MATH_FP64, MATH_I8, MATH_I8X7 = 0, 1, 2, 3
FMT_CSR, FMT_BSR, FMT_HYBRID = 0, 1, 2
_STATUS = {0: "OK", 1: "INVALID_ARG", 2: "UNSUPPORTED", 3: "WORKSPACE_TOO_SMALL", 4: "NOT_SYMMETRIC", 5: "CUDA", 6: "BREAKDOWN"}

# every symbol include/ttdft.h declares
exported_symbols = [
    "ttdft_h_storage_bytes", "ttdft_h_build", "ttdft_h_info", "ttdft_h_destroy", "ttdft_spmm", "ttdft_cheb_step",
    "ttdft_cheb_scalars", "ttdft_cheb_filter_work_bytes", "ttdft_cheb_filter", "ttdft_cheb_filter_host_work_bytes",
    "ttdft_cheb_filter_host", "ttdft_probe_fp64_peak", "ttdft_launch_count", "ttdft_last_error",
    "ttdft_h_set_math_mode", "ttdft_step_work_bytes", "ttdft_spmm_ws", "ttdft_cheb_step_ws", "ttdft_cheb_step_static",
    "ttdft_timing_enable", "ttdft_timing_read",
    "ttdft_gram_work_bytes", "ttdft_gram", "ttdft_project_work_bytes", "ttdft_project",
    "ttdft_rotate_work_bytes", "ttdft_rotate", "ttdft_orthonormalize_work_bytes", "ttdft_orthonormalize", "ttdft_orthonormalize_async",
    "ttdft_lanczos_work_bytes", "ttdft_lanczos_bounds",
    "ttdft_recover_subdomains_work_bytes", "ttdft_recover_subdomains",
]


class TTDFTError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"TTDFT_ERR_{_STATUS.get(status, status)}: {message}")
        self.status = status
        self.status_name = _STATUS.get(status, str(status))


class _Desc(ctypes.Structure):
    _fields_ = [("fmt", c_int32), ("M", c_int64), ("block", c_int32), ("row_ptr", c_void_p), ("col_idx", c_void_p),
                ("values", c_void_p), ("subdomain_of_row", c_void_p), ("flags", c_uint32), ("diag_values", c_void_p),
                ("diag_block", c_int64)]


class _Info(ctypes.Structure):
    _fields_ = [("M", c_int64), ("nnz_stored", c_int64), ("block", c_int32), ("kernel", c_int32), ("nblocks", c_int64),
                ("storage_bytes", c_size_t), ("i8_planes", c_int32), ("math", c_int32), ("reordered", c_int32), ("padded", c_int32),
                ("packed_bytes", c_int64)]


_lib = None


def library_path() -> str:
    return _LIB_PATH


def _load() -> ctypes.CDLL:
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_2110_15853_b200.build` "
                          "(there is no CPU fallback)")
    L = ctypes.CDLL(_LIB_PATH)
    st = c_int32
    L.ttdft_h_storage_bytes.restype = st
    L.ttdft_h_storage_bytes.argtypes = [POINTER(_Desc), POINTER(c_size_t)]
    L.ttdft_h_build.restype = st
    L.ttdft_h_build.argtypes = [POINTER(_Desc), c_void_p, c_size_t, c_void_p, POINTER(c_void_p)]
    L.ttdft_h_info.restype = st
    L.ttdft_h_info.argtypes = [c_void_p, POINTER(_Info)]
    L.ttdft_h_destroy.restype = st
    L.ttdft_h_destroy.argtypes = [c_void_p]
    L.ttdft_spmm.restype = st
    L.ttdft_spmm.argtypes = [c_void_p, c_double, c_void_p, c_int64, c_double, c_void_p, c_int64, c_int64, c_void_p]
    L.ttdft_cheb_step.restype = st
    L.ttdft_cheb_step.argtypes = [c_void_p, c_double, c_double, c_double, c_void_p, c_int64, c_void_p, c_int64, c_void_p,
                                  c_int64, c_int64, c_void_p]
    L.ttdft_cheb_step_static.restype = st
    L.ttdft_cheb_step_static.argtypes = list(L.ttdft_cheb_step.argtypes)
    L.ttdft_h_set_math_mode.restype = st
    L.ttdft_h_set_math_mode.argtypes = [c_void_p, c_int32]
    L.ttdft_step_work_bytes.restype = st
    L.ttdft_step_work_bytes.argtypes = [c_void_p, c_int64, POINTER(c_size_t)]
    L.ttdft_spmm_ws.restype = st
    L.ttdft_spmm_ws.argtypes = [c_void_p, c_double, c_void_p, c_int64, c_double, c_void_p, c_int64, c_int64, c_void_p, c_size_t,
                                c_void_p]
    L.ttdft_cheb_step_ws.restype = st
    L.ttdft_cheb_step_ws.argtypes = [c_void_p, c_double, c_double, c_double, c_void_p, c_int64, c_void_p, c_int64, c_void_p,
                                     c_int64, c_int64, c_void_p, c_size_t, c_void_p]
    L.ttdft_cheb_scalars.restype = st
    L.ttdft_cheb_scalars.argtypes = [c_int32, c_double, c_double, c_double, POINTER(c_double), POINTER(c_double),
                                     POINTER(c_double)]
    L.ttdft_cheb_filter_work_bytes.restype = st
    L.ttdft_cheb_filter_work_bytes.argtypes = [c_void_p, c_int64, c_int64, POINTER(c_size_t)]
    L.ttdft_cheb_filter_host_work_bytes.restype = st
    L.ttdft_cheb_filter_host_work_bytes.argtypes = [c_void_p, c_int64, c_int64, POINTER(c_size_t)]
    for name in ("ttdft_cheb_filter", "ttdft_cheb_filter_host"):
        fn = getattr(L, name)
        fn.restype = st
        fn.argtypes = [c_void_p, c_void_p, c_int64, c_void_p, c_int64, c_int64, c_int32, c_double, c_double, c_double,
                       c_int64, c_void_p, c_size_t, c_void_p]
    L.ttdft_gram_work_bytes.restype = st
    L.ttdft_gram_work_bytes.argtypes = [c_int64, c_int64, POINTER(c_size_t)]
    L.ttdft_gram.restype = st
    L.ttdft_gram.argtypes = [c_int64, c_void_p, c_int64, c_void_p, c_int64, c_int64, c_void_p, c_int64, c_void_p, c_size_t, c_void_p]
    L.ttdft_project_work_bytes.restype = st
    L.ttdft_project_work_bytes.argtypes = [c_void_p, c_int64, POINTER(c_size_t)]
    L.ttdft_project.restype = st
    L.ttdft_project.argtypes = [c_void_p, c_void_p, c_int64, c_int64, c_void_p, c_int64, c_void_p, c_size_t, c_void_p]
    L.ttdft_rotate_work_bytes.restype = st
    L.ttdft_rotate_work_bytes.argtypes = [c_int64, c_int64, c_int64, POINTER(c_size_t)]
    L.ttdft_rotate.restype = st
    L.ttdft_rotate.argtypes = [c_int64, c_void_p, c_int64, c_int64, c_void_p, c_int64, c_int64, c_void_p, c_int64, c_void_p, c_size_t, c_void_p]
    L.ttdft_orthonormalize_work_bytes.restype = st
    L.ttdft_orthonormalize_work_bytes.argtypes = [c_int64, c_int64, c_int32, POINTER(c_size_t)]
    L.ttdft_orthonormalize.restype = st
    L.ttdft_orthonormalize.argtypes = [c_int64, c_void_p, c_int64, c_int64, c_void_p, c_int64, c_int32, c_void_p, c_size_t, c_void_p]
    L.ttdft_orthonormalize_async.restype = st
    L.ttdft_orthonormalize_async.argtypes = [c_int64, c_void_p, c_int64, c_int64, c_void_p, c_int64, c_int32, c_void_p, c_size_t, c_void_p,
                                             c_void_p]
    L.ttdft_lanczos_work_bytes.restype = st
    L.ttdft_lanczos_work_bytes.argtypes = [c_void_p, POINTER(c_size_t)]
    L.ttdft_lanczos_bounds.restype = st
    L.ttdft_lanczos_bounds.argtypes = [c_void_p, c_int32, c_void_p, c_void_p, c_size_t, c_void_p, POINTER(c_double), POINTER(c_double),
                                       POINTER(c_double), POINTER(c_int32)]
    L.ttdft_recover_subdomains_work_bytes.restype = st
    L.ttdft_recover_subdomains_work_bytes.argtypes = [c_int64, POINTER(c_size_t)]
    L.ttdft_recover_subdomains.restype = st
    L.ttdft_recover_subdomains.argtypes = [POINTER(_Desc), c_void_p, c_void_p, c_size_t, c_void_p, POINTER(c_int32)]
    L.ttdft_probe_fp64_peak.restype = st
    L.ttdft_probe_fp64_peak.argtypes = [c_int32, c_int32, c_void_p, POINTER(c_double)]
    L.ttdft_timing_enable.restype = st
    L.ttdft_timing_enable.argtypes = [c_int32]
    L.ttdft_timing_read.restype = st
    L.ttdft_timing_read.argtypes = [c_int32, POINTER(c_double), POINTER(c_int64)]
    L.ttdft_launch_count.restype = c_int64
    L.ttdft_launch_count.argtypes = []
    L.ttdft_last_error.restype = c_char_p
    L.ttdft_last_error.argtypes = []
    _lib = L
    return L


def last_error() -> str:
    return _load().ttdft_last_error().decode()


KERNEL_IDS = {"bsr_dmma": 1, "generic": 2, "bsr_i8": 3, "y_digits": 4, "colmax": 5, "gram_i8": 6, "y_digits_fix": 7}


def timing_enable(on: bool = True):
    """ttdft_timing_enable: bracket the library's kernel launches with CUDA events on their stream."""
    _check(_load().ttdft_timing_enable(1 if on else 0))


def timing_read(kernel: str):
    """(total milliseconds, launches) of one kernel since the last read (ttdft_timing_read)."""
    ms, n = c_double(), c_int64()
    _check(_load().ttdft_timing_read(KERNEL_IDS[kernel], byref(ms), byref(n)))
    return ms.value, int(n.value)


def launch_count() -> int:
    return int(_load().ttdft_launch_count())


def _check(status: int):
    if status != 0:
        raise TTDFTError(status, last_error())


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2110_15853_b200 needs a CUDA device (no CPU fallback)")
    return torch


def _stream(stream=None) -> int:
    torch = _torch()
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def _keep(t, stream):
    """A scratch tensor allocated here and used by kernels on a foreign stream: tell the caching allocator, so that the
    memory is not handed out again before that stream has passed the call."""
    if stream is not None and t is not None:
        t.record_stream(stream)


def _mat(t, name="matrix"):
    """(device pointer, leading dimension) of a row-major fp64 CUDA matrix view."""
    torch = _torch()
    if t.dtype != torch.float64 or not t.is_cuda or t.dim() != 2:
        raise TypeError(f"{name} must be a 2-D float64 CUDA tensor")
    if t.shape[1] > 1 and t.stride(1) != 1:
        raise ValueError(f"{name} must be row-major with unit column stride")
    ld = t.stride(0) if t.shape[0] > 1 else max(t.shape[1], t.stride(0))
    return t.data_ptr(), int(ld)


class Hamiltonian:
    """A built H: owns the device storage tensor and the library handle (ttdft_h_t)."""

    def __init__(self, handle: int, storage, M: int):
        self._h = c_void_p(handle)
        self.storage = storage
        self.M = M

    @property
    def handle(self) -> c_void_p:
        if self._h is None:
            raise RuntimeError("Hamiltonian was destroyed")
        return self._h

    def info(self) -> dict:
        inf = _Info()
        _check(_load().ttdft_h_info(self.handle, byref(inf)))
        return {k: getattr(inf, k) for k, _ in _Info._fields_}

    def set_math_mode(self, mode: int):
        """ttdft_h_set_math_mode: MATH_AUTO / MATH_FP64 / MATH_I8 / MATH_I8X7 for the calls that take `work`."""
        _check(_load().ttdft_h_set_math_mode(self.handle, mode))
        return self

    def destroy(self):
        if self._h is not None:
            _load().ttdft_h_destroy(self._h)
            self._h = None
            self.storage = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def _desc(fmt, M, block, row_ptr, col_idx, values, subdomain_of_row, flags, diag_values=None, diag_block=0) -> _Desc:
    torch = _torch()
    for t, dt, nm in ((row_ptr, torch.int32, "row_ptr"), (col_idx, torch.int32, "col_idx"), (values, torch.float64, "values"),
                      (diag_values, torch.float64, "diag_values")):
        if t is not None and (t.dtype != dt or not t.is_cuda or not t.is_contiguous()):
            raise TypeError(f"{nm} must be a contiguous {dt} CUDA tensor")
    d = _Desc()
    d.fmt, d.M, d.block, d.flags = fmt, M, block, flags
    d.row_ptr = row_ptr.data_ptr() if row_ptr is not None else None
    d.col_idx = col_idx.data_ptr() if col_idx is not None and col_idx.numel() else None
    d.values = values.data_ptr() if values is not None and values.numel() else None
    d.subdomain_of_row = subdomain_of_row.data_ptr() if subdomain_of_row is not None else None
    d.diag_values = diag_values.data_ptr() if diag_values is not None and diag_values.numel() else None
    d.diag_block = diag_block
    return d


def h_storage_bytes(fmt, M, block, row_ptr, col_idx, values, subdomain_of_row=None, flags=0, diag_values=None, diag_block=0) -> int:
    d = _desc(fmt, M, block, row_ptr, col_idx, values, subdomain_of_row, flags, diag_values, diag_block)
    n = c_size_t()
    _check(_load().ttdft_h_storage_bytes(byref(d), byref(n)))
    return int(n.value)


def h_build(fmt, M, block, row_ptr, col_idx, values, subdomain_of_row=None, flags=0, stream=None, diag_values=None,
            diag_block=0) -> Hamiltonian:
    """ttdft_h_build: validate + convert H into library-format device storage (allocated here by torch)."""
    torch = _torch()
    d = _desc(fmt, M, block, row_ptr, col_idx, values, subdomain_of_row, flags, diag_values, diag_block)
    n = c_size_t()
    L = _load()
    _check(L.ttdft_h_storage_bytes(byref(d), byref(n)))
    dev = next((t.device for t in (values, diag_values, row_ptr) if t is not None), "cuda")
    storage = torch.empty(max(int(n.value), 1024) + 1024, dtype=torch.uint8, device=dev)
    base = storage.data_ptr()
    aligned = (base + 1023) // 1024 * 1024
    h = c_void_p()
    _check(L.ttdft_h_build(byref(d), c_void_p(aligned), c_size_t(int(n.value)), c_void_p(_stream(stream)), byref(h)))
    return Hamiltonian(h.value, storage, M)


def h_build_bsr(M, block, row_ptr, col_idx, values, flags=0, stream=None) -> Hamiltonian:
    return h_build(FMT_BSR, M, block, row_ptr, col_idx, values.reshape(-1), None, flags, stream)


def h_build_csr(M, row_ptr, col_idx, values, subdomain_of_row=None, flags=0, stream=None, recover=False) -> Hamiltonian:
    """CSR build.  recover=True and no labels: ttdft_recover_subdomains first, its labels (if any) go to ttdft_h_build."""
    if recover and subdomain_of_row is None and M > 0:
        try:
            subdomain_of_row, _ = recover_subdomains(M, row_ptr, col_idx, stream)
        except TTDFTError as e:
            if e.status_name != "UNSUPPORTED":      # pattern too large for the shared-memory column map: build without labels
                raise
    return h_build(FMT_CSR, M, 0, row_ptr, col_idx, values, subdomain_of_row, flags, stream)


def h_build_hybrid(M, diag_block, diag_values, row_ptr, col_idx, values, subdomain_of_row=None, flags=0, stream=None) -> Hamiltonian:
    """The paper's own layout: dense diagonal blocks (ceil(M / diag_block) row-major diag_block x diag_block
    blocks) + a CSR of the entries outside them.  Argument marshalling only: the union is formed by ttdft_h_build."""
    return h_build(FMT_HYBRID, M, 0, row_ptr, col_idx, values, subdomain_of_row, flags, stream, diag_values.reshape(-1), diag_block)


def step_work_bytes(H: Hamiltonian, ncols: int) -> int:
    n = c_size_t()
    _check(_load().ttdft_step_work_bytes(H.handle, ncols, byref(n)))
    return int(n.value)


def _work(H: Hamiltonian, ncols: int, work, device):
    """(aligned pointer, usable bytes, keep-alive tensor) of the scratch of the *_ws calls."""
    torch = _torch()
    if work is None:
        work = torch.empty(step_work_bytes(H, ncols) + 16, dtype=torch.uint8, device=device)
    wp = (work.data_ptr() + 15) // 16 * 16
    return wp, work.numel() * work.element_size() - (wp - work.data_ptr()), work


def spmm(H: Hamiltonian, alpha: float, X, beta: float, Y, stream=None, work=None, use_work=False):
    """Y = alpha*H*X + beta*Y (ttdft_spmm; with work / use_work: ttdft_spmm_ws in the handle's math mode)."""
    xp, ldx = _mat(X, "X")
    yp, ldy = _mat(Y, "Y")
    if X.shape != Y.shape or X.shape[0] != H.M:
        raise ValueError("shape mismatch")
    if work is not None or use_work:
        wp, wb, keep = _work(H, X.shape[1], work, X.device)
        _check(_load().ttdft_spmm_ws(H.handle, alpha, xp, ldx, beta, yp, ldy, X.shape[1], wp, wb, _stream(stream)))
        _keep(keep, stream)
        return Y
    _check(_load().ttdft_spmm(H.handle, alpha, xp, ldx, beta, yp, ldy, X.shape[1], _stream(stream)))
    return Y


def cheb_step(H: Hamiltonian, alpha: float, c: float, beta: float, Yk, Ykm1, Yout, stream=None, work=None, use_work=False):
    """Yout = alpha*(H*Yk - c*Yk) + beta*Ykm1 (ttdft_cheb_step[_ws]); Ykm1 None = beta term absent."""
    kp, ldk = _mat(Yk, "Yk")
    op, ldo = _mat(Yout, "Yout")
    mp, ldm = (None, 0) if Ykm1 is None else _mat(Ykm1, "Ykm1")
    if Yk.shape != Yout.shape or Yk.shape[0] != H.M or (Ykm1 is not None and Ykm1.shape != Yk.shape):
        raise ValueError("shape mismatch")
    if work is not None or use_work:
        wp, wb, keep = _work(H, Yk.shape[1], work, Yk.device)
        _check(_load().ttdft_cheb_step_ws(H.handle, alpha, c, beta, kp, ldk, mp, ldm, op, ldo, Yk.shape[1], wp, wb,
                                          _stream(stream)))
        _keep(keep, stream)
        return Yout
    _check(_load().ttdft_cheb_step(H.handle, alpha, c, beta, kp, ldk, mp, ldm, op, ldo, Yk.shape[1], _stream(stream)))
    return Yout


STATIC_SCRATCH_BYTES = 32 << 20


def cheb_step_static(H: Hamiltonian, alpha: float, c: float, beta: float, Yk, Ykm1, Yout, stream=None):
    """ttdft_cheb_step_static: the fused step in the handle's math mode with the library's own static device scratch (no device
    allocation by the library or by this binding; steps that need more than STATIC_SCRATCH_BYTES are rejected; calls that
    overlap on the GPU race on the shared scratch).  Argument marshalling only."""
    kp, ldk = _mat(Yk, "Yk")
    op, ldo = _mat(Yout, "Yout")
    mp, ldm = (None, 0) if Ykm1 is None else _mat(Ykm1, "Ykm1")
    if Yk.shape != Yout.shape or Yk.shape[0] != H.M or (Ykm1 is not None and Ykm1.shape != Yk.shape):
        raise ValueError("shape mismatch")
    _check(_load().ttdft_cheb_step_static(H.handle, alpha, c, beta, kp, ldk, mp, ldm, op, ldo, Yk.shape[1], _stream(stream)))
    return Yout


def cheb_scalars(m: int, a: float, b: float, a0: float):
    """(c, alpha[m], beta[m]) of Algorithm 1 (ttdft_cheb_scalars); host-only, needs no GPU."""
    n = max(m, 1)
    al = (c_double * n)()
    be = (c_double * n)()
    c = c_double()
    _check(_load().ttdft_cheb_scalars(m, a, b, a0, byref(c), al, be))
    return c.value, list(al)[:max(m, 0)], list(be)[:max(m, 0)]


def cheb_filter_work_bytes(H: Hamiltonian, ncols: int, panel_cols: int = 0) -> int:
    n = c_size_t()
    _check(_load().ttdft_cheb_filter_work_bytes(H.handle, ncols, panel_cols, byref(n)))
    return int(n.value)


def cheb_filter(H: Hamiltonian, X, Y, m: int, a: float, b: float, a0: float, panel_cols: int = 0, work=None, stream=None):
    """Y = p_m(H) X (ttdft_cheb_filter).  `work`: uint8/float64 CUDA tensor of >= cheb_filter_work_bytes."""
    torch = _torch()
    xp, ldx = _mat(X, "X")
    yp, ldy = _mat(Y, "Y")
    if X.shape != Y.shape or X.shape[0] != H.M:
        raise ValueError("shape mismatch")
    ncols = X.shape[1]
    if work is None:
        work = torch.empty(cheb_filter_work_bytes(H, ncols, panel_cols) + 16, dtype=torch.uint8, device=X.device)
    wp = (work.data_ptr() + 15) // 16 * 16
    wbytes = work.numel() * work.element_size() - (wp - work.data_ptr())
    _check(_load().ttdft_cheb_filter(H.handle, xp, ldx, yp, ldy, ncols, m, a, b, a0, panel_cols, wp, wbytes, _stream(stream)))
    _keep(work, stream)
    return Y


def cheb_filter_host_work_bytes(H: Hamiltonian, ncols: int, panel_cols: int = 0) -> int:
    n = c_size_t()
    _check(_load().ttdft_cheb_filter_host_work_bytes(H.handle, ncols, panel_cols, byref(n)))
    return int(n.value)


def cheb_filter_host(H: Hamiltonian, X_host, Y_host, m: int, a: float, b: float, a0: float, panel_cols: int = 0, work=None,
                     stream=None):
    """The filter with X, Y in HOST memory (CPU float64 tensors, pinned for speed); copies are inside the call."""
    torch = _torch()
    for t in (X_host, Y_host):
        if t.dtype != torch.float64 or t.is_cuda or t.dim() != 2 or (t.shape[1] > 1 and t.stride(1) != 1):
            raise TypeError("X_host/Y_host must be row-major 2-D float64 CPU tensors")
    if X_host.shape != Y_host.shape or X_host.shape[0] != H.M:
        raise ValueError("shape mismatch")
    ncols = X_host.shape[1]
    ldx = X_host.stride(0) if X_host.shape[0] > 1 else ncols
    ldy = Y_host.stride(0) if Y_host.shape[0] > 1 else ncols
    if work is None:
        work = torch.empty(cheb_filter_host_work_bytes(H, ncols, panel_cols) + 1024, dtype=torch.uint8, device="cuda")
    wp = (work.data_ptr() + 1023) // 1024 * 1024
    wbytes = work.numel() * work.element_size() - (wp - work.data_ptr())
    _check(_load().ttdft_cheb_filter_host(H.handle, X_host.data_ptr(), ldx, Y_host.data_ptr(), ldy, ncols, m, a, b, a0,
                                          panel_cols, wp, wbytes, _stream(stream)))
    return Y_host


def _aligned_work(nbytes: int, work, device):
    torch = _torch()
    if work is None:
        work = torch.empty(nbytes + 1024, dtype=torch.uint8, device=device)
    wp = (work.data_ptr() + 1023) // 1024 * 1024
    return wp, work.numel() * work.element_size() - (wp - work.data_ptr()), work


def gram_work_bytes(M: int, ncols: int) -> int:
    out = c_size_t(0)
    _check(_load().ttdft_gram_work_bytes(M, ncols, byref(out)))
    return int(out.value)


def gram(X, W, G, work=None, stream=None):
    """G = X^T W (ttdft_gram): X, W row-major M x N device float64, G row-major N x N."""
    xp, ldx = _mat(X, "X")
    wp_, ldw = _mat(W, "W")
    gp, ldg = _mat(G, "G")
    M, N = X.shape
    if W.shape != X.shape or tuple(G.shape) != (N, N):
        raise ValueError("shape mismatch")
    wp, wb, keep = _aligned_work(gram_work_bytes(M, N), work, X.device)
    _check(_load().ttdft_gram(M, xp, ldx, wp_, ldw, N, gp, ldg, wp, wb, _stream(stream)))
    _keep(keep, stream)
    return G


def project_work_bytes(H: Hamiltonian, ncols: int) -> int:
    out = c_size_t(0)
    _check(_load().ttdft_project_work_bytes(H.handle, ncols, byref(out)))
    return int(out.value)


def project(H: Hamiltonian, X, G, work=None, stream=None):
    """G = X^T (H X) (ttdft_project; Algorithm 1 step 3): X row-major M x N, G row-major N x N."""
    xp, ldx = _mat(X, "X")
    gp, ldg = _mat(G, "G")
    N = X.shape[1]
    if X.shape[0] != H.M or tuple(G.shape) != (N, N):
        raise ValueError("shape mismatch")
    wp, wb, keep = _aligned_work(project_work_bytes(H, N), work, X.device)
    _check(_load().ttdft_project(H.handle, xp, ldx, N, gp, ldg, wp, wb, _stream(stream)))
    _keep(keep, stream)
    return G


def rotate_work_bytes(M: int, k: int, n: int) -> int:
    out = c_size_t(0)
    _check(_load().ttdft_rotate_work_bytes(M, k, n, byref(out)))
    return int(out.value)


def rotate(X, Q, Y, work=None, stream=None):
    """Y = X Q (ttdft_rotate; Algorithm 1 step 5): X row-major M x k, Q row-major k x n, Y row-major M x n."""
    xp, ldx = _mat(X, "X")
    qp, ldq = _mat(Q, "Q")
    yp, ldy = _mat(Y, "Y")
    M, k = X.shape
    n = Q.shape[1]
    if Q.shape[0] != k or tuple(Y.shape) != (M, n):
        raise ValueError("shape mismatch")
    wp, wb, keep = _aligned_work(rotate_work_bytes(M, k, n), work, X.device)
    _check(_load().ttdft_rotate(M, xp, ldx, k, qp, ldq, n, yp, ldy, wp, wb, _stream(stream)))
    _keep(keep, stream)
    return Y


def orthonormalize_work_bytes(M: int, n: int, passes: int = 2) -> int:
    out = c_size_t(0)
    _check(_load().ttdft_orthonormalize_work_bytes(M, n, passes, byref(out)))
    return int(out.value)


def orthonormalize(X, Y, passes: int = 2, work=None, stream=None):
    """Y = X R^-1 with X^T X = R^T R (ttdft_orthonormalize; Algorithm 1 step 2): columns of Y are orthonormal."""
    xp, ldx = _mat(X, "X")
    yp, ldy = _mat(Y, "Y")
    M, n = X.shape
    if tuple(Y.shape) != (M, n):
        raise ValueError("shape mismatch")
    wp, wb, keep = _aligned_work(orthonormalize_work_bytes(M, n, passes), work, X.device)
    _check(_load().ttdft_orthonormalize(M, xp, ldx, n, yp, ldy, passes, wp, wb, _stream(stream)))
    _keep(keep, stream)
    return Y


def orthonormalize_async(X, Y, status, passes: int = 2, work=None, stream=None):
    """ttdft_orthonormalize_async: the same without any synchronisation (capturable into a CUDA graph).  status: int32 CUDA tensor
    of `passes` entries; entry p becomes 0, or 1 + the first non-positive pivot of pass p + 1 (Y is then meaningless)."""
    torch = _torch()
    xp, ldx = _mat(X, "X")
    yp, ldy = _mat(Y, "Y")
    M, n = X.shape
    if tuple(Y.shape) != (M, n):
        raise ValueError("shape mismatch")
    if status.dtype != torch.int32 or not status.is_cuda or not status.is_contiguous() or status.numel() < passes:
        raise TypeError("status must be a contiguous int32 CUDA tensor with one entry per pass")
    wp, wb, keep = _aligned_work(orthonormalize_work_bytes(M, n, passes), work, X.device)
    _check(_load().ttdft_orthonormalize_async(M, xp, ldx, n, yp, ldy, passes, wp, wb, c_void_p(status.data_ptr()), _stream(stream)))
    _keep(keep, stream)
    return Y


def lanczos_bounds(H: Hamiltonian, v0, k: int = 30, stream=None):
    """(a0, b, theta) from k Lanczos steps (ttdft_lanczos_bounds): a0 <= lambda_min (nearly always), b >= lambda_max, theta the Ritz values."""
    torch = _torch()
    if v0.dtype != torch.float64 or not v0.is_cuda or v0.dim() != 1 or v0.shape[0] != H.M or (H.M > 1 and v0.stride(0) != 1):
        raise TypeError("v0 must be a contiguous 1-D float64 CUDA tensor of length M")
    out = c_size_t(0)
    _check(_load().ttdft_lanczos_work_bytes(H.handle, byref(out)))
    wp, wb, keep = _aligned_work(int(out.value), None, v0.device)
    a0, b = c_double(0.0), c_double(0.0)
    theta = (c_double * 64)()
    steps = c_int32(0)
    _check(_load().ttdft_lanczos_bounds(H.handle, k, v0.data_ptr(), wp, wb, _stream(stream), byref(a0), byref(b), theta, byref(steps)))
    return a0.value, b.value, [theta[i] for i in range(steps.value)]


def recover_subdomains(M, row_ptr, col_idx, stream=None):
    """ttdft_recover_subdomains: (labels int32[M] CUDA tensor, n_groups) from the sparsity pattern of an unlabelled CSR;
    (None, 0) if the pattern has no recoverable structure.  Pass the labels as subdomain_of_row to h_build_csr."""
    torch = _torch()
    d = _desc(FMT_CSR, M, 0, row_ptr, col_idx, None, None, 0)
    out = c_size_t(0)
    _check(_load().ttdft_recover_subdomains_work_bytes(M, byref(out)))
    wp, wb, keep = _aligned_work(int(out.value), None, row_ptr.device)
    labels = torch.empty(max(M, 1), dtype=torch.int32, device=row_ptr.device)[:M]
    n = c_int32(0)
    _check(_load().ttdft_recover_subdomains(byref(d), labels.data_ptr(), wp, wb, _stream(stream), byref(n)))
    del keep
    return (labels, n.value) if n.value > 0 else (None, 0)


def probe_fp64_peak(kind: int = 1, millis: int = 200, stream=None) -> float:
    """Measured fp64 TFLOP/s of this GPU (0: DFMA loop, 1: DMMA m8n8k4 loop)."""
    v = c_double()
    _check(_load().ttdft_probe_fp64_peak(kind, millis, _stream(stream), byref(v)))
    return v.value
