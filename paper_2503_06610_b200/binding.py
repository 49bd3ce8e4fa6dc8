"""ctypes binding of libnh_b200.so -- argument marshalling only (include/nh.h is the contract).

Function names mirror the C ABI: init_lattice / set_director / step / get_fields.  PyTorch is
used for device memory (the workspace tensor) and the CUDA stream, nothing else.  There is no
CPU path: constructing a Lattice without a CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libnh_b200.so")

FP64_SHIFTED, FP32_SHIFTED, FP32_UNSHIFTED, FP64_UNSHIFTED = 0, 1, 2, 3
OPT_GRAPH, OPT_TIMING, OPT_FD_DIRECT, OPT_NO_SERPENTINE, OPT_FD_NOVEC, OPT_LB_TWOSTEP, OPT_LB_ONESTEP = 1, 2, 4, 16, 32, 64, 128
OPT_CHECK_FINITE = 256
# keys of nh_debug_tune (include/nh_debug.h: tuning and test hooks, not part of the contract)
TUNE = {"fd_planes": 0, "lb2_lead": 1, "lb2_ring": 2, "lb2_strips": 3, "lb2_cells": 4, "lb2_threads": 5,
        "lb2_blockorder": 6, "lb2_timeout_ms": 7, "lb2_fault": 8}
KERNEL_CLASSES = ("lb", "velocity", "predictor", "corrector", "force", "other", "lb2")

EXPORTS = ("nh_workspace_bytes", "nh_init_lattice", "nh_set_director", "nh_step", "nh_get_fields",
           "nh_time", "nh_launch_count", "nh_set_options", "nh_kernel_time", "nh_free", "nh_last_error",
           "nh_rows_bytes", "nh_get_rows", "nh_set_rows", "nh_update_force", "nh_defer_force", "nh_debug_tune",
           "nh_get_rows_pair", "nh_set_rows_pair", "nh_lb_two_steps_noalloc")
NOALLOC_SCRATCH_BYTES = 16 * 1024 * 1024      # NH_NOALLOC_SCRATCH_BYTES of include/nh_noalloc.h


class NhParams(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("tau", C.c_double), ("K", C.c_double), ("pitch", C.c_double),
                ("xi", C.c_double), ("gamma1", C.c_double), ("g", C.c_double * 3),
                ("anchoring", C.c_int), ("W0", C.c_double), ("fd_ratio", C.c_int),
                ("precision", C.c_int), ("coupling", C.c_int), ("alpha", C.c_double * 6),
                ("K3", C.c_double * 3)]


FIELDS = ("populations", "director", "velocity", "force")   # NH_FIELD_* of include/nh.h, in order


class NhError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("nh error %d: %s" % (code, msg))
        self.code = code


_lib = None


def load():
    """Load the in-tree library (built by paper_2503_06610_b200.build); fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s is missing: run `python -m paper_2503_06610_b200.build` "
                              "(there is no fallback path)" % LIB_PATH)
        lib = C.CDLL(LIB_PATH)
        dp = C.POINTER(C.c_double)
        lib.nh_workspace_bytes.argtypes = [C.POINTER(NhParams)]
        lib.nh_workspace_bytes.restype = C.c_size_t
        lib.nh_init_lattice.argtypes = [C.POINTER(NhParams), C.c_void_p, C.c_size_t, C.c_void_p,
                                        C.POINTER(C.c_void_p)]
        lib.nh_set_director.argtypes = [C.c_void_p, C.c_void_p]
        lib.nh_step.argtypes = [C.c_void_p, C.c_int, C.c_int]
        lib.nh_get_fields.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.nh_time.argtypes = [C.c_void_p]
        lib.nh_time.restype = C.c_long
        lib.nh_launch_count.argtypes = [C.c_void_p]
        lib.nh_launch_count.restype = C.c_long
        lib.nh_set_options.argtypes = [C.c_void_p, C.c_int]
        lib.nh_kernel_time.argtypes = [C.c_void_p, C.c_int, dp, C.POINTER(C.c_long)]
        lib.nh_rows_bytes.argtypes = [C.c_void_p, C.c_int, C.c_int]
        lib.nh_rows_bytes.restype = C.c_size_t
        lib.nh_get_rows.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p]
        lib.nh_set_rows.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p]
        lib.nh_get_rows_pair.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]
        lib.nh_set_rows_pair.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]
        lib.nh_update_force.argtypes = [C.c_void_p]
        lib.nh_defer_force.argtypes = [C.c_void_p, C.c_int]
        lib.nh_debug_tune.argtypes = [C.c_void_p, C.c_int, C.c_int]
        lib.nh_lb_two_steps_noalloc.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.POINTER(C.c_double),
                                                C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.nh_free.argtypes = [C.c_void_p]
        lib.nh_free.restype = None
        lib.nh_last_error.restype = C.c_char_p
        _lib = lib
    return _lib


def _check(rc):
    if rc != 0:
        raise NhError(rc, load().nh_last_error().decode())


def make_params(nx, ny, nz, tau, K=0.0, pitch=0.0, xi=0.0, gamma1=1.0, g=(0.0, 0.0, 0.0), anchoring=0,
                W0=0.0, fd_ratio=1, precision=FP32_SHIFTED, coupling=3, alpha=(0.0,) * 6, K3=(0.0, 0.0, 0.0)) -> NhParams:
    return NhParams(nx, ny, nz, tau, K, pitch, xi, gamma1, (C.c_double * 3)(*g), anchoring, W0,
                    fd_ratio, precision, coupling, (C.c_double * 6)(*alpha), (C.c_double * 3)(*K3))


def workspace_bytes(params: NhParams) -> int:
    return int(load().nh_workspace_bytes(C.byref(params)))


def _host_ptr(a):
    """Pointer of a host FP64 buffer: numpy array or (pinned) CPU torch tensor; None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    import torch
    assert isinstance(a, torch.Tensor) and a.device.type == "cpu" and a.dtype == torch.float64
    assert a.is_contiguous()
    return a.data_ptr()


def lb_two_steps_noalloc(nx, ny, nz, precision, tau, g, f_in, F_lc, f_out, stream=None):
    """nh_lb_two_steps_noalloc (include/nh_noalloc.h): f_out := two LB steps of f_in, for callers that may not allocate
    device memory -- the kernel's ring and flags sit in an array inside the library, nothing is allocated here or there.
    f_in, f_out: CUDA tensors holding [19][nz][ny][nx] words of the precision's type; F_lc: [3][nz][ny][nx] or None.
    All on the current device; `stream` a torch stream of that device (default: the current one).  Returns when done."""
    import torch
    for t in (f_in, f_out) + ((F_lc,) if F_lc is not None else ()):
        assert t.is_cuda and t.is_contiguous()
    s = stream if stream is not None else torch.cuda.current_stream(f_in.device)
    _check(load().nh_lb_two_steps_noalloc(int(nx), int(ny), int(nz), int(precision), float(tau), (C.c_double * 3)(*g),
                                          f_in.data_ptr(), F_lc.data_ptr() if F_lc is not None else None,
                                          f_out.data_ptr(), s.cuda_stream))


class Lattice:
    """One lattice on the current CUDA device.  Thin wrapper: every method is one C-ABI call."""

    def __init__(self, nx, ny, nz, tau, device="cuda:0", stream=None, workspace=None, **kw):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2503_06610_b200 needs a CUDA device (no CPU fallback)")
        lib = load()
        self.params = make_params(nx, ny, nz, tau, **kw)
        self.shape = (nz, ny, nx)
        nbytes = workspace_bytes(self.params)
        if nbytes == 0:
            _check(lib.nh_init_lattice(C.byref(self.params), None, 0, None, C.byref(C.c_void_p())))
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        if workspace is None:
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            off = (-self._ws.data_ptr()) % 256
        else:       # the caller's own device memory (uint8 CUDA tensor, 256-byte aligned, >= workspace_bytes)
            assert workspace.is_cuda and workspace.dtype == torch.uint8 and workspace.is_contiguous()
            assert workspace.numel() >= nbytes and workspace.data_ptr() % 256 == 0
            self._ws, off = workspace, 0
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._h = C.c_void_p()
        _check(lib.nh_init_lattice(C.byref(self.params), self._ws.data_ptr() + off, nbytes,
                                   self._stream.cuda_stream, C.byref(self._h)))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load().nh_free(self._h)
            self._h = C.c_void_p()
        self._ws = None

    __del__ = close

    def set_director(self, n):
        if isinstance(n, np.ndarray):
            n = np.ascontiguousarray(n, dtype=np.float64)
            assert n.shape == (3,) + self.shape
        _check(load().nh_set_director(self._h, _host_ptr(n)))

    def step(self, n_lb, n_fd=-1):
        _check(load().nh_step(self._h, int(n_lb), int(n_fd)))

    def get_fields(self, out=None, which=("rho", "u", "n", "F")):
        """Returns dict of numpy FP64 arrays; `out` may hold preallocated (pinned) host buffers."""
        out = dict(out or {})
        for k in which:
            if k not in out:
                out[k] = np.empty(self.shape if k == "rho" else (3,) + self.shape)
        ptr = {k: _host_ptr(out.get(k)) if k in which else None for k in ("rho", "u", "n", "F")}
        _check(load().nh_get_fields(self._h, ptr["rho"], ptr["u"], ptr["n"], ptr["F"]))
        return {k: out[k] for k in which}

    @property
    def time(self):
        return int(load().nh_time(self._h))

    @property
    def launch_count(self):
        return int(load().nh_launch_count(self._h))

    def set_options(self, options):
        _check(load().nh_set_options(self._h, int(options)))

    def debug_tune(self, **knobs):
        """nh_debug_tune for each name=value (names: binding.TUNE); 0 = the library decides."""
        for name, value in knobs.items():
            _check(load().nh_debug_tune(self._h, TUNE[name], int(value)))

    def kernel_time(self, which):
        """(total ms, launches) of a kernel class since the last set_options (needs OPT_TIMING)."""
        k = KERNEL_CLASSES.index(which) if isinstance(which, str) else int(which)
        ms, cnt = C.c_double(0.0), C.c_long(0)
        _check(load().nh_kernel_time(self._h, k, C.byref(ms), C.byref(cnt)))
        return ms.value, cnt.value

    def synchronize(self):
        self._stream.synchronize()

    # ---- halo rows of a y-slab (include/nh.h, "Slab decomposition along y") ----
    def rows_bytes(self, field, nrows):
        return int(load().nh_rows_bytes(self._h, FIELDS.index(field), int(nrows)))

    def new_rows_buffer(self, field, nrows):
        """Device buffer that holds `nrows` packed rows of `field` ([component][z][row][x], storage type)."""
        import torch
        return torch.empty(self.rows_bytes(field, nrows), dtype=torch.uint8, device=self.device)

    def get_rows(self, field, y0, nrows, buf):
        assert buf.is_cuda and buf.is_contiguous() and buf.numel() * buf.element_size() >= self.rows_bytes(field, nrows)
        _check(load().nh_get_rows(self._h, FIELDS.index(field), int(y0), int(nrows), buf.data_ptr()))

    def set_rows(self, field, y0, nrows, buf):
        assert buf.is_cuda and buf.is_contiguous() and buf.numel() * buf.element_size() >= self.rows_bytes(field, nrows)
        _check(load().nh_set_rows(self._h, FIELDS.index(field), int(y0), int(nrows), buf.data_ptr()))

    def get_rows_pair(self, field, y0_a, y0_b, nrows, buf):
        """Rows [y0_a, +nrows) and [y0_b, +nrows) into the two halves of `buf` (2 x rows_bytes), one launch."""
        assert buf.is_cuda and buf.is_contiguous() and buf.numel() * buf.element_size() >= 2 * self.rows_bytes(field, nrows)
        _check(load().nh_get_rows_pair(self._h, FIELDS.index(field), int(y0_a), int(y0_b), int(nrows), buf.data_ptr()))

    def set_rows_pair(self, field, y0_a, y0_b, nrows, buf):
        assert buf.is_cuda and buf.is_contiguous() and buf.numel() * buf.element_size() >= 2 * self.rows_bytes(field, nrows)
        _check(load().nh_set_rows_pair(self._h, FIELDS.index(field), int(y0_a), int(y0_b), int(nrows), buf.data_ptr()))

    def update_force(self):
        _check(load().nh_update_force(self._h))

    def defer_force(self, on=True):
        _check(load().nh_defer_force(self._h, 1 if on else 0))
