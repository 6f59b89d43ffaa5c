"""Thin ctypes binding of libshg (include/shg.h).  Argument marshalling only: every step of the path runs
in the CUDA kernels.  PyTorch supplies device memory and streams, nothing else.

The library is loaded on first use; if ``libshg.so`` is missing (or cannot be loaded) an ImportError is
raised -- there is no CPU or PyTorch fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libshg.so")

SHG_OK, SHG_EINVAL, SHG_ESTATE, SHG_ECUDA, SHG_ENOMEM, SHG_ELIMIT = 0, -1, -2, -3, -4, -5
STATIC_MAX_BATCH = 256          # SHG_STATIC_MAX_BATCH
OPT_PERSISTENT, OPT_PRECISE, OPT_TRACE, OPT_ACQUIRE_FENCE, OPT_UNDEPLETED, OPT_SCHEME = 1, 2, 3, 4, 5, 6
OPT_SPIN_LIMIT, OPT_TABLES_SMEM, OPT_CLUSTER, OPT_PIPELINE = 7, 8, 9, 10

EXPORTS = ("shg_create", "shg_set_option", "shg_set_temperature", "shg_set_temperature_host", "shg_propagate",
           "shg_propagate_host", "shg_set_heat_output", "shg_power", "shg_power_history", "shg_gaussian_input",
           "shg_enable_timing", "shg_last_main_loop_ms", "shg_read_trace",
           "shg_last_launch_count", "shg_destroy", "shg_strerror", "shg_synchronize", "shg_history_length",
           "shg_history_nodes", "shg_last_cluster_size", "shg_last_kernel",
           "shg_field_power_static")


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("nzt", C.c_int32),
                ("batch", C.c_int32), ("record_every", C.c_int32)]


class Crystal(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("L", "lambda1", "n1", "n2", "d_eff", "dk0", "ddk_dT", "T_pm",
                                          "alpha1", "alpha2", "beta1", "beta2", "rho1", "rho2")]


class Beam(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("P", "w0", "focus_z", "lx", "ly")]


class ShgError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libshg error %d: %s" % (code, msg))
        self.code = code


_lib = None


def lib():
    """Load libshg.so (once).  Fails loudly when the CUDA extension is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libshg.so not found at %s -- build it with `python -m paper_2410_04994_b200.build` "
                          "(there is no CPU fallback)" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    vp, dp = C.c_void_p, C.POINTER(C.c_double)
    L.shg_create.argtypes = [C.POINTER(Grid), C.POINTER(Crystal), C.POINTER(Beam), C.POINTER(vp)]
    L.shg_set_option.argtypes = [vp, C.c_int, C.c_int]
    L.shg_set_temperature.argtypes = [vp, vp, C.c_double, C.c_int]
    L.shg_set_temperature_host.argtypes = [vp, vp, C.c_double, C.c_int, vp]
    L.shg_propagate.argtypes = [vp, vp, vp, vp, vp, C.c_int, vp]
    L.shg_propagate_host.argtypes = [vp, vp, vp, vp, vp, C.c_int, vp]
    L.shg_power.argtypes = [vp, C.c_int, C.c_double, dp, dp]
    L.shg_power_history.argtypes = [vp, C.c_int, vp]
    L.shg_synchronize.argtypes = [vp]
    L.shg_history_length.argtypes = [vp]
    L.shg_history_nodes.argtypes = [vp, vp]
    L.shg_gaussian_input.argtypes = [vp, vp, C.c_int, vp]
    L.shg_enable_timing.argtypes = [vp, C.c_int]
    L.shg_last_main_loop_ms.argtypes = [vp, C.POINTER(C.c_float)]
    L.shg_read_trace.argtypes = [vp, vp, C.POINTER(C.c_int), C.POINTER(C.c_int)]
    L.shg_last_launch_count.argtypes = [vp]
    L.shg_last_cluster_size.argtypes = [vp]
    L.shg_last_kernel.argtypes = [vp]
    L.shg_set_heat_output.argtypes = [vp, vp, C.c_int]
    L.shg_field_power_static.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, vp, vp]
    L.shg_destroy.argtypes = [vp]
    L.shg_destroy.restype = None
    L.shg_strerror.argtypes = [C.c_int]
    L.shg_strerror.restype = C.c_char_p
    _lib = L
    return L


def _check(rc):
    if rc != SHG_OK:
        raise ShgError(rc, lib().shg_strerror(rc).decode())


def _mk(struct, d):
    s = struct()
    for k, _ in struct._fields_:
        if k in d:
            setattr(s, k, d[k])
    return s


def _stream_ptr(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(int(stream.cuda_stream))


def _dev_ptr(t, dtype_names):
    import torch
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
        raise TypeError("expected a contiguous CUDA tensor")
    if str(t.dtype).replace("torch.", "") not in dtype_names:
        raise TypeError("expected dtype in %s, got %s" % (dtype_names, t.dtype))
    return C.c_void_p(t.data_ptr())


def field_power_static(A1, A2, scale1: float, scale2: float, out, stream=None):
    """shg_field_power_static: out[b][j] = scale_j * sum |A_j[b]|^2 with no context and no allocation.

    For callers that may not allocate device memory (code running inside another allocator, a host application that
    owns all of HBM, a loop that cannot take the driver's allocation lock): this wrapper allocates nothing either, so
    the caller passes every buffer.  A1, A2 (or None): CUDA complex64 [batch][ny][nx]; out: CUDA float64 [batch][2],
    written on `stream` (default: torch's current stream) -- synchronise before reading it.  batch is at most
    STATIC_MAX_BATCH; beyond it the call raises ShgError (SHG_ELIMIT) and enqueues nothing.  All calls on a device
    share one fixed scratch array inside the library: do not let two of them overlap on the GPU.  The first call on
    a device looks the array up; make it before any stream capture.  See include/shg.h.
    """
    if A1.dim() != 3:
        raise ValueError("A1 must be [batch][ny][nx]")
    batch, ny, nx = A1.shape
    if A2 is not None and tuple(A2.shape) != tuple(A1.shape):
        raise ValueError("A2 must have the shape of A1")
    if out.numel() != 2 * batch:
        raise ValueError("out must hold batch*2 float64 values")
    _check(lib().shg_field_power_static(_dev_ptr(A1, ("complex64",)), _dev_ptr(A2, ("complex64",)), nx, ny, batch,
                                        float(scale1), float(scale2), _dev_ptr(out, ("float64",)),
                                        _stream_ptr(stream)))
    return out


class Shg:
    """One libshg context (``shg_create`` .. ``shg_destroy``).

    grid / crystal / beams are the dictionaries of ``workloads.make`` (field names of include/shg.h).
    """

    def __init__(self, grid: dict, crystal: dict, beams, persistent: bool | None = None,
                 precise: bool | None = None):
        L = lib()
        beams = list(beams)
        self.grid = dict(grid)
        self.grid.setdefault("batch", len(beams))
        self.grid.setdefault("nzt", 0)
        self.crystal = dict(crystal)
        self.beams = beams
        arr = (Beam * len(beams))(*[_mk(Beam, b) for b in beams])
        h = C.c_void_p()
        _check(L.shg_create(C.byref(_mk(Grid, self.grid)), C.byref(_mk(Crystal, crystal)), arr, C.byref(h)))
        self._h = h
        self._keep = []
        if persistent is not None:
            self.set_option(OPT_PERSISTENT, int(persistent))
        if precise is not None:
            self.set_option(OPT_PRECISE, int(precise))

    # -- shg_set_option
    def set_option(self, option: int, value: int):
        _check(lib().shg_set_option(self._h, option, value))
        return self

    # -- shg_set_temperature (device tensor, borrowed) / shg_set_temperature_host (numpy or pinned tensor)
    def set_temperature(self, T=None, T_uniform: float = 0.0, per_member: bool = False, stream=None):
        import torch
        if T is None:
            _check(lib().shg_set_temperature(self._h, None, float(T_uniform), int(per_member)))
        elif isinstance(T, torch.Tensor) and T.is_cuda:
            self._check_T(T.numel(), per_member)
            self._keep = [T]
            _check(lib().shg_set_temperature(self._h, _dev_ptr(T, ("float32",)), float(T_uniform), int(per_member)))
        else:
            host = T if isinstance(T, torch.Tensor) else np.ascontiguousarray(T, dtype=np.float32)
            n = host.numel() if isinstance(host, torch.Tensor) else host.size
            self._check_T(n, per_member)
            ptr = host.data_ptr() if isinstance(host, torch.Tensor) else host.ctypes.data
            self._keep = [host]
            _check(lib().shg_set_temperature_host(self._h, C.c_void_p(ptr), float(T_uniform), int(per_member),
                                                  _stream_ptr(stream)))
        return self

    def _check_T(self, numel, per_member):
        g = self.grid
        want = (g["batch"] if per_member else 1) * g["nzt"] * g["ny"] * g["nx"]
        if numel != want:
            raise ValueError("T has %d elements, expected %d" % (numel, want))

    # -- shg_propagate: CUDA complex64 tensors [batch][ny][nx]
    def propagate(self, A1_in, A2_in=None, A1_out=None, A2_out=None, stream=None, batch=None):
        """A1_in None: the library's own Gaussian pump of Eq. 6 (then `batch` members, default the capacity)."""
        import torch
        g = self.grid
        if A1_in is None:
            batch = g["batch"] if batch is None else batch
            shape = (batch, g["ny"], g["nx"])
            if A1_out is None:
                A1_out = torch.empty(shape, dtype=torch.complex64, device="cuda")
            if A2_out is None:
                A2_out = torch.empty(shape, dtype=torch.complex64, device="cuda")
        else:
            A1_in = A1_in.reshape(-1, g["ny"], g["nx"])
            batch = A1_in.shape[0]
            if A1_out is None:
                A1_out = torch.empty_like(A1_in)
            if A2_out is None:
                A2_out = torch.empty_like(A1_in)
        for t in (A1_in, A2_in, A1_out, A2_out):
            if t is not None and t.numel() != batch * g["ny"] * g["nx"]:
                raise ValueError("field tensors must hold batch*ny*nx complex64 values")
        _check(lib().shg_propagate(self._h, _dev_ptr(A1_in, ("complex64",)), _dev_ptr(A2_in, ("complex64",)),
                                   _dev_ptr(A1_out, ("complex64",)), _dev_ptr(A2_out, ("complex64",)),
                                   batch, _stream_ptr(stream)))
        return A1_out, A2_out

    # -- shg_set_heat_output: Q is a CUDA float32 tensor [batch][nq][ny][nx] (kept alive here), None = off
    def set_heat_output(self, Q=None):
        g = self.grid
        if Q is None:
            self._Q = None
            _check(lib().shg_set_heat_output(self._h, None, 0))
            return self
        if Q.dim() != 4 or Q.shape[0] != g["batch"] or Q.shape[2] != g["ny"] or Q.shape[3] != g["nx"]:
            raise ValueError("Q must be [batch][nq][ny][nx]")
        self._Q = Q
        _check(lib().shg_set_heat_output(self._h, _dev_ptr(Q, ("float32",)), int(Q.shape[1])))
        return self

    # -- shg_propagate_host: numpy complex64 arrays or (pinned) CPU tensors
    def propagate_host(self, A1_in, A2_in=None, A1_out=None, A2_out=None, stream=None):
        g = self.grid

        def ptr(a):
            if a is None:
                return None
            return C.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data)

        def numel(a):
            return a.numel() if hasattr(a, "numel") else a.size
        batch = numel(A1_in) // (g["ny"] * g["nx"])
        if A1_out is None:
            A1_out = np.empty((batch, g["ny"], g["nx"]), np.complex64)
        if A2_out is None:
            A2_out = np.empty((batch, g["ny"], g["nx"]), np.complex64)
        _check(lib().shg_propagate_host(self._h, ptr(A1_in), ptr(A2_in), ptr(A1_out), ptr(A2_out), batch,
                                        _stream_ptr(stream)))
        return A1_out, A2_out

    # -- shg_power / shg_power_history
    def power(self, member: int, z: float):
        p1, p2 = C.c_double(), C.c_double()
        _check(lib().shg_power(self._h, member, float(z), C.byref(p1), C.byref(p2)))
        return p1.value, p2.value

    def power_history(self, member: int = 0) -> np.ndarray:
        out = np.empty((lib().shg_history_length(self._h), 2), dtype=np.float64)
        _check(lib().shg_power_history(self._h, member, C.c_void_p(out.ctypes.data)))
        return out

    def history_nodes(self) -> np.ndarray:
        """Step indices n of the recorded nodes (shg_grid.record_every)."""
        out = np.empty(lib().shg_history_length(self._h), dtype=np.int32)
        _check(lib().shg_history_nodes(self._h, C.c_void_p(out.ctypes.data)))
        return out

    def synchronize(self):
        """shg_synchronize: wait for the last propagate; raises if the run failed."""
        _check(lib().shg_synchronize(self._h))
        return self

    def efficiency(self, member: int = 0) -> float:
        """eta = P2(L) / (P1(0) + P2(0))  (on-grid input power)."""
        h = self.power_history(member)
        return float(h[-1, 1] / (h[0, 0] + h[0, 1]))

    # -- shg_gaussian_input
    def gaussian_input(self, batch=None, stream=None):
        import torch
        g = self.grid
        batch = g["batch"] if batch is None else batch
        A = torch.empty((batch, g["ny"], g["nx"]), dtype=torch.complex64, device="cuda")
        _check(lib().shg_gaussian_input(self._h, _dev_ptr(A, ("complex64",)), batch, _stream_ptr(stream)))
        return A

    def enable_timing(self, on: bool = True):
        _check(lib().shg_enable_timing(self._h, int(on)))
        return self

    def last_main_loop_ms(self) -> float:
        ms = C.c_float()
        _check(lib().shg_last_main_loop_ms(self._h, C.byref(ms)))
        return float(ms.value)

    def read_trace(self) -> np.ndarray:
        """int64 [steps][grid][2][4] phase timeline (see SHG_OPT_TRACE in include/shg.h)."""
        steps, grid = C.c_int(), C.c_int()
        _check(lib().shg_read_trace(self._h, None, C.byref(steps), C.byref(grid)))
        out = np.zeros((steps.value, grid.value, 2, 4), dtype=np.int64)
        _check(lib().shg_read_trace(self._h, C.c_void_p(out.ctypes.data), C.byref(steps), C.byref(grid)))
        return out

    def last_launch_count(self) -> int:
        return int(lib().shg_last_launch_count(self._h))

    def last_cluster_size(self) -> int:
        return int(lib().shg_last_cluster_size(self._h))

    def last_kernel(self) -> int:
        """0 k_row + k_col, 1 k_persist, 2 k_persist_flat, 3 k_persist_pipe, 4 k_cluster, 5 k_persist_paper."""
        return int(lib().shg_last_kernel(self._h))

    def close(self):
        if getattr(self, "_h", None):
            lib().shg_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
