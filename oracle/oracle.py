"""ctypes binding of ``liboracle.so`` (oracle/shg_oracle.c).  TEST INFRASTRUCTURE ONLY.

Argument marshalling only; every number is computed by the C oracle.  Fields are complex128 numpy
arrays ``[batch][ny][nx]``; temperatures are float32 ``[members][nzt][ny][nx]``.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "shg_oracle.c")
_HDR = os.path.join(_HERE, "shg_oracle.h")
_LIB = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("nzt", C.c_int32),
                ("batch", C.c_int32)]


class Crystal(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("L", "lambda1", "n1", "n2", "d_eff", "dk0", "ddk_dT", "T_pm",
                                          "alpha1", "alpha2", "beta1", "beta2", "rho1", "rho2")]


class Beam(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("P", "w0", "focus_z", "lx", "ly")]


class Options(C.Structure):
    _fields_ = [("scheme", C.c_int32), ("undepleted", C.c_int32), ("brute_dft", C.c_int32),
                ("merged", C.c_int32)]


def build(force: bool = False) -> str:
    """Compile oracle/shg_oracle.c -> oracle/liboracle.so with gcc (-O2 -fopenmp, no -ffast-math)."""
    with _lock:
        stale = (not os.path.exists(_LIB)
                 or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)))
        if force or stale:
            tmp = _LIB + ".%d.tmp" % os.getpid()
            subprocess.check_call(["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-Wall",
                                   "-o", tmp, _SRC, "-lm"])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(build())
    dp = C.POINTER(C.c_double)
    lib.orc_create.argtypes = [C.POINTER(Grid), C.POINTER(Crystal), C.POINTER(Beam), C.POINTER(Options),
                               C.POINTER(C.c_void_p)]
    lib.orc_set_temperature.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_int]
    lib.orc_propagate.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
    lib.orc_set_heat_output.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
    lib.orc_power.argtypes = [C.c_void_p, C.c_int, C.c_double, dp, dp]
    lib.orc_power_history.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
    lib.orc_destroy.argtypes = [C.c_void_p]
    lib.orc_destroy.restype = None
    lib.orc_gaussian_input.argtypes = [C.POINTER(Grid), C.POINTER(Crystal), C.POINTER(Beam), C.c_void_p]
    lib.orc_set_num_threads.argtypes = [C.c_int]
    lib.orc_set_num_threads.restype = None
    lib.orc_fft2.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
    lib.orc_dft2_brute.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int]
    lib.orc_num_threads.restype = C.c_int
    _lib = lib
    return lib


def set_num_threads(n: int) -> None:
    _load().orc_set_num_threads(int(n))


def num_threads() -> int:
    return int(_load().orc_num_threads())


def fft2(a: np.ndarray, sign: int) -> np.ndarray:
    """Own radix-2 2-D transform.  sign=-1 forward (unnormalised), +1 inverse (1/(nx ny))."""
    out = np.ascontiguousarray(a, dtype=np.complex128).copy()
    ny, nx = out.shape
    rc = _load().orc_fft2(out.ctypes.data, ny, nx, sign)
    if rc:
        raise ValueError("orc_fft2 failed: %d" % rc)
    return out


def dft2_brute(a: np.ndarray, sign: int) -> np.ndarray:
    """The 2-D DFT definition, O((nx ny)^2)."""
    src = np.ascontiguousarray(a, dtype=np.complex128)
    out = np.empty_like(src)
    ny, nx = src.shape
    rc = _load().orc_dft2_brute(src.ctypes.data, out.ctypes.data, ny, nx, sign)
    if rc:
        raise ValueError("orc_dft2_brute failed: %d" % rc)
    return out


def _mk(struct, d):
    s = struct()
    for k, _ in struct._fields_:
        if k in d:
            setattr(s, k, d[k])
    return s


def gaussian_input(grid: dict, crystal: dict, beam: dict) -> np.ndarray:
    """Eq. 6 / Eq. 5 input on the grid of one member, complex128 [ny][nx]."""
    g = _mk(Grid, dict(grid, batch=1))
    out = np.empty((grid["ny"], grid["nx"]), dtype=np.complex128)
    rc = _load().orc_gaussian_input(C.byref(g), C.byref(_mk(Crystal, crystal)), C.byref(_mk(Beam, beam)),
                                    out.ctypes.data)
    if rc:
        raise ValueError("orc_gaussian_input failed: %d" % rc)
    return out


class Oracle:
    """One oracle context: ``Oracle(grid, crystal, beams).set_temperature(...).propagate(A1, A2)``."""

    def __init__(self, grid: dict, crystal: dict, beams, scheme: int = 0, undepleted: bool = False,
                 brute_dft: bool = False, merged: bool = False):
        lib = _load()
        beams = list(beams)
        self.grid = dict(grid)
        self.grid.setdefault("batch", len(beams))
        self.grid.setdefault("nzt", 0)
        self.crystal = dict(crystal)
        self.beams = beams
        g = _mk(Grid, self.grid)
        arr = (Beam * len(beams))(*[_mk(Beam, b) for b in beams])
        opt = Options(int(scheme), int(bool(undepleted)), int(bool(brute_dft)), int(bool(merged)))
        h = C.c_void_p()
        rc = lib.orc_create(C.byref(g), C.byref(_mk(Crystal, crystal)), arr, C.byref(opt), C.byref(h))
        if rc:
            raise ValueError("orc_create failed: %d" % rc)
        self._h = h
        self._T = None
        self._Q = None

    def set_temperature(self, T=None, T_uniform: float = 0.0, per_member: bool = False):
        ptr = None
        if T is not None:
            self._T = np.ascontiguousarray(T, dtype=np.float32)
            members = self.grid["batch"] if per_member else 1
            want = members * self.grid["nzt"] * self.grid["ny"] * self.grid["nx"]
            if self._T.size != want:
                raise ValueError("T has %d elements, expected %d" % (self._T.size, want))
            ptr = self._T.ctypes.data
        rc = _load().orc_set_temperature(self._h, ptr, float(T_uniform), int(per_member))
        if rc:
            raise ValueError("orc_set_temperature failed: %d" % rc)
        return self

    def set_heat_output(self, nq: int):
        """Ask the next propagate for the heat source of P:118 (Eq. 8) on nq planes; returns the float64 array
        [batch][nq][ny][nx] that the propagate fills (nq = 0 switches it off)."""
        if nq <= 0:
            self._Q = None
            rc = _load().orc_set_heat_output(self._h, None, 0)
        else:
            self._Q = np.zeros((self.grid["batch"], nq, self.grid["ny"], self.grid["nx"]), dtype=np.float64)
            rc = _load().orc_set_heat_output(self._h, self._Q.ctypes.data, int(nq))
        if rc:
            raise ValueError("orc_set_heat_output failed: %d" % rc)
        return self._Q

    def propagate(self, A1, A2=None):
        ny, nx = self.grid["ny"], self.grid["nx"]
        a1 = np.ascontiguousarray(A1, dtype=np.complex128).reshape(-1, ny, nx)
        batch = a1.shape[0]
        a2 = None if A2 is None else np.ascontiguousarray(A2, dtype=np.complex128).reshape(batch, ny, nx)
        o1 = np.empty_like(a1)
        o2 = np.empty_like(a1)
        rc = _load().orc_propagate(self._h, a1.ctypes.data, None if a2 is None else a2.ctypes.data,
                                   o1.ctypes.data, o2.ctypes.data, batch)
        if rc:
            raise ValueError("orc_propagate failed: %d" % rc)
        return o1, o2

    def power(self, member: int, z: float):
        p1, p2 = C.c_double(), C.c_double()
        rc = _load().orc_power(self._h, member, float(z), C.byref(p1), C.byref(p2))
        if rc:
            raise ValueError("orc_power failed: %d" % rc)
        return p1.value, p2.value

    def power_history(self, member: int = 0) -> np.ndarray:
        out = np.empty((self.grid["nz"] + 1, 2), dtype=np.float64)
        rc = _load().orc_power_history(self._h, member, out.ctypes.data)
        if rc:
            raise ValueError("orc_power_history failed: %d" % rc)
        return out

    def close(self):
        if getattr(self, "_h", None):
            _load().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
