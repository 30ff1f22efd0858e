"""ctypes front end of the 3-D CPU oracle (oracle/gpe3_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline leg may import this module.  It never imports the CUDA package and the CUDA package
never imports it.  The arithmetic is all in the C file; this module only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gpe3_oracle.c")
_LOCK = threading.Lock()
_LIBS: dict[str, C.CDLL] = {}

NREC3 = 3   # {step, norm, norm_pre}
OBS3_NAMES = ("norm", "e_kin", "e_pot", "e_int", "x2", "y2", "z2", "reserved")


def lib_path(real: str) -> str:
    return os.path.join(_HERE, f"libgpe3_oracle_{real}.so")


def build(force: bool = False) -> None:
    for real, define in (("f64", []), ("f32", ["-DREAL=float"])):
        out = lib_path(real)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(_SRC):
            continue
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-Wall", *define, "-o", out + ".tmp", _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(out + ".tmp", out)


class _Params(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
        ("Lx", C.c_double), ("Ly", C.c_double), ("Lz", C.c_double),
        ("v_static", C.c_void_p), ("vx", C.c_void_p), ("vy", C.c_void_p), ("vz", C.c_void_p),
        ("g", C.c_double),
    ]


def _load(real: str) -> C.CDLL:
    with _LOCK:
        if real not in _LIBS:
            build()
            lib = C.CDLL(lib_path(real))
            lib.oracle3_evolve.restype = C.c_int
            lib.oracle3_evolve.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_double, C.c_long, C.c_int, C.c_long,
                                           C.c_long, C.c_void_p]
            lib.oracle3_observables.restype = C.c_int
            lib.oracle3_observables.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_void_p]
            lib.oracle3_fft3.restype = None
            lib.oracle3_fft3.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int]
            lib.oracle3_real_bytes.restype = C.c_int
            lib.oracle3_potential_half_step.restype = C.c_int
            lib.oracle3_potential_half_step.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_double, C.c_int]
            lib.oracle3_kinetic_step.restype = C.c_int
            lib.oracle3_kinetic_step.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_double, C.c_int]
            _LIBS[real] = lib
        return _LIBS[real]


class Oracle3:
    """One (grid, potential) set-up.  `p` is a workload dict of workloads.config3d():
    nx, ny, nz, Lx, Ly, Lz, g, v_static (None | [nz, nx, ny]), vx [nx], vy [ny], vz [nz] (each optional).
    psi is [nz, nx, ny], y fastest."""

    def __init__(self, p: dict, precision: str = "f64"):
        assert precision in ("f64", "f32")
        self.lib = _load(precision)
        self.cdtype = np.complex128 if precision == "f64" else np.complex64
        assert self.lib.oracle3_real_bytes() == (8 if precision == "f64" else 4)
        self.nx, self.ny, self.nz = int(p["nx"]), int(p["ny"]), int(p["nz"])
        self._keep = []
        P = _Params()
        P.nx, P.ny, P.nz = self.nx, self.ny, self.nz
        P.Lx, P.Ly, P.Lz = float(p["Lx"]), float(p["Ly"]), float(p["Lz"])
        P.g = float(p.get("g", 0.0))
        for name, n in (("v_static", self.nx * self.ny * self.nz), ("vx", self.nx), ("vy", self.ny), ("vz", self.nz)):
            a = p.get(name)
            if a is None:
                setattr(P, name, None)
                continue
            a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
            if a.size != n:
                raise ValueError(f"{name} has the wrong size")
            self._keep.append(a)
            setattr(P, name, a.ctypes.data)
        self.P = P
        self.step = 0

    def _check(self, psi):
        assert psi.dtype == self.cdtype and psi.flags.c_contiguous
        assert psi.size == self.nx * self.ny * self.nz

    def evolve(self, psi: np.ndarray, dt: float, n_steps: int, imag_time: bool, record_every: int = 0):
        self._check(psi)
        rec = None
        if record_every > 0:
            nrec = (self.step + n_steps) // record_every - self.step // record_every
            rec = np.zeros((nrec, NREC3), dtype=np.float64)
        self.lib.oracle3_evolve(C.byref(self.P), psi.ctypes.data, float(dt), int(n_steps), 1 if imag_time else 0,
                                int(self.step), int(record_every), rec.ctypes.data if rec is not None else None)
        self.step += int(n_steps)
        return rec

    def observables(self, psi: np.ndarray) -> dict:
        self._check(psi)
        out = np.zeros(8, dtype=np.float64)
        self.lib.oracle3_observables(C.byref(self.P), psi.ctypes.data, out.ctypes.data)
        return dict(zip(OBS3_NAMES, out))

    def potential_half_step(self, psi: np.ndarray, dt: float, imag_time: bool) -> None:
        self._check(psi)
        self.lib.oracle3_potential_half_step(C.byref(self.P), psi.ctypes.data, float(dt), 1 if imag_time else 0)

    def kinetic_step(self, psi: np.ndarray, dt: float, imag_time: bool) -> None:
        self._check(psi)
        self.lib.oracle3_kinetic_step(C.byref(self.P), psi.ctypes.data, float(dt), 1 if imag_time else 0)


def fft3(a: np.ndarray, sign: int = -1) -> np.ndarray:
    """Oracle 3-D FFT of a [nz, nx, ny] complex128 array (copy).  sign = -1 forward, +1 inverse (1/P)."""
    a = np.ascontiguousarray(a, dtype=np.complex128).copy()
    _load("f64").oracle3_fft3(a.ctypes.data, a.shape[0], a.shape[1], a.shape[2], int(sign))
    return a
