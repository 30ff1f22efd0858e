"""ctypes front end of the CPU oracle (oracle/gpe_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It never imports the CUDA
package and the CUDA package never imports it.

The arithmetic is all in the C file (which cites PAPER.md line by line); this module only
marshals numpy arrays.  `Oracle(params)` mirrors the shape of the product boundary
(set potential -> evolve -> observables) so a test can drive both sides identically.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gpe_oracle.c")
_LOCK = threading.Lock()
_LIBS: dict[str, C.CDLL] = {}

NREC = 6   # {step, norm, theta, re_alpha, im_alpha, A}
NOBS = 8   # {norm, e_kin, e_pot, e_int, e_cav, theta, re_alpha, im_alpha}
OBS_NAMES = ("norm", "e_kin", "e_pot", "e_int", "e_cav", "theta", "re_alpha", "im_alpha")


def lib_path(real: str) -> str:
    return os.path.join(_HERE, f"libgpe_oracle_{real}.so")


def build(force: bool = False) -> None:
    """Compile the oracle with gcc (double build = the oracle; float build = fp32-floor probe)."""
    for real, define in (("f64", []), ("f32", ["-DREAL=float"])):
        out = lib_path(real)
        if (not force and os.path.exists(out)
                and os.path.getmtime(out) >= os.path.getmtime(_SRC)):
            continue
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-Wall", *define,
               "-o", out + ".tmp", _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(out + ".tmp", out)


class _Params(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("batch", C.c_int),
        ("Lx", C.c_double), ("Ly", C.c_double),
        ("v_static", C.c_void_p), ("v_static_batched", C.c_int),
        ("g", C.c_void_p),
        ("lattice_axis", C.c_int), ("lattice_k", C.c_double),
        ("sched_len", C.c_int), ("sched_step", C.c_void_p), ("sched_amp", C.c_void_p),
        ("sched_batched", C.c_int),
        ("cavity_on", C.c_int), ("cavity_k", C.c_double), ("eta_mode", C.c_int),
        ("eta_or_u", C.c_void_p), ("n_atoms", C.c_void_p), ("delta", C.c_void_p),
        ("kappa", C.c_void_p),
        ("probe_omega", C.c_void_p), ("probe_delta", C.c_void_p), ("probe_phi", C.c_void_p),
        ("cav_u0", C.c_void_p),
        ("sched_midpoint", C.c_int),
        ("ordering", C.c_int),
    ]


def _load(real: str) -> C.CDLL:
    with _LOCK:
        if real not in _LIBS:
            build()
            lib = C.CDLL(lib_path(real))
            lib.oracle_evolve.restype = C.c_int
            lib.oracle_evolve.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_double, C.c_long,
                                          C.c_int, C.c_long, C.c_long, C.c_void_p]
            lib.oracle_observables.restype = C.c_int
            lib.oracle_observables.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_long,
                                               C.c_void_p, C.c_void_p, C.c_void_p]
            lib.oracle_populations.restype = C.c_int
            lib.oracle_populations.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_int,
                                               C.c_double, C.c_int, C.c_void_p]
            lib.oracle_fft2.restype = None
            lib.oracle_fft2.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int]
            lib.oracle_fft1.restype = None
            lib.oracle_fft1.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
            lib.oracle_schedule.restype = C.c_double
            lib.oracle_schedule.argtypes = [C.POINTER(_Params), C.c_int, C.c_double]
            lib.oracle_real_bytes.restype = C.c_int
            lib.oracle_potential_half_step.restype = C.c_int
            lib.oracle_potential_half_step.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_double,
                                                       C.c_int, C.c_long]
            lib.oracle_kinetic_step.restype = C.c_int
            lib.oracle_kinetic_step.argtypes = [C.POINTER(_Params), C.c_void_p, C.c_double, C.c_int]
            _LIBS[real] = lib
        return _LIBS[real]


def _f64(a, n=None):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    if n is not None and a.size != n:
        raise ValueError(f"expected {n} values, got {a.size}")
    return a


class Oracle:
    """One oracle instance = one (grid, potential) set-up, like a gpe_plan + gpe_set_potential.

    `p` is a workload dict as produced by workloads.py (keys mirror gpe_potential_desc):
      nx, ny, Lx, Ly, batch, g[batch], v_static (None | [nx,ny] | [batch,nx,ny]),
      lattice_axis, lattice_k, sched_step[len], sched_amp ([len] | [batch,len]),
      cavity_on, cavity_k, eta_mode, eta_or_u[batch], n_atoms[batch], delta[batch], kappa[batch],
      probe_omega[batch], probe_delta[batch], probe_phi[batch] (optional: on-axis probe, real time)
    precision: "f64" (the oracle) or "f32" (fp32-floor probe of the same statements).
    """

    def __init__(self, p: dict, precision: str = "f64"):
        assert precision in ("f64", "f32")
        self.lib = _load(precision)
        self.cdtype = np.complex128 if precision == "f64" else np.complex64
        assert self.lib.oracle_real_bytes() == (8 if precision == "f64" else 4)
        self.nx, self.ny, self.batch = int(p["nx"]), int(p["ny"]), int(p.get("batch", 1))
        B = self.batch
        self._keep = []
        P = _Params()
        P.nx, P.ny, P.batch = self.nx, self.ny, B
        P.Lx, P.Ly = float(p["Lx"]), float(p["Ly"])

        def ptr(a):
            self._keep.append(a)
            return a.ctypes.data

        vs = p.get("v_static")
        if vs is None:
            P.v_static, P.v_static_batched = None, 0
        else:
            vs = _f64(vs)
            if vs.size == self.nx * self.ny:
                P.v_static_batched = 0
            elif vs.size == B * self.nx * self.ny:
                P.v_static_batched = 1
            else:
                raise ValueError("v_static has the wrong size")
            P.v_static = ptr(vs)
        P.g = ptr(_f64(np.broadcast_to(np.asarray(p.get("g", 0.0), dtype=np.float64), (B,)), B))
        P.lattice_axis = int(p.get("lattice_axis", -1))
        P.lattice_k = float(p.get("lattice_k", 0.0))
        ss = p.get("sched_step")
        if ss is None or len(ss) == 0:
            P.sched_len, P.sched_step, P.sched_amp, P.sched_batched = 0, None, None, 0
        else:
            ss = _f64(ss)
            sa = _f64(p["sched_amp"])
            P.sched_len = ss.size
            P.sched_step = ptr(ss)
            if sa.size == ss.size:
                P.sched_batched = 0
            elif sa.size == B * ss.size:
                P.sched_batched = 1
            else:
                raise ValueError("sched_amp has the wrong size")
            P.sched_amp = ptr(sa)
        P.cavity_on = int(p.get("cavity_on", 0))
        P.cavity_k = float(p.get("cavity_k", 0.0))
        P.eta_mode = int(p.get("eta_mode", 0))
        for name, default in (("eta_or_u", 0.0), ("n_atoms", 1.0), ("delta", -1.0), ("kappa", 1.0)):
            a = _f64(np.broadcast_to(np.asarray(p.get(name, default), dtype=np.float64), (B,)), B)
            setattr(P, name, ptr(a))
        if p.get("probe_omega") is not None:   # on-axis probe, PAPER.md:216-221 (Eq. 17)
            for name, default in (("probe_omega", 0.0), ("probe_delta", 0.0), ("probe_phi", 0.0)):
                a = _f64(np.broadcast_to(np.asarray(p.get(name, default), dtype=np.float64), (B,)), B)
                setattr(P, name, ptr(a))
        if p.get("cav_u0") is not None:   # full cavity model, PAPER.md:177,188 (Eqs. 12, 15)
            P.cav_u0 = ptr(_f64(np.broadcast_to(np.asarray(p["cav_u0"], dtype=np.float64), (B,)), B))
        P.sched_midpoint = int(p.get("sched_midpoint", 0))
        P.ordering = int(p.get("ordering", 0))   # 0: V/2 T V/2; 1: T/2 V T/2
        self.P = P
        self.step = 0

    # ---- the three calls that mirror the boundary
    def evolve(self, psi: np.ndarray, dt: float, n_steps: int, imag_time: bool,
               record_every: int = 0) -> np.ndarray | None:
        """In place on `psi` ([batch,]nx,ny complex of this oracle's precision)."""
        assert psi.dtype == self.cdtype and psi.flags.c_contiguous
        assert psi.size == self.batch * self.nx * self.ny
        rec = None
        if record_every > 0:
            nrec = (self.step + n_steps) // record_every - self.step // record_every
            rec = np.zeros((nrec, self.batch, NREC), dtype=np.float64)
        self.lib.oracle_evolve(C.byref(self.P), psi.ctypes.data, float(dt), int(n_steps),
                               1 if imag_time else 0, int(self.step), int(record_every),
                               rec.ctypes.data if rec is not None else None)
        self.step += int(n_steps)
        return rec

    def observables(self, psi: np.ndarray, density: bool = False, kdensity: bool = False):
        assert psi.dtype == self.cdtype and psi.flags.c_contiguous
        out = np.zeros((self.batch, NOBS), dtype=np.float64)
        shape = (self.batch, self.nx, self.ny)
        d = np.zeros(shape, dtype=np.float64) if density else None
        k = np.zeros(shape, dtype=np.float64) if kdensity else None
        self.lib.oracle_observables(C.byref(self.P), psi.ctypes.data, int(self.step),
                                    out.ctypes.data,
                                    d.ctypes.data if d is not None else None,
                                    k.ctypes.data if k is not None else None)
        obs = [dict(zip(OBS_NAMES, row)) for row in out]
        return obs, d, k

    def populations(self, psi: np.ndarray, axis: int, k_l: float, m_max: int) -> np.ndarray:
        assert psi.dtype == self.cdtype and psi.flags.c_contiguous
        out = np.zeros((self.batch, 2 * m_max + 1), dtype=np.float64)
        self.lib.oracle_populations(C.byref(self.P), psi.ctypes.data, int(axis), float(k_l),
                                    int(m_max), out.ctypes.data)
        return out

    def potential_half_step(self, psi: np.ndarray, dt: float, imag_time: bool) -> None:
        """One factor exp(-sigma (V_n + g|psi|^2) dt/2) alone, n = the current step index."""
        assert psi.dtype == self.cdtype and psi.flags.c_contiguous
        self.lib.oracle_potential_half_step(C.byref(self.P), psi.ctypes.data, float(dt),
                                            1 if imag_time else 0, int(self.step))

    def kinetic_step(self, psi: np.ndarray, dt: float, imag_time: bool) -> None:
        """FFT2 -> exp(-sigma k^2 dt/2) -> IFFT2 alone."""
        assert psi.dtype == self.cdtype and psi.flags.c_contiguous
        self.lib.oracle_kinetic_step(C.byref(self.P), psi.ctypes.data, float(dt),
                                     1 if imag_time else 0)

    def schedule(self, b: int, n: float) -> float:
        return float(self.lib.oracle_schedule(C.byref(self.P), int(b), float(n)))


def fft2(a: np.ndarray, sign: int = -1, force_direct: bool = False) -> np.ndarray:
    """Oracle 2-D FFT of a [nx,ny] complex128 array (copy). sign=-1 forward, +1 inverse (1/P)."""
    a = np.ascontiguousarray(a, dtype=np.complex128).copy()
    _load("f64").oracle_fft2(a.ctypes.data, a.shape[0], a.shape[1], int(sign), int(force_direct))
    return a


def fft1(a: np.ndarray, sign: int = -1, force_direct: bool = False) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.complex128).copy()
    _load("f64").oracle_fft1(a.ctypes.data, a.size, int(sign), int(force_direct))
    return a
