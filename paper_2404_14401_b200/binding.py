"""ctypes binding of include/gpe.h.  Marshalling only -- no arithmetic of the method here."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

GPE_C64, GPE_C128 = 0, 1
GPE_REAL_TIME, GPE_IMAG_TIME = 0, 1
GPE_NREC = 6
GPE_ABI_VERSION = 4   # include/gpe.h
GPE3_NREC = 3
_STATUS = {0: "GPE_OK", 1: "GPE_EINVAL", 2: "GPE_EUNSUPPORTED", 3: "GPE_ENOMEM", 4: "GPE_ECUDA",
           5: "GPE_ESTATE", 6: "GPE_ENONFINITE"}


class GpeError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__(f"{_STATUS.get(status, status)}: {text}")
        self.status = status


class gpe_potential_desc(C.Structure):
    _fields_ = [
        ("v_static", C.c_void_p), ("v_static_batched", C.c_int),
        ("vx", C.c_void_p), ("vy", C.c_void_p), ("g", C.c_void_p),
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


class gpe_obs(C.Structure):
    _fields_ = [(n, C.c_double) for n in
                ("norm", "e_kin", "e_pot", "e_int", "e_cav", "theta", "re_alpha", "im_alpha")]


def library_path() -> str:
    return os.path.join(_HERE, "libgpe.so")


def load_library() -> C.CDLL:
    """Loads libgpe.so; raises if it has not been built (no fallback of any kind)."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = library_path()
    # libgpe.so is git-ignored: a fresh checkout, or one whose csrc/ or include/gpe.h is newer than the
    # library, compiles it with nvcc first (build.build() returns at once when it is up to date).  Still
    # no fallback of any kind -- if the build fails and no library exists, the import fails.
    from . import build as _build
    if not _build.up_to_date():
        try:
            _build.build()
        except Exception as exc:  # noqa: BLE001
            if not os.path.exists(path):
                raise ImportError(f"{path} is missing and could not be built: {exc}") from exc
            raise ImportError(f"{path} is older than its sources and could not be rebuilt: {exc}") from exc
    lib = C.CDLL(path)
    vp, i, d, l = C.c_void_p, C.c_int, C.c_double, C.c_long
    lib.gpe_plan_create.restype = i
    lib.gpe_plan_create.argtypes = [C.POINTER(vp), i, i, d, d, i, i]
    lib.gpe_plan_set_stream.restype = i
    lib.gpe_plan_set_stream.argtypes = [vp, vp]
    lib.gpe_plan_destroy.restype = i
    lib.gpe_plan_destroy.argtypes = [vp]
    lib.gpe_set_potential.restype = i
    lib.gpe_set_potential.argtypes = [vp, C.POINTER(gpe_potential_desc)]
    lib.gpe_evolve.restype = i
    lib.gpe_evolve.argtypes = [vp, vp, d, l, i, l, vp]
    lib.gpe_observables.restype = i
    lib.gpe_observables.argtypes = [vp, vp, C.POINTER(gpe_obs), vp, vp]
    lib.gpe_populations.restype = i
    lib.gpe_populations.argtypes = [vp, vp, i, d, i, vp]
    lib.gpe_fft2_forward.restype = i
    lib.gpe_fft2_forward.argtypes = [vp, vp, vp]
    lib.gpe_profile_passes.restype = i
    lib.gpe_profile_passes.argtypes = [vp, vp, d, l, i, C.POINTER(C.c_double)]
    lib.gpe_measure_roofs.restype = i
    lib.gpe_measure_roofs.argtypes = [vp, C.POINTER(C.c_double)]
    lib.gpe_norm_theta_noalloc.restype = i
    lib.gpe_norm_theta_noalloc.argtypes = [vp, i, i, d, d, i, i, d, vp, vp]
    lib.gpe_noalloc_last_error.restype = C.c_char_p
    lib.gpe_noalloc_last_error.argtypes = []
    ll = C.c_longlong
    lib.gpe3_plan_create.restype = i
    lib.gpe3_plan_create.argtypes = [C.POINTER(vp), i, i, i, d, d, d, i]
    lib.gpe3_plan_set_stream.restype = i
    lib.gpe3_plan_set_stream.argtypes = [vp, vp]
    lib.gpe3_plan_destroy.restype = i
    lib.gpe3_plan_destroy.argtypes = [vp]
    lib.gpe3_set_potential.restype = i
    lib.gpe3_set_potential.argtypes = [vp, vp, vp, vp, vp, d]
    lib.gpe3_evolve.restype = i
    lib.gpe3_evolve.argtypes = [vp, vp, d, ll, i, ll, vp]
    lib.gpe3_observables.restype = i
    lib.gpe3_observables.argtypes = [vp, vp, C.POINTER(C.c_double)]
    lib.gpe3_synchronize.restype = i
    lib.gpe3_synchronize.argtypes = [vp]
    lib.gpe3_get_step.restype = i
    lib.gpe3_get_step.argtypes = [vp, C.POINTER(ll)]
    lib.gpe3_set_step.restype = i
    lib.gpe3_set_step.argtypes = [vp, ll]
    lib.gpe3_last_error.restype = C.c_char_p
    lib.gpe3_last_error.argtypes = [vp]
    lib.gpe_get_step.restype = i
    lib.gpe_get_step.argtypes = [vp, C.POINTER(l)]
    lib.gpe_set_step.restype = i
    lib.gpe_set_step.argtypes = [vp, l]
    lib.gpe_last_error.restype = C.c_char_p
    lib.gpe_last_error.argtypes = [vp]
    lib.gpe_version.restype = C.c_char_p
    lib.gpe_version.argtypes = []
    lib.gpe_abi_version.restype = i
    lib.gpe_abi_version.argtypes = []
    lib.gpe_sizeof_potential_desc.restype = C.c_size_t
    lib.gpe_sizeof_potential_desc.argtypes = []
    # layout drift between this file and the built library must fail loudly, not corrupt a descriptor
    if lib.gpe_abi_version() != GPE_ABI_VERSION or lib.gpe_sizeof_potential_desc() != C.sizeof(gpe_potential_desc):
        raise ImportError(f"{path}: ABI {lib.gpe_abi_version()} / descriptor of {lib.gpe_sizeof_potential_desc()} bytes, "
                          f"the binding expects ABI {GPE_ABI_VERSION} / {C.sizeof(gpe_potential_desc)} bytes: rebuild "
                          "with `python -m paper_2404_14401_b200.build --force`")
    _LIB = lib
    return lib


def _check(status: int, plan) -> None:
    if status != 0:
        raise GpeError(status, gpe_last_error(plan))


# ---- the C ABI, same names --------------------------------------------------------------
def gpe_version() -> str:
    return load_library().gpe_version().decode()


def gpe_last_error(plan) -> str:
    return load_library().gpe_last_error(plan).decode()


def gpe_plan_create(nx: int, ny: int, Lx: float, Ly: float, dtype: int, batch: int = 1):
    out = C.c_void_p()
    st = load_library().gpe_plan_create(C.byref(out), int(nx), int(ny), float(Lx), float(Ly),
                                        int(dtype), int(batch))
    _check(st, None)
    return out


def gpe_plan_set_stream(plan, cuda_stream: int) -> None:
    _check(load_library().gpe_plan_set_stream(plan, C.c_void_p(cuda_stream)), plan)


def gpe_plan_destroy(plan) -> None:
    load_library().gpe_plan_destroy(plan)


def gpe_set_potential(plan, desc: gpe_potential_desc) -> None:
    _check(load_library().gpe_set_potential(plan, C.byref(desc)), plan)


def gpe_evolve(plan, psi_ptr: int, dt: float, n_steps: int, mode: int, record_every: int = 0,
               records_ptr: int | None = None) -> None:
    _check(load_library().gpe_evolve(plan, C.c_void_p(psi_ptr), float(dt), int(n_steps), int(mode),
                                     int(record_every), C.c_void_p(records_ptr or 0)), plan)


def gpe_observables(plan, psi_ptr: int, batch: int, density_ptr: int | None = None,
                    kdensity_ptr: int | None = None):
    out = (gpe_obs * batch)()
    _check(load_library().gpe_observables(plan, C.c_void_p(psi_ptr), out, C.c_void_p(density_ptr or 0),
                                          C.c_void_p(kdensity_ptr or 0)), plan)
    return [{n: getattr(o, n) for n, _ in gpe_obs._fields_} for o in out]


def gpe_populations(plan, psi_ptr: int, batch: int, axis: int, k_l: float, m_max: int) -> np.ndarray:
    out = np.zeros((batch, 2 * m_max + 1), dtype=np.float64)
    _check(load_library().gpe_populations(plan, C.c_void_p(psi_ptr), int(axis), float(k_l), int(m_max),
                                          C.c_void_p(out.ctypes.data)), plan)
    return out


def gpe_fft2_forward(plan, src_ptr: int, dst_ptr: int) -> None:
    _check(load_library().gpe_fft2_forward(plan, C.c_void_p(src_ptr), C.c_void_p(dst_ptr)), plan)


def gpe_profile_passes(plan, psi_ptr: int, dt: float, n_steps: int, mode: int):
    out = (C.c_double * 3)()
    _check(load_library().gpe_profile_passes(plan, C.c_void_p(psi_ptr), float(dt), int(n_steps), int(mode), out),
           plan)
    return [out[0], out[1], out[2]]


def gpe_measure_roofs(cuda_stream: int = 0) -> dict:
    out = (C.c_double * 5)()
    _check(load_library().gpe_measure_roofs(C.c_void_p(cuda_stream), out), None)
    return {"l2_rw_32MiB_gbs": out[0], "l2_rw_64MiB_gbs": out[1], "hbm_rw_1GiB_gbs": out[2],
            "fp32_fma_tflops": out[3], "fp64_fma_tflops": out[4]}


def gpe_norm_theta_noalloc(psi_ptr: int, nx: int, ny: int, Lx: float, Ly: float, dtype: int, batch: int,
                           cavity_k: float, out_ptr: int, cuda_stream: int = 0) -> None:
    """out[b] = {norm, theta} of member b, written on the device; allocates nothing (include/gpe.h)."""
    lib = load_library()
    st = lib.gpe_norm_theta_noalloc(C.c_void_p(psi_ptr), int(nx), int(ny), float(Lx), float(Ly), int(dtype), int(batch),
                                    float(cavity_k), C.c_void_p(out_ptr), C.c_void_p(cuda_stream))
    if st != 0:
        raise GpeError(st, lib.gpe_noalloc_last_error().decode())


def gpe_get_step(plan) -> int:
    v = C.c_long()
    _check(load_library().gpe_get_step(plan, C.byref(v)), plan)
    return v.value


def gpe_set_step(plan, step: int) -> None:
    _check(load_library().gpe_set_step(plan, int(step)), plan)


# ---- convenience wrapper (still marshalling only) ----------------------------------------
def _h(a, n=None):
    if a is None:
        return None
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    if n is not None and a.size != n:
        raise ValueError(f"expected {n} values, got {a.size}")
    return a


class Plan:
    """gpe_plan with torch tensors for device memory.  `p` is a workload dict (workloads/)."""

    def __init__(self, nx, ny, Lx, Ly, dtype="c64", batch=1, stream=None):
        import torch
        self.torch = torch
        self.nx, self.ny, self.batch = int(nx), int(ny), int(batch)
        self.dtype = dtype
        self.cdtype = torch.complex64 if dtype == "c64" else torch.complex128
        self.rdtype = torch.float32 if dtype == "c64" else torch.float64
        self.plan = gpe_plan_create(nx, ny, Lx, Ly, GPE_C64 if dtype == "c64" else GPE_C128, batch)
        if stream is not None:
            gpe_plan_set_stream(self.plan, stream)
        self._keep = []

    def close(self):
        if self.plan is not None:
            gpe_plan_destroy(self.plan)
            self.plan = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_potential(self, p: dict, use_separable: bool = True) -> None:
        torch, B = self.torch, self.batch
        d = gpe_potential_desc()
        keep = []

        def hp(a, n=None):
            a = _h(a, n)
            if a is None:
                return None
            keep.append(a)
            return a.ctypes.data

        vs = p.get("v_static")
        if use_separable and p.get("vx") is not None and p.get("vy") is not None:
            d.vx, d.vy = hp(p["vx"], self.nx), hp(p["vy"], self.ny)
            d.v_static = None
        elif vs is not None:
            t = torch.as_tensor(np.asarray(vs), dtype=self.rdtype).contiguous().cuda()
            keep.append(t)
            d.v_static = t.data_ptr()
            d.v_static_batched = 1 if t.numel() == B * self.nx * self.ny and B > 1 else 0
        d.g = hp(np.broadcast_to(np.asarray(p.get("g", 0.0), dtype=np.float64), (B,)), B)
        d.lattice_axis = int(p.get("lattice_axis", -1))
        d.lattice_k = float(p.get("lattice_k", 0.0))
        ss = p.get("sched_step")
        if ss is not None and len(ss) > 0:
            d.sched_len = len(ss)
            d.sched_step = hp(ss)
            sa = _h(p["sched_amp"])
            d.sched_batched = 1 if (sa.size == B * len(ss) and B > 1) else 0
            d.sched_amp = hp(sa)
        d.cavity_on = int(p.get("cavity_on", 0))
        d.cavity_k = float(p.get("cavity_k", 0.0))
        d.eta_mode = int(p.get("eta_mode", 0))
        for name, default in (("eta_or_u", 0.0), ("n_atoms", 1.0), ("delta", -1.0), ("kappa", 1.0)):
            a = np.broadcast_to(np.asarray(p.get(name, default), dtype=np.float64), (B,))
            setattr(d, name, hp(a, B))
        if p.get("probe_omega") is not None:
            for name in ("probe_omega", "probe_delta", "probe_phi"):
                a = np.broadcast_to(np.asarray(p.get(name, 0.0), dtype=np.float64), (B,))
                setattr(d, name, hp(a, B))
        if p.get("cav_u0") is not None:
            d.cav_u0 = hp(np.broadcast_to(np.asarray(p["cav_u0"], dtype=np.float64), (B,)), B)
        d.sched_midpoint = int(p.get("sched_midpoint", 0))
        d.ordering = int(p.get("ordering", 0))
        gpe_set_potential(self.plan, d)
        torch.cuda.current_stream().synchronize()
        self._keep = keep

    def evolve(self, psi, dt, n_steps, mode, record_every=0):
        """psi: CUDA tensor [batch,]nx,ny of the plan's complex dtype, evolved in place.
        Returns the records tensor [n_rec, batch, 6] (device, float64) or None."""
        torch = self.torch
        assert psi.is_cuda and psi.dtype == self.cdtype and psi.is_contiguous()
        assert psi.numel() == self.batch * self.nx * self.ny
        m = GPE_IMAG_TIME if mode in ("imag", GPE_IMAG_TIME) else GPE_REAL_TIME
        rec = None
        if record_every > 0:
            s0 = gpe_get_step(self.plan)
            nrec = (s0 + n_steps) // record_every - s0 // record_every
            rec = torch.zeros((max(nrec, 1), self.batch, GPE_NREC), dtype=torch.float64, device=psi.device)
        gpe_evolve(self.plan, psi.data_ptr(), dt, n_steps, m, record_every,
                   rec.data_ptr() if rec is not None else None)
        return rec

    def observables(self, psi, density=False, kdensity=False):
        torch = self.torch
        assert psi.is_cuda and psi.dtype == self.cdtype and psi.is_contiguous()
        shape = (self.batch, self.nx, self.ny)
        dn = torch.empty(shape, dtype=self.rdtype, device=psi.device) if density else None
        kd = torch.empty(shape, dtype=self.rdtype, device=psi.device) if kdensity else None
        obs = gpe_observables(self.plan, psi.data_ptr(), self.batch,
                              dn.data_ptr() if dn is not None else None,
                              kd.data_ptr() if kd is not None else None)
        return obs, dn, kd

    def populations(self, psi, axis, k_l, m_max):
        return gpe_populations(self.plan, psi.data_ptr(), self.batch, axis, k_l, m_max)

    @property
    def step(self):
        return gpe_get_step(self.plan)

    @step.setter
    def step(self, v):
        gpe_set_step(self.plan, v)


# ---- three dimensions (include/gpe.h, gpe3_*) -----------------------------------------------
OBS3_NAMES = ("norm", "e_kin", "e_pot", "e_int", "x2", "y2", "z2", "reserved")


def _check3(status: int, plan) -> None:
    if status != 0:
        raise GpeError(status, load_library().gpe3_last_error(plan).decode())


def gpe3_plan_create(nx: int, ny: int, nz: int, Lx: float, Ly: float, Lz: float, dtype: int):
    out = C.c_void_p()
    _check3(load_library().gpe3_plan_create(C.byref(out), int(nx), int(ny), int(nz), float(Lx), float(Ly), float(Lz),
                                            int(dtype)), None)
    return out


def gpe3_plan_set_stream(plan, cuda_stream: int) -> None:
    _check3(load_library().gpe3_plan_set_stream(plan, C.c_void_p(cuda_stream)), plan)


def gpe3_plan_destroy(plan) -> None:
    _check3(load_library().gpe3_plan_destroy(plan), None)


def gpe3_set_potential(plan, v_static_ptr, vx, vy, vz, g: float) -> None:
    """v_static_ptr: device pointer or None; vx, vy, vz: host float64 arrays or None."""
    keep = [None if a is None else np.ascontiguousarray(np.asarray(a, dtype=np.float64)) for a in (vx, vy, vz)]
    ptrs = [None if a is None else a.ctypes.data for a in keep]
    _check3(load_library().gpe3_set_potential(plan, v_static_ptr, ptrs[0], ptrs[1], ptrs[2], float(g)), plan)


def gpe3_evolve(plan, psi_ptr: int, dt: float, n_steps: int, mode: int, record_every: int = 0,
                records_ptr: int | None = None) -> None:
    _check3(load_library().gpe3_evolve(plan, psi_ptr, float(dt), int(n_steps), int(mode), int(record_every), records_ptr), plan)


def gpe3_observables(plan, psi_ptr: int) -> dict:
    out = (C.c_double * 8)()
    _check3(load_library().gpe3_observables(plan, psi_ptr, out), plan)
    return dict(zip(OBS3_NAMES, [float(v) for v in out]))


def gpe3_synchronize(plan) -> None:
    _check3(load_library().gpe3_synchronize(plan), plan)


def gpe3_get_step(plan) -> int:
    v = C.c_longlong()
    _check3(load_library().gpe3_get_step(plan, C.byref(v)), plan)
    return int(v.value)


def gpe3_set_step(plan, step: int) -> None:
    _check3(load_library().gpe3_set_step(plan, int(step)), plan)


class Plan3:
    """gpe3_plan with torch tensors for device memory.  `p` is a workload dict of workloads.config3d()."""

    def __init__(self, nx, ny, nz, Lx, Ly, Lz, dtype="c64", stream=None):
        import torch
        self.torch = torch
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.dtype = dtype
        self.cdtype = torch.complex64 if dtype == "c64" else torch.complex128
        self.rdtype = torch.float32 if dtype == "c64" else torch.float64
        self.plan = gpe3_plan_create(nx, ny, nz, Lx, Ly, Lz, GPE_C64 if dtype == "c64" else GPE_C128)
        if stream is not None:
            gpe3_plan_set_stream(self.plan, stream)

    def close(self):
        if self.plan is not None:
            gpe3_plan_destroy(self.plan)
            self.plan = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_potential(self, p: dict) -> None:
        vs = p.get("v_static")
        t = None
        if vs is not None:
            t = self.torch.as_tensor(np.asarray(vs), dtype=self.rdtype).contiguous().cuda()
            assert t.numel() == self.nx * self.ny * self.nz
        gpe3_set_potential(self.plan, None if t is None else t.data_ptr(), p.get("vx"), p.get("vy"), p.get("vz"),
                           float(p.get("g", 0.0)))

    def evolve(self, psi, dt, n_steps, mode, record_every=0):
        """psi: CUDA tensor [nz, nx, ny] of the plan's complex dtype, evolved in place.
        Returns the records tensor [n_rec, 3] (device, float64) or None."""
        torch = self.torch
        assert psi.is_cuda and psi.dtype == self.cdtype and psi.is_contiguous()
        assert psi.numel() == self.nx * self.ny * self.nz
        m = GPE_IMAG_TIME if mode in ("imag", GPE_IMAG_TIME) else GPE_REAL_TIME
        rec = None
        if record_every > 0:
            s0 = gpe3_get_step(self.plan)
            nrec = (s0 + n_steps) // record_every - s0 // record_every
            rec = torch.zeros((max(nrec, 1), GPE3_NREC), dtype=torch.float64, device=psi.device)
        gpe3_evolve(self.plan, psi.data_ptr(), dt, n_steps, m, record_every, rec.data_ptr() if rec is not None else None)
        return rec

    def observables(self, psi) -> dict:
        assert psi.is_cuda and psi.dtype == self.cdtype and psi.is_contiguous()
        return gpe3_observables(self.plan, psi.data_ptr())

    def synchronize(self) -> None:
        gpe3_synchronize(self.plan)

    @property
    def step(self):
        return gpe3_get_step(self.plan)

    @step.setter
    def step(self, v):
        gpe3_set_step(self.plan, v)
