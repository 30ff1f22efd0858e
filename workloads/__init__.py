"""Seeded synthetic inputs and the five BASELINE.json configurations.

This module holds NONE of the method's arithmetic (no FFT, no split-step, no reductions): it
only builds input arrays (initial wavefunctions, static potential arrays) and parameter
dictionaries.  It is the one module that both the oracle-side tests and the CUDA-side
tests / bench import, so that both sides see the same seeded inputs.

The paper measures on no public dataset; its workloads are parametrised physics set-ups in
physical units.  The inputs here take their shapes -- power-of-two
square grids 2^6..2^11, harmonic trap, cos^2 lattice, chequerboard cavity mode, noisy Gaussian
start -- and stand in for them (dimensionless, hbar = m = 1).  Readings Q9, Q11-Q13 of
SURVEY.md 8(c) are implemented here and listed in DESIGN.md.
"""
from __future__ import annotations

import copy
import math

import numpy as np

TWO_PI = 2.0 * math.pi


def axis(n: int, L: float) -> np.ndarray:
    """Grid coordinates x_i = -L/2 + i L/n (periodic box, end point excluded; reading Q9)."""
    return -0.5 * L + np.arange(n, dtype=np.float64) * (L / n)


def noisy_gaussian(nx: int, ny: int, Lx: float, Ly: float, sigma: float = 1.5,
                   seed: int = 1234, noise: float = 0.05) -> np.ndarray:
    """psi0 = exp(-(x^2+y^2)/(2 sigma^2)) * (1 + noise*xi), xi = (2u1-1) + i(2u2-1),
    u1 then u2 drawn as rng.random((nx,ny)) from numpy default_rng(seed) (PCG64);
    normalised to sum |psi|^2 dx dy = 1 (reading Q11).  complex128."""
    x = axis(nx, Lx)[:, None]
    y = axis(ny, Ly)[None, :]
    psi = np.exp(-(x * x + y * y) / (2.0 * sigma * sigma)).astype(np.complex128)
    if noise != 0.0:
        rng = np.random.default_rng(seed)
        u1 = rng.random((nx, ny))
        u2 = rng.random((nx, ny))
        psi = psi * (1.0 + noise * ((2.0 * u1 - 1.0) + 1j * (2.0 * u2 - 1.0)))
    dxdy = (Lx / nx) * (Ly / ny)
    psi /= math.sqrt(float(np.sum(psi.real ** 2 + psi.imag ** 2)) * dxdy)
    return np.ascontiguousarray(psi)


def harmonic_trap(nx, ny, Lx, Ly, wx2: float = 1.0, wy2: float = 1.0):
    """V = 0.5 (wx2 x^2 + wy2 y^2) as (v2d, vx, vy) with v2d = vx[:,None] + vy[None,:]."""
    x = axis(nx, Lx)
    y = axis(ny, Ly)
    vx = 0.5 * wx2 * x * x
    vy = 0.5 * wy2 * y * y
    return vx[:, None] + vy[None, :], vx, vy


def _base(nx, ny, L, batch=1):
    return dict(nx=nx, ny=ny, Lx=L, Ly=L, batch=batch, g=np.zeros(batch),
                v_static=None, vx=None, vy=None,
                lattice_axis=-1, lattice_k=0.0, sched_step=None, sched_amp=None,
                cavity_on=0, cavity_k=0.0, eta_mode=0,
                eta_or_u=np.zeros(batch), n_atoms=np.ones(batch),
                delta=-np.ones(batch), kappa=np.ones(batch))


def _with_trap(p, wx2=1.0, wy2=1.0):
    v2d, vx, vy = harmonic_trap(p["nx"], p["ny"], p["Lx"], p["Ly"], wx2, wy2)
    p["v_static"], p["vx"], p["vy"] = v2d, vx, vy
    return p


def config1(g: float = 0.0, n: int = 64, noise: float = 0.05):
    """BASELINE.json configs[0]: 64^2 complex128, box [-8,8]^2, V = 0.5(x^2+y^2), g in {0,10},
    imaginary time dt=1e-3 x 2000, psi0 = Gaussian(sigma 1.5) x (1 + 0.05 noise), seed 1234."""
    p = _with_trap(_base(n, n, 16.0))
    p["g"] = np.array([g])
    p["dtype"] = "c128"
    p["psi0"] = noisy_gaussian(n, n, 16.0, 16.0, 1.5, 1234, noise)
    p["phases"] = [dict(mode="imag", dt=1e-3, n_steps=2000, record_every=0, reset_step=True)]
    return p


def config2(V0: float = 10.0, g: float = 50.0, n: int = 256, dtype: str = "c64",
            n_ground: int = 5000, n_pulse: int = 200, n_free: int = 500):
    """BASELINE.json configs[1] (Kapitza-Dirac), readings Q12: box [-4pi,4pi]^2, trap
    0.5(0.1x^2+y^2); ground state dt=1e-3 x 5000 imaginary steps; pulse V0 cos^2(4x) for 200
    real-time steps dt=1e-4 (n < 200), then 500 steps with the lattice off (trap and g on)."""
    L = 4.0 * TWO_PI
    p = _with_trap(_base(n, n, L), wx2=0.1, wy2=1.0)
    p["g"] = np.array([g])
    p["dtype"] = dtype
    p["lattice_axis"], p["lattice_k"] = 0, 4.0
    p["sched_step"] = np.array([0.0, float(n_pulse), float(n_pulse)])
    p["sched_amp"] = np.array([V0, V0, 0.0])
    p["psi0"] = noisy_gaussian(n, n, L, L, 1.5, 1234)
    p["phases"] = [
        dict(mode="imag", dt=1e-3, n_steps=n_ground, record_every=0, reset_step=True,
             lattice_off=True),
        dict(mode="real", dt=1e-4, n_steps=n_pulse, record_every=0, reset_step=True),
        dict(mode="real", dt=1e-4, n_steps=n_free, record_every=0, reset_step=False),
    ]
    p["populations"] = dict(axis=0, k_l=4.0, m_max=3)
    return p


def _cavity(p, batch, Vp, delta, g, u=4.0, kappa=0.5, k=4.0):
    p["g"] = np.full(batch, float(g))
    p["lattice_axis"], p["lattice_k"] = 1, k
    p["cavity_on"], p["cavity_k"], p["eta_mode"] = 1, k, 1
    p["eta_or_u"] = np.full(batch, u)
    p["n_atoms"] = np.ones(batch)
    p["delta"] = np.broadcast_to(np.asarray(delta, dtype=np.float64), (batch,)).copy()
    p["kappa"] = np.full(batch, kappa)
    return p


def config3(n: int = 1024, n_steps: int = 5000, Vp: float = 15.0, delta: float = -1.0,
            g: float = 100.0, dtype: str = "c64"):
    """BASELINE.json configs[2], readings Q13: box [-4pi,4pi]^2, V_trap = 0.5(x^2+y^2),
    V_p cos^2(4y) + 2 eta Re(alpha) cos(4x)cos(4y), eta = sqrt(V_p u), u=4, N_at=1,
    Delta=-1, kappa=0.5, g=100; imaginary time dt=5e-4 x 5000; seed-7 noisy Gaussian."""
    L = 4.0 * TWO_PI
    p = _cavity(_with_trap(_base(n, n, L)), 1, Vp, delta, g)
    p["dtype"] = dtype
    p["sched_step"] = np.array([0.0])
    p["sched_amp"] = np.array([Vp])
    p["psi0"] = noisy_gaussian(n, n, L, L, 1.5, 7)
    p["phases"] = [dict(mode="imag", dt=5e-4, n_steps=n_steps, record_every=0, reset_step=True)]
    return p


def config4(n: int = 2048, n_steps: int = 10000, ramp_steps: int | None = None,
            Vmax: float = 20.0, g: float = 200.0, dtype: str = "c64", record_every: int = 100):
    """BASELINE.json configs[3], readings Q13: as config 3 with g=200, real time dt=1e-4,
    A_n = 20 n / 10000 (linear ramp), record the order parameter every 100 steps; the initial
    state is the seed-7 noisy Gaussian itself."""
    L = 4.0 * TWO_PI
    ramp_steps = n_steps if ramp_steps is None else ramp_steps
    p = _cavity(_with_trap(_base(n, n, L)), 1, 0.0, -1.0, g)
    p["dtype"] = dtype
    p["sched_step"] = np.array([0.0, float(ramp_steps)])
    p["sched_amp"] = np.array([0.0, Vmax])
    p["psi0"] = noisy_gaussian(n, n, L, L, 1.5, 7)
    p["phases"] = [dict(mode="real", dt=1e-4, n_steps=n_steps, record_every=record_every,
                        reset_step=True)]
    return p


def config5(n: int = 512, side: int = 8, n_steps: int = 3000, g: float = 100.0,
            dtype: str = "c64"):
    """BASELINE.json configs[4], readings Q13: side x side sweep, V_p = 20 a/(side-1),
    Delta = -3 + 2.8 b/(side-1), member index side*b + a; all members share the seed-7 state."""
    L = 4.0 * TWO_PI
    B = side * side
    a = np.arange(B) % side
    b = np.arange(B) // side
    Vp = 20.0 * a / (side - 1)
    delta = -3.0 + 2.8 * b / (side - 1)
    p = _cavity(_with_trap(_base(n, n, L, B)), B, Vp, delta, g)
    p["dtype"] = dtype
    p["sched_step"] = np.array([0.0])
    p["sched_amp"] = Vp.reshape(B, 1).copy()
    one = noisy_gaussian(n, n, L, L, 1.5, 7)
    p["psi0"] = np.ascontiguousarray(np.broadcast_to(one, (B, n, n)))
    p["phases"] = [dict(mode="imag", dt=5e-4, n_steps=n_steps, record_every=0, reset_step=True)]
    return p


def sweep_s(n: int, dtype: str = "c64", n_steps: int = 1000):
    """The paper's own Sec. 4.1 workload shape: non-interacting gas, fixed
    harmonic trap, imaginary time, 10^3 steps, N_x = N_y = 2^n."""
    p = _with_trap(_base(n, n, 16.0))
    p["dtype"] = dtype
    p["psi0"] = noisy_gaussian(n, n, 16.0, 16.0, 1.5, 1234)
    p["phases"] = [dict(mode="imag", dt=1e-3, n_steps=n_steps, record_every=0, reset_step=True)]
    return p


def member(p: dict, b: int) -> dict:
    """The single-grid workload equal to member b of a batched workload."""
    q = copy.deepcopy(p)
    B = p["batch"]
    q["batch"] = 1
    for k in ("g", "eta_or_u", "n_atoms", "delta", "kappa"):
        q[k] = np.asarray(p[k], dtype=np.float64).reshape(B)[b:b + 1].copy()
    if p.get("sched_amp") is not None:
        sa = np.asarray(p["sched_amp"], dtype=np.float64)
        L = len(p["sched_step"])
        if sa.size == B * L and B > 1:
            q["sched_amp"] = sa.reshape(B, L)[b].copy()
    if p.get("v_static") is not None and np.asarray(p["v_static"]).ndim == 3:
        q["v_static"] = np.asarray(p["v_static"])[b].copy()
    if p.get("psi0") is not None and np.asarray(p["psi0"]).ndim == 3:
        q["psi0"] = np.ascontiguousarray(np.asarray(p["psi0"])[b])
    return q


def shard_members(batch: int, rank: int, world: int) -> range:
    """Batch members owned by `rank` when the independent grids of a batched workload are
    partitioned over `world` processes (contiguous blocks, sizes differ by at most one).
    No data-path collective is needed: members never interact."""
    if world < 1 or not (0 <= rank < world) or batch < 0:
        raise ValueError("need world >= 1, 0 <= rank < world, batch >= 0")
    base, extra = divmod(batch, world)
    lo = rank * base + min(rank, extra)
    return range(lo, lo + base + (1 if rank < extra else 0))


def select_members(p: dict, idx) -> dict:
    """The sub-workload holding only the members `idx` of a batched workload `p` (same order)."""
    return _select(p, [int(i) for i in idx])


def shard(p: dict, rank: int, world: int) -> dict:
    """The sub-workload holding only this rank's members of a batched workload `p`."""
    return _select(p, list(shard_members(p["batch"], rank, world)))


def _select(p: dict, idx: list) -> dict:
    B = p["batch"]
    q = copy.deepcopy(p)
    q["batch"] = len(idx)
    for k in ("g", "eta_or_u", "n_atoms", "delta", "kappa"):
        q[k] = np.asarray(p[k], dtype=np.float64).reshape(B)[idx].copy()
    if p.get("sched_amp") is not None:
        sa = np.asarray(p["sched_amp"], dtype=np.float64)
        L = len(p["sched_step"])
        if sa.size == B * L and B > 1:
            q["sched_amp"] = sa.reshape(B, L)[idx].copy()
    if p.get("v_static") is not None and np.asarray(p["v_static"]).ndim == 3:
        q["v_static"] = np.asarray(p["v_static"])[idx].copy()
    if p.get("psi0") is not None and np.asarray(p["psi0"]).ndim == 3:
        q["psi0"] = np.ascontiguousarray(np.asarray(p["psi0"])[idx])
    return q


# ---------------------------------------------------------------- three dimensions
def noisy_gaussian3(nx: int, ny: int, nz: int, Lx: float, Ly: float, Lz: float, sigma=(1.5, 1.5, 1.5),
                    seed: int = 1234, noise: float = 0.05) -> np.ndarray:
    """psi0[z, x, y] = exp(-x^2/(2 sx^2) - y^2/(2 sy^2) - z^2/(2 sz^2)) * (1 + noise*xi), xi = (2u1-1) + i(2u2-1),
    u1 then u2 drawn as rng.random((nz, nx, ny)) from numpy default_rng(seed); normalised to
    sum |psi|^2 dx dy dz = 1.  complex128, layout [nz][nx][ny] (y fastest)."""
    x = axis(nx, Lx)[None, :, None]
    y = axis(ny, Ly)[None, None, :]
    z = axis(nz, Lz)[:, None, None]
    sx, sy, sz = sigma
    psi = np.exp(-x * x / (2.0 * sx * sx) - y * y / (2.0 * sy * sy) - z * z / (2.0 * sz * sz)).astype(np.complex128)
    if noise != 0.0:
        rng = np.random.default_rng(seed)
        u1 = rng.random((nz, nx, ny))
        u2 = rng.random((nz, nx, ny))
        psi = psi * (1.0 + noise * ((2.0 * u1 - 1.0) + 1j * (2.0 * u2 - 1.0)))
    dV = (Lx / nx) * (Ly / ny) * (Lz / nz)
    psi /= math.sqrt(float(np.sum(np.abs(psi) ** 2)) * dV)
    return np.ascontiguousarray(psi)


def config3d(nx: int = 128, ny: int | None = None, nz: int | None = None, L: float = 16.0, g: float = 50.0,
             w2=(1.0, 1.44, 0.64), dtype: str = "c64", dimple: float = 2.0, separable: bool = True,
             mode: str = "imag", dt: float = 1e-3, n_steps: int = 100, seed: int = 11):
    """The 3-D stand-in workload (the paper has none: three dimensions is the first item of its outlook,
    PAPER.md:231): an anisotropic harmonic trap w2 = (wx^2, wy^2, wz^2) given as the separable arrays vx, vy, vz,
    plus a non-separable Gaussian dimple -dimple * exp(-(x^2+y^2+z^2)/2) as the 3-D array v_static (None when
    dimple = 0), contact interaction g, the seeded noisy Gaussian as the initial state.  With separable=False the
    whole potential goes into v_static."""
    ny = nx if ny is None else ny
    nz = nx if nz is None else nz
    x, y, z = axis(nx, L), axis(ny, L), axis(nz, L)
    vx, vy, vz = 0.5 * w2[0] * x * x, 0.5 * w2[1] * y * y, 0.5 * w2[2] * z * z
    p = dict(nx=nx, ny=ny, nz=nz, Lx=L, Ly=L, Lz=L, g=float(g), dtype=dtype, vx=vx, vy=vy, vz=vz, v_static=None)
    if dimple != 0.0:
        r2 = x[None, :, None] ** 2 + y[None, None, :] ** 2 + z[:, None, None] ** 2
        p["v_static"] = np.ascontiguousarray(-dimple * np.exp(-0.5 * r2))
    if not separable:
        full = vz[:, None, None] + vx[None, :, None] + vy[None, None, :]
        p["v_static"] = np.ascontiguousarray(full + (p["v_static"] if p["v_static"] is not None else 0.0))
        p["vx"] = p["vy"] = p["vz"] = None
    p["psi0"] = noisy_gaussian3(nx, ny, nz, L, L, L, (1.5, 1.3, 1.7), seed)
    p["phases"] = [dict(mode=mode, dt=dt, n_steps=n_steps, record_every=0)]
    return p
