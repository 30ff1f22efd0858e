"""Pins for the 3-D oracle (oracle/gpe3_oracle.c), CPU only.

SURVEY.md 8(f) f4 (second half) / PAPER.md:231: the split-step of PAPER.md:60-76 on a three-dimensional grid.
Each test compares the oracle with something fixed by mathematics or by an independent implementation
(numpy.fft, the plain DFT sum, closed forms, the 2-D oracle with its own pins), never with itself; together they
catch a dropped term, a wrong sign, a wrong factor order and any mix-up of the three axes (every grid below has
three different sizes, box lengths and trap frequencies).
"""
import math

import numpy as np
import pytest

import workloads as W
from oracle.gpe3_oracle import Oracle3, fft3
from oracle.gpe_oracle import Oracle


def _grid(nx, ny, nz, Lx, Ly, Lz, **kw):
    p = dict(nx=nx, ny=ny, nz=nz, Lx=Lx, Ly=Ly, Lz=Lz, g=0.0, v_static=None, vx=None, vy=None, vz=None)
    p.update(kw)
    return p


def _gauss(p, a):
    """normalised exp(-(ax x^2 + ay y^2 + az z^2)/2) on the grid of p, [nz, nx, ny]"""
    x = W.axis(p["nx"], p["Lx"])[None, :, None]
    y = W.axis(p["ny"], p["Ly"])[None, None, :]
    z = W.axis(p["nz"], p["Lz"])[:, None, None]
    psi = np.exp(-0.5 * (a[0] * x * x + a[1] * y * y + a[2] * z * z)).astype(np.complex128)
    dV = (p["Lx"] / p["nx"]) * (p["Ly"] / p["ny"]) * (p["Lz"] / p["nz"])
    return np.ascontiguousarray(psi / math.sqrt(float(np.sum(np.abs(psi) ** 2)) * dV))


def _rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


# ------------------------------------------------------------------ the transform
def test_fft3_is_the_dft_sum():
    """the definition, written out: X[r,p,q] = sum_{l,i,j} x[l,i,j] e^{-2 pi i (r l/nz + p i/nx + q j/ny)}"""
    rng = np.random.default_rng(5)
    nz, nx, ny = 4, 6, 8
    a = rng.standard_normal((nz, nx, ny)) + 1j * rng.standard_normal((nz, nx, ny))
    Fz = np.exp(-2j * np.pi * np.outer(np.arange(nz), np.arange(nz)) / nz)
    Fx = np.exp(-2j * np.pi * np.outer(np.arange(nx), np.arange(nx)) / nx)
    Fy = np.exp(-2j * np.pi * np.outer(np.arange(ny), np.arange(ny)) / ny)
    want = np.einsum("rl,pi,qj,lij->rpq", Fz, Fx, Fy, a)
    assert np.abs(fft3(a) - want).max() <= 1e-12
    assert np.abs(fft3(want, +1) - a).max() <= 1e-13     # the inverse carries 1/(nx ny nz)


@pytest.mark.parametrize("shape", [(16, 32, 64), (64, 16, 32), (12, 20, 48)])
def test_fft3_matches_numpy(shape):
    rng = np.random.default_rng(sum(shape))
    a = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    assert _rel(fft3(a), np.fft.fftn(a)) <= 1e-13
    assert _rel(fft3(a, +1), np.fft.ifftn(a)) <= 1e-13


def test_plane_wave_lands_on_its_own_bin():
    """axis order and sign of the kernel: e^{+i(kx x + ky y + kz z)} with mode numbers (3, -5, 2) -> one bin"""
    p = _grid(16, 32, 8, 5.0, 7.0, 3.0)
    x = W.axis(16, 5.0)[None, :, None]; y = W.axis(32, 7.0)[None, None, :]; z = W.axis(8, 3.0)[:, None, None]
    a = np.exp(1j * (2 * np.pi * 3 / 5.0 * x + 2 * np.pi * (-5) / 7.0 * y + 2 * np.pi * 2 / 3.0 * z))
    h = np.abs(fft3(np.ascontiguousarray(a)))
    r, pp, q = np.unravel_index(np.argmax(h), h.shape)
    assert (r, pp, q) == (2, 3, 32 - 5)
    assert h[r, pp, q] == pytest.approx(16 * 32 * 8, rel=1e-12)
    # and the kinetic factor multiplies that wave by e^{-i |k|^2 dt/2}
    k2 = (2 * np.pi * 3 / 5.0) ** 2 + (2 * np.pi * 5 / 7.0) ** 2 + (2 * np.pi * 2 / 3.0) ** 2
    b = np.ascontiguousarray(a).copy()
    Oracle3(p).kinetic_step(b, 1e-2, False)
    assert np.abs(b - a * np.exp(-1j * k2 * 1e-2 / 2)).max() <= 1e-12
    c = np.ascontiguousarray(a).copy()
    Oracle3(p).kinetic_step(c, 1e-2, True)
    assert np.abs(c - a * np.exp(-k2 * 1e-2 / 2)).max() <= 1e-12


# ------------------------------------------------------------------ closed forms
def test_gaussian_recurrence_anisotropic_trap():
    """SURVEY.md appendix, per axis with V = w^2 x^2 / 2: a half potential step takes a -> a + w^2 dt/2, a kinetic
    step a -> a / (1 + a dt); the renormalisation does not change a.  The whole wavefunction is compared."""
    w2 = (1.0, 2.25, 0.49)
    p = _grid(32, 64, 48, 14.0, 12.0, 18.0)
    x, y, z = W.axis(32, 14.0), W.axis(64, 12.0), W.axis(48, 18.0)
    p.update(vx=0.5 * w2[0] * x * x, vy=0.5 * w2[1] * y * y, vz=0.5 * w2[2] * z * z)
    a = [0.8, 1.3, 0.6]
    psi = _gauss(p, a)
    o = Oracle3(p)
    dt = 0.02
    for n in range(25):
        o.evolve(psi, dt, 1, True)
        for d in range(3):
            b = a[d] + w2[d] * dt / 2
            b = b / (1 + b * dt)
            a[d] = b + w2[d] * dt / 2
    want = _gauss(p, a)
    assert _rel(psi, want) <= 1e-9
    ob = o.observables(psi)
    assert ob["x2"] == pytest.approx(1 / (2 * a[0]), rel=1e-9)
    assert ob["y2"] == pytest.approx(1 / (2 * a[1]), rel=1e-9)
    assert ob["z2"] == pytest.approx(1 / (2 * a[2]), rel=1e-9)
    # energies of a Gaussian: per axis a/4 (kinetic) and w^2/(4a) (potential)
    assert ob["e_kin"] == pytest.approx(sum(a) / 4, rel=1e-9)
    assert ob["e_pot"] == pytest.approx(sum(w2[d] / (4 * a[d]) for d in range(3)), rel=1e-9)
    assert ob["e_int"] == 0.0


def test_ground_state_energy_limit():
    """imaginary time converges to E = (wx + wy + wz)/2 up to the O(dt^2) of the splitting"""
    w = (1.0, 1.5, 0.7)
    p = _grid(32, 32, 32, 14.0, 12.0, 16.0)
    x, y, z = W.axis(32, 14.0), W.axis(32, 12.0), W.axis(32, 16.0)
    p.update(vx=0.5 * w[0] ** 2 * x * x, vy=0.5 * w[1] ** 2 * y * y, vz=0.5 * w[2] ** 2 * z * z)
    psi = _gauss(p, [0.6, 0.6, 0.6])
    o = Oracle3(p)
    rec = o.evolve(psi, 0.025, 300, True, record_every=300)
    ob = o.observables(psi)
    E = ob["e_kin"] + ob["e_pot"]
    assert E == pytest.approx(sum(w) / 2, abs=2e-4)
    # norm_pre of the last step: e^{-2 mu dt} up to O(dt^3)  ->  mu = E for g = 0
    assert -math.log(rec[-1, 2]) / (2 * 0.025) == pytest.approx(sum(w) / 2, abs=2e-4)
    assert rec[-1, 1] == pytest.approx(1.0, abs=1e-13)


def test_free_expansion():
    """<x^2>(t) = s0^2/2 + t^2/(2 s0^2) per axis, exact for the spectral kinetic factor"""
    p = _grid(64, 48, 96, 40.0, 36.0, 44.0)
    s0 = (1.0, 1.4, 0.8)
    psi = _gauss(p, [1 / s ** 2 for s in s0])
    o = Oracle3(p)
    o.evolve(psi, 0.05, 40, False)
    t = 2.0
    ob = o.observables(psi)
    for name, s in zip(("x2", "y2", "z2"), s0):
        assert ob[name] == pytest.approx(s * s / 2 + t * t / (2 * s * s), rel=1e-8)
    assert ob["norm"] == pytest.approx(1.0, abs=1e-12)


# ------------------------------------------------------------------ against the 2-D oracle (independent code, own pins)
@pytest.mark.parametrize("imag", [False, True])
def test_single_slab_is_the_2d_method(imag):
    """nz = 1, Lz = 1: k_z = 0 and dz = 1, so every statement of the 3-D step is the 2-D one"""
    nx, ny, L = 32, 64, 12.0
    rng = np.random.default_rng(9)
    V = rng.standard_normal((nx, ny)) * 0.5 + W.harmonic_trap(nx, ny, L, L, 1.0, 2.0)[0]
    psi0 = W.noisy_gaussian(nx, ny, L, L, 1.2, 21)
    p3 = _grid(nx, ny, 1, L, L, 1.0, g=35.0, v_static=V.reshape(1, nx, ny))
    p2 = W._base(nx, ny, L)
    p2.update(Ly=L, v_static=V, g=np.array([35.0]))
    a = np.ascontiguousarray(psi0.reshape(1, nx, ny)).copy()
    b = psi0.copy()
    Oracle3(p3).evolve(a, 2e-3, 12, imag)
    Oracle(p2).evolve(b, 2e-3, 12, imag)
    assert _rel(a[0], b) <= 1e-12


def test_separable_problem_factorises():
    """g = 0 and V = vx + vy + vz: the propagator is a product, psi(x, y, z) = f(x, y) h(z); f comes from the 2-D
    oracle, h from the 2-D oracle on an nz x 2 grid that is constant along its second axis (Ly = 1).  Exercises the z axis against independent code."""
    nx, ny, nz = 16, 32, 64
    Lx, Ly, Lz = 10.0, 12.0, 14.0
    x, y, z = W.axis(nx, Lx), W.axis(ny, Ly), W.axis(nz, Lz)
    vx, vy, vz = 0.5 * x * x, 0.8 * np.cos(1.3 * y) + 0.6 * y * y, 0.4 * z * z + 0.3 * np.sin(2 * np.pi * z / Lz)
    rng = np.random.default_rng(2)
    f0 = np.exp(-0.4 * x[:, None] ** 2 - 0.5 * y[None, :] ** 2) * (1 + 0.1 * rng.standard_normal((nx, ny)))
    h0 = np.exp(-0.3 * z * z) * (1 + 0.1 * rng.standard_normal(nz))
    for imag in (False, True):
        p3 = _grid(nx, ny, nz, Lx, Ly, Lz, vx=vx, vy=vy, vz=vz)
        psi = np.ascontiguousarray((h0[:, None, None] * f0[None, :, :]).astype(np.complex128))
        Oracle3(p3).evolve(psi, 5e-3, 8, imag)
        pf = W._base(nx, ny, Lx); pf.update(Ly=Ly, v_static=vx[:, None] + vy[None, :])
        ph = W._base(nz, 2, Lz); ph.update(Ly=1.0, v_static=np.repeat(vz[:, None], 2, axis=1))   # constant along y: k_y = 0 only
        f = np.ascontiguousarray(f0.astype(np.complex128)); h = np.ascontiguousarray(np.repeat(h0[:, None], 2, axis=1).astype(np.complex128))
        Oracle(pf).evolve(f, 5e-3, 8, imag)
        Oracle(ph).evolve(h, 5e-3, 8, imag)
        want = h[:, 0][:, None, None] * f[None, :, :]
        if not imag:
            assert _rel(psi, want) <= 1e-12
        else:   # each renormalises its own factor to 1
            dV = (Lx / nx) * (Ly / ny) * (Lz / nz)
            assert float(np.sum(np.abs(psi) ** 2)) * dV == pytest.approx(1.0, abs=1e-12)
            assert _rel(psi, want) <= 1e-12


# ------------------------------------------------------------------ invariants of the scheme
def test_norm_conservation_and_time_reversal():
    p = W.config3d(16, 32, 8, g=40.0)
    o = Oracle3(p)
    psi = p["psi0"].copy()
    rec = o.evolve(psi, 1e-3, 20, False, record_every=5)
    assert np.abs(rec[:, 1] - 1.0).max() <= 1e-12 and np.abs(rec[:, 1] - rec[:, 2]).max() <= 1e-14
    assert list(rec[:, 0]) == [5.0, 10.0, 15.0, 20.0]
    o.evolve(psi, -1e-3, 20, False)       # V/2 T V/2 is symmetric: it is its own inverse under dt -> -dt
    assert _rel(psi, p["psi0"]) <= 1e-11


def test_energy_conservation_real_time():
    p = W.config3d(16, 16, 32, g=30.0)
    o = Oracle3(p)
    psi = p["psi0"].copy()
    o.evolve(psi, 2e-3, 50, True)
    e0 = o.observables(psi)
    o.evolve(psi, 1e-3, 200, False)
    e1 = o.observables(psi)
    E0 = e0["e_kin"] + e0["e_pot"] + e0["e_int"]
    E1 = e1["e_kin"] + e1["e_pot"] + e1["e_int"]
    assert abs(E1 - E0) <= 1e-5 * abs(E0)


def test_second_order_in_dt():
    p = W.config3d(16, 16, 16, g=40.0)
    ref = p["psi0"].copy()
    Oracle3(p).evolve(ref, 0.1 / 256, 256, False)
    errs = []
    for n in (4, 8, 16):
        a = p["psi0"].copy()
        Oracle3(p).evolve(a, 0.1 / n, n, False)
        errs.append(_rel(a, ref))
    assert 3.5 <= errs[0] / errs[1] <= 4.5 and 3.5 <= errs[1] / errs[2] <= 4.5


def test_axis_permutation_covariance():
    """relabelling the axes of the input relabels the output: catches Lx/Ly/Lz, nx/ny/nz and vx/vy/vz mix-ups"""
    p = W.config3d(16, 32, 8, g=25.0, w2=(1.0, 2.0, 0.5))
    p.update(Lx=10.0, Ly=13.0, Lz=9.0)
    a = p["psi0"].copy()
    Oracle3(p).evolve(a, 2e-3, 6, False)
    # new z = old x, new x = old y, new y = old z:  arrays [z, x, y] -> [x, y, z]
    q = dict(nx=p["ny"], ny=p["nz"], nz=p["nx"], Lx=p["Ly"], Ly=p["Lz"], Lz=p["Lx"], g=p["g"],
             vx=p["vy"], vy=p["vz"], vz=p["vx"], v_static=np.ascontiguousarray(np.transpose(p["v_static"], (1, 2, 0))))
    b = np.ascontiguousarray(np.transpose(p["psi0"], (1, 2, 0)))
    Oracle3(q).evolve(b, 2e-3, 6, False)
    assert _rel(np.transpose(b, (2, 0, 1)), a) <= 1e-12


def test_fp32_build_is_the_same_statements():
    p = W.config3d(16, 16, 16, g=20.0)
    a = p["psi0"].copy()
    b = p["psi0"].astype(np.complex64)
    Oracle3(p).evolve(a, 1e-3, 10, True)
    Oracle3(p, "f32").evolve(b, 1e-3, 10, True)
    assert _rel(b.astype(np.complex128), a) <= 2e-6
