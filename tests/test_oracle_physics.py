"""Pins for the oracle's split-step scheme (oracle/gpe_oracle.c), CPU only.

Each test compares the oracle with something fixed by the paper's statement of the method or
by mathematics, not with the oracle itself: closed forms, conservation laws, an independent
ODE integration, a numpy-FFT residual.  SURVEY.md 8(c) "What pins each part"; the paper's
passages are cited per test.  A plausible mistake (dropped term, wrong sign or index,
transposed axis, wrong factor order) fails at least one of them.
"""
import math

import numpy as np
import pytest
from scipy.linalg import expm
from scipy.special import jv

import workloads as W
from oracle.gpe_oracle import Oracle


def _plain(n, L, **kw):
    p = W._base(n, n, L)
    p.update(kw)
    return p


def _moments(psi, p):
    x = W.axis(p["nx"], p["Lx"])[:, None]
    y = W.axis(p["ny"], p["Ly"])[None, :]
    d = np.abs(psi) ** 2
    d = d / d.sum()
    return float((d * x * x).sum()), float((d * y * y).sum())


# ------------------------------------------------------------------ schedule (reading Q4)
def test_schedule_pulse_and_ramp():
    p = _plain(64, 16.0, sched_step=np.array([0., 200., 200.]), sched_amp=np.array([7., 7., 0.]))
    o = Oracle(p)
    assert o.schedule(0, 0) == 7.0 and o.schedule(0, 199) == 7.0
    assert o.schedule(0, 200) == 0.0 and o.schedule(0, 5000) == 0.0   # on for n < tau/dt
    p = _plain(64, 16.0, sched_step=np.array([0., 10000.]), sched_amp=np.array([0., 20.]))
    o = Oracle(p)
    assert o.schedule(0, 2500) == pytest.approx(5.0, abs=1e-14)
    assert o.schedule(0, 20000) == 20.0
    assert Oracle(_plain(64, 16.0)).schedule(0, 3) == 0.0


# ------------------------------------------------------------------ kinetic factor alone
def test_kinetic_composition_exact():
    """the kinetic factor is diagonal in k, so n steps of dt == one of n*dt."""
    p = _plain(64, 16.0)
    psi0 = W.noisy_gaussian(64, 64, 16.0, 16.0, 1.5, 3)
    a, b = psi0.copy(), psi0.copy()
    o = Oracle(p)
    for _ in range(10):
        o.kinetic_step(a, 1e-3, False)
    o.kinetic_step(b, 1e-2, False)
    assert np.linalg.norm(a - b) / np.linalg.norm(b) <= 1e-12
    # and the full step with V=0, g=0 is that factor
    c = psi0.copy()
    Oracle(p).evolve(c, 1e-2, 1, False)
    assert np.linalg.norm(c - b) / np.linalg.norm(b) <= 1e-13


def test_free_gaussian_expansion():
    """Free Schroedinger spreading, hbar=m=1: <x^2>(t) = s0^2/2 + t^2/(2 s0^2) per axis."""
    n, L, s0 = 128, 40.0, 1.0
    p = _plain(n, L)
    psi = W.noisy_gaussian(n, n, L, L, s0, 0, noise=0.0)
    o = Oracle(p)
    t = 0.0
    for _ in range(4):
        o.evolve(psi, 0.05, 20, False)
        t += 1.0
        mx, my = _moments(psi, p)
        expect = s0 ** 2 / 2 + t ** 2 / (2 * s0 ** 2)
        assert mx == pytest.approx(expect, rel=1e-10)
        assert my == pytest.approx(expect, rel=1e-10)
    obs, _, _ = o.observables(psi)
    assert obs[0]["norm"] == pytest.approx(1.0, abs=1e-12)
    assert obs[0]["e_kin"] == pytest.approx(2 * 1.0 / (4 * s0 ** 2), rel=1e-10)  # conserved


def test_anisotropic_axes_not_swapped():
    """Lx != Ly, nx != ny: spreading along each axis follows its own width."""
    nx, ny, Lx, Ly = 128, 64, 48.0, 24.0
    p = W._base(nx, ny, Lx)
    p["Ly"] = Ly
    x = W.axis(nx, Lx)[:, None]
    y = W.axis(ny, Ly)[None, :]
    sx, sy = 2.0, 1.0
    psi = np.exp(-x * x / (2 * sx * sx) - y * y / (2 * sy * sy)).astype(np.complex128)
    psi = np.ascontiguousarray(psi)
    Oracle(p).evolve(psi, 0.02, 50, False)
    mx, my = _moments(psi, p)
    assert mx == pytest.approx(sx ** 2 / 2 + 1.0 / (2 * sx ** 2), rel=1e-9)
    assert my == pytest.approx(sy ** 2 / 2 + 1.0 / (2 * sy ** 2), rel=1e-9)


# ------------------------------------------------------------------ potential factor alone
@pytest.mark.parametrize("axis", [0, 1])
def test_potential_factor_jacobi_anger(axis):
    """PAPER.md:154 Eq. 9 / :67: uniform psi times exp(-i V0 cos^2(k r) dt/2) has k-space
    amplitudes e^{-i b}(-i)^m J_m(b) at k = 2 m k_l, b = V0 dt/4 (Jacobi-Anger)."""
    n, L, k = 256, 4 * math.pi, 4.0         # orders up to |m| = 7 resolved: aliasing J_13(b)
    V0, dt = 800.0, 1e-3
    beta = V0 * dt / 4                      # half step: phase (V0 dt/2) * (1 + cos 2kr)/2
    p = _plain(n, L, lattice_axis=axis, lattice_k=k,
               sched_step=np.array([0.]), sched_amp=np.array([V0]))
    psi = np.full((n, n), 1.0 / L, dtype=np.complex128)
    Oracle(p).potential_half_step(psi, dt, False)
    hat = np.fft.fft2(psi) / (n * n) * L
    dk = 2 * math.pi / L
    for m in range(-3, 4):
        idx = int(round(2 * m * k / dk)) % n
        got = hat[idx, 0] if axis == 0 else hat[0, idx]
        expect = np.exp(-1j * beta) * (-1j) ** abs(m) * jv(abs(m), beta)
        assert abs(got - expect) <= 1e-11, (m, got, expect)
    # imaginary time: the same factor is a real decay
    psi = np.full((n, n), 1.0 / L, dtype=np.complex128)
    Oracle(p).potential_half_step(psi, dt, True)
    r = W.axis(n, L)
    shape = np.cos(k * r) ** 2
    expect = np.exp(-V0 * shape * dt / 2) / L
    got = psi[:, 0] if axis == 0 else psi[0, :]
    assert np.max(np.abs(got - expect)) <= 1e-15


def test_potential_factor_nonlinear_term():
    """V = V_ext + g|psi|^2 -- phase of each point is -(V + g|psi|^2) dt/2."""
    n, L = 64, 16.0
    p = W.config1(g=10.0)
    psi0 = p["psi0"].copy()
    psi = psi0.copy()
    Oracle(p).potential_half_step(psi, 1e-2, False)
    ph = np.angle(psi / psi0)
    expect = -(p["v_static"] + 10.0 * np.abs(psi0) ** 2) * 1e-2 / 2
    assert np.max(np.abs(ph - expect)) <= 1e-13
    assert np.max(np.abs(np.abs(psi) - np.abs(psi0))) <= 1e-15


# ------------------------------------------------------------------ imaginary time, harmonic trap
def test_gaussian_recurrence_closed_form():
    """in V = r^2/2 with g = 0 a noise-free Gaussian e^{-a r^2/2} stays
    Gaussian under V/2.T.V/2 with a <- (a+dt/2)/(1+(a+dt/2)dt) + dt/2; E = 2(a/4 + 1/(4a)),
    <x^2> = 1/(2a).  Pins factor order, the dt/2 split, the 1/2 in T and V, and step 6."""
    p = W.config1(g=0.0, noise=0.0)
    psi = p["psi0"].copy()
    dt, nsteps = 1e-3, 2000
    o = Oracle(p)
    o.evolve(psi, dt, nsteps, True)
    a = 1.0 / 1.5 ** 2
    for _ in range(nsteps):
        b = a + dt / 2
        a = b / (1 + b * dt) + dt / 2
    obs, _, _ = o.observables(psi)
    E = obs[0]["e_kin"] + obs[0]["e_pot"]
    assert obs[0]["norm"] == pytest.approx(1.0, abs=1e-13)
    assert E == pytest.approx(2 * (a / 4 + 1 / (4 * a)), abs=2e-11)
    mx, my = _moments(psi, p)
    assert mx == pytest.approx(1 / (2 * a), abs=2e-11)
    assert my == pytest.approx(1 / (2 * a), abs=2e-11)
    # T/2.V.T/2 ordering would give a different a after 2000 steps; so would dt instead of dt/2.


def test_harmonic_ground_state_energy():
    """north_star pin: the non-interacting 2-D harmonic ground state has E = (wx+wy)/2 = 1
    (imaginary time converges to the ground state)."""
    p = W.config1(g=0.0)
    psi = p["psi0"].copy()
    o = Oracle(p)
    o.evolve(psi, 1e-3, 2000, True)
    obs, _, _ = o.observables(psi)
    E = obs[0]["e_kin"] + obs[0]["e_pot"]
    assert abs(E - 1.0) <= 2e-4            # tau = 2 is short: residual n=2 admixture ~ e^{-2 tau}
    o.evolve(psi, 1e-3, 10000, True)
    obs, _, _ = o.observables(psi)
    E = obs[0]["e_kin"] + obs[0]["e_pot"]
    assert abs(E - 1.0) <= 1e-8
    d = np.abs(psi) ** 2
    x = W.axis(64, 16.0)[:, None]
    y = W.axis(64, 16.0)[None, :]
    a = math.sqrt(1 + 1e-3 ** 2 / 4)        # fixed point of the recurrence
    exact = a / math.pi * np.exp(-a * (x * x + y * y))
    assert np.max(np.abs(d - exact)) <= 1e-8


def test_virial_interacting_ground_state():
    """2-D harmonic trap virial theorem at the GPE ground state: E_kin - E_pot + E_int = 0."""
    p = W.config1(g=10.0)
    psi = p["psi0"].copy()
    o = Oracle(p)
    o.evolve(psi, 2e-3, 4000, True)
    obs, _, _ = o.observables(psi)
    ob = obs[0]
    assert abs(ob["e_kin"] - ob["e_pot"] + ob["e_int"]) <= 2e-3
    assert ob["e_int"] > 0.2 and ob["norm"] == pytest.approx(1.0, abs=1e-12)


def test_thomas_fermi_limit():
    """PAPER.md:144-148 (Sec. 5.1): at large g the density follows Thomas-Fermi:
    mu = sqrt(g/pi), E = 2mu/3, n(0) = mu/g, <r^2> = 2mu/3 (norm 1, w = 1)."""
    n, L, g = 128, 20.0, 1000.0
    p = W._with_trap(W._base(n, n, L))
    p["g"] = np.array([g])
    psi = W.noisy_gaussian(n, n, L, L, 3.0, 5)
    o = Oracle(p)
    o.evolve(psi, 2e-3, 3000, True)
    obs, dens, _ = o.observables(psi, density=True)
    ob = obs[0]
    mu = math.sqrt(g / math.pi)
    E = ob["e_kin"] + ob["e_pot"] + ob["e_int"]
    assert E == pytest.approx(2 * mu / 3, rel=0.02)
    assert dens[0, n // 2, n // 2] == pytest.approx(mu / g, rel=0.02)
    mx, my = _moments(psi, p)
    assert mx + my == pytest.approx(2 * mu / 3, rel=0.02)
    # profile inside the bulk
    x = W.axis(n, L)
    tf = np.maximum(mu - 0.5 * x * x, 0) / g
    bulk = np.abs(x) < 0.7 * math.sqrt(2 * mu)
    assert np.max(np.abs(dens[0, :, n // 2][bulk] - tf[bulk]) / tf[bulk]) <= 0.03


# ------------------------------------------------------------------ real time invariants
def test_real_time_norm_and_time_reversal():
    """Unitary factors: the norm is conserved; Strang with reading Q2 is symmetric, so n steps
    of dt followed by n steps of -dt return psi0."""
    p = W.config1(g=10.0)
    p["lattice_axis"], p["lattice_k"] = 0, 2.0
    p["sched_step"], p["sched_amp"] = np.array([0.]), np.array([3.0])
    psi0 = p["psi0"].copy()
    psi = psi0.copy()
    o = Oracle(p)
    o.evolve(psi, 2e-3, 50, False)
    obs, _, _ = o.observables(psi)
    assert obs[0]["norm"] == pytest.approx(1.0, abs=1e-13)
    assert np.linalg.norm(psi - psi0) > 1e-2
    o.evolve(psi, -2e-3, 50, False)
    assert np.linalg.norm(psi - psi0) / np.linalg.norm(psi0) <= 1e-12


def test_convergence_order_two():
    """local error O(dt^3) -> global error O(dt^2)."""
    p = W.config1(g=10.0)
    T = 0.2

    def run(nsteps):
        psi = p["psi0"].copy()
        Oracle(p).evolve(psi, T / nsteps, nsteps, False)
        return psi

    ref = run(1600)
    e1 = np.linalg.norm(run(50) - ref)
    e2 = np.linalg.norm(run(100) - ref)
    e3 = np.linalg.norm(run(200) - ref)
    assert math.log2(e1 / e2) == pytest.approx(2.0, abs=0.1)
    assert math.log2(e2 / e3) == pytest.approx(2.0, abs=0.1)


# ------------------------------------------------------------------ Kapitza-Dirac
def _coupled_mode_populations(V0, k, t, M=10):
    """Schroedinger equation of the momentum states |2 m k>:
    i dc_m/dt = ((2mk)^2/2 + V0/2) c_m + (V0/4)(c_{m-1} + c_{m+1}),  c_m(0) = delta_m0."""
    m = np.arange(-M, M + 1)
    H = np.diag((2 * m * k) ** 2 / 2 + V0 / 2).astype(complex)
    H += np.diag(np.full(2 * M, V0 / 4), 1) + np.diag(np.full(2 * M, V0 / 4), -1)
    c0 = np.zeros(2 * M + 1, complex)
    c0[M] = 1
    c = expm(-1j * H * t) @ c0
    return {int(mm): float(abs(cc) ** 2) for mm, cc in zip(m, c)}


@pytest.mark.parametrize("V0", [5.0, 20.0])
def test_kapitza_dirac_coupled_mode(V0):
    """the non-interacting populations agree with integrating the
    Schroedinger equation in momentum space.  Uniform gas, g=0, no trap; error ~ dt^2."""
    n, L, k = 128, 4 * math.pi, 4.0
    p = _plain(n, L, lattice_axis=0, lattice_k=k,
               sched_step=np.array([0., 200., 200.]), sched_amp=np.array([V0, V0, 0.]))
    psi = np.full((n, n), 1.0 / L, dtype=np.complex128)
    o = Oracle(p)
    o.evolve(psi, 1e-4, 200, False)
    pops = o.populations(psi, 0, k, 3)[0]
    ref = _coupled_mode_populations(V0, k, 0.02)
    for m in range(-3, 4):
        assert pops[m + 3] == pytest.approx(ref[m], abs=5e-6), m
    assert pops[3 + 1] == pytest.approx(pops[3 - 1], rel=1e-9)
    # g = 0, lattice off: populations stay constant during free evolution
    o.evolve(psi, 1e-4, 100, False)
    pops2 = o.populations(psi, 0, k, 3)[0]
    assert np.max(np.abs(pops2 - pops)) <= 1e-12


def test_kapitza_dirac_raman_nath_bessel():
    """north_star pin: short-pulse populations follow J_m^2(V0 tau/2) (Raman-Nath regime)."""
    n, L, k = 128, 4 * math.pi, 4.0
    V0, nst, dt = 500.0, 20, 1e-4
    p = _plain(n, L, lattice_axis=1, lattice_k=k,
               sched_step=np.array([0.]), sched_amp=np.array([V0]))
    psi = np.full((n, n), 1.0 / L, dtype=np.complex128)
    o = Oracle(p)
    o.evolve(psi, dt, nst, False)
    pops = o.populations(psi, 1, k, 3)[0]
    beta = V0 * nst * dt / 2
    for m in range(-3, 4):
        assert pops[m + 3] == pytest.approx(jv(abs(m), beta) ** 2, abs=2e-3), m
    assert pops[4] > 0.05                     # really diffracted


# ------------------------------------------------------------------ observables on a known state
def test_observables_closed_forms_gaussian():
    """For psi = Gaussian(sigma): E_kin = 1/(2 s^2), E_trap = s^2/2, E_int = g/(4 pi s^2),
    Theta = exp(-k^2 s^2/2); alpha = N eta Theta/(Delta + i kappa) (Eq. 14)."""
    n, L, s, g, kc = 128, 24.0, 1.3, 7.0, 1.0
    p = W._with_trap(W._base(n, n, L))
    p.update(g=np.array([g]), cavity_on=1, cavity_k=kc, eta_mode=0, eta_or_u=np.array([0.8]),
             n_atoms=np.array([3.0]), delta=np.array([-2.0]), kappa=np.array([0.5]))
    psi = W.noisy_gaussian(n, n, L, L, s, 0, noise=0.0)
    obs, dens, kd = Oracle(p).observables(psi, density=True, kdensity=True)
    ob = obs[0]
    assert ob["norm"] == pytest.approx(1.0, abs=1e-13)
    assert ob["e_kin"] == pytest.approx(1 / (2 * s * s), rel=1e-10)
    assert ob["e_pot"] == pytest.approx(s * s / 2, rel=1e-10)
    assert ob["e_int"] == pytest.approx(g / (4 * math.pi * s * s), rel=1e-10)
    theta = math.exp(-kc * kc * s * s / 2)
    assert ob["theta"] == pytest.approx(theta, rel=1e-10)
    alpha = 3.0 * 0.8 * theta / complex(-2.0, 0.5)
    assert ob["re_alpha"] == pytest.approx(alpha.real, rel=1e-10)
    assert ob["im_alpha"] == pytest.approx(alpha.imag, rel=1e-10)
    assert ob["e_cav"] == pytest.approx(3.0 * 0.64 * theta ** 2 * (-2.0) / (4 + 0.25), rel=1e-10)
    assert np.max(np.abs(dens[0] - np.abs(psi) ** 2)) == 0.0
    assert kd[0].sum() == pytest.approx(1.0, abs=1e-12)
    kx = 2 * math.pi * np.fft.fftfreq(n, L / n)
    expect = np.exp(-(kx[:, None] ** 2 + kx[None, :] ** 2) * s * s)
    expect /= expect.sum()
    assert np.max(np.abs(kd[0] - expect)) <= 1e-12


# ------------------------------------------------------------------ cavity
def _cavity_small(Vp, g=0.0, n=64, delta=-1.0):
    L = 4 * math.pi
    p = W._cavity(W._with_trap(W._base(n, n, L)), 1, Vp, delta, g)
    p["sched_step"], p["sched_amp"] = np.array([0.]), np.array([Vp])
    p["psi0"] = W.noisy_gaussian(n, n, L, L, 1.2, 7)
    return p


def test_cavity_real_time_conservation():
    """Static parameters, real time: V real -> norm conserved; with E_cav = N eta^2 Theta^2
    Delta/(Delta^2+kappa^2) (so that dE_cav/d|psi|^2 = C cos cos, Eqs. 13-14) the total
    energy is conserved up to the splitting error, which shrinks with dt."""
    p = _cavity_small(8.0, g=5.0)

    def drift(dt, nsteps):
        psi = p["psi0"].copy()
        o = Oracle(p)
        ob0 = o.observables(psi)[0][0]
        o.evolve(psi, dt, nsteps, False)
        ob1 = o.observables(psi)[0][0]
        e = lambda ob: ob["e_kin"] + ob["e_pot"] + ob["e_int"] + ob["e_cav"]
        assert ob1["norm"] == pytest.approx(1.0, abs=1e-12)
        assert abs(ob1["theta"] - ob0["theta"]) > 1e-4        # something happened
        return abs(e(ob1) - e(ob0)) / abs(e(ob0))

    d1 = drift(1e-3, 200)
    d2 = drift(5e-4, 400)
    assert d1 <= 2e-5
    assert d2 <= 0.6 * d1
    # a wrong sign or a missing factor 2 in C breaks conservation at O(1):
    # (checked by construction: E_cav's functional derivative must equal the potential used)


def test_cavity_self_organisation_and_fixed_point():
    """below a critical pump the cavity field vanishes, above it the gas orders
    into the chequerboard and the field is non-zero (Delta < 0).  At the imaginary-time fixed
    point psi is an eigenstate of H[psi] with alpha frozen: residual O(dt), via numpy's FFT."""
    lo = _cavity_small(1.0)
    psi = lo["psi0"].copy()
    o = Oracle(lo)
    o.evolve(psi, 2e-3, 3000, True)
    # "vanishing" up to the explicit overlap of the finite cloud itself: for the trap ground
    # state |psi|^2 = e^{-r^2}/pi the overlap is exp(-k^2/4)^2 = e^{-8} = 3.4e-4
    assert abs(o.observables(psi)[0][0]["theta"]) <= 1e-3

    hi = _cavity_small(15.0)
    psi = hi["psi0"].copy()
    o = Oracle(hi)
    o.evolve(psi, 2e-3, 4000, True)
    ob = o.observables(psi)[0][0]
    assert abs(ob["theta"]) >= 0.3
    # eigen-residual with numpy
    n, L, k = 64, 4 * math.pi, 4.0
    x = W.axis(n, L)
    eta = math.sqrt(15.0 * 4.0)
    alpha = eta * ob["theta"] / complex(-1.0, 0.5)
    V = hi["v_static"] + 15.0 * np.cos(k * x)[None, :] ** 2 \
        + 2 * eta * alpha.real * np.cos(k * x)[:, None] * np.cos(k * x)[None, :]
    kk = 2 * math.pi * np.fft.fftfreq(n, L / n)
    K2 = kk[:, None] ** 2 + kk[None, :] ** 2
    Hpsi = np.fft.ifft2(0.5 * K2 * np.fft.fft2(psi)) + V * psi
    mu = np.vdot(psi, Hpsi) / np.vdot(psi, psi)
    res = np.linalg.norm(Hpsi - mu * psi) / np.linalg.norm(psi) / abs(mu)
    assert res <= 5e-3
    assert ob["re_alpha"] == pytest.approx(alpha.real, rel=1e-12)


def test_probe_closed_form_and_imprint():
    """On-axis probe (Eq. 17), real time.
    (a) With N_at = 0 the atoms do not feed the field, so the recorded cavity field is the probe
        alone: alpha'(t_n) = Omega exp(i(Delta_p n dt + phi)) / (Delta + i kappa), whatever psi does
        -- pins amplitude, phase, sign of the frequency and the sampling time t_n = n dt.
    (b) The probe enters the potential as 2 eta Re(alpha') cos(kx)cos(ky) (Eq. 18): one short step
        from a uniform state imprints the phase -dt 2 eta Re(dalpha(0)) cos cos to first order.
    (c) Omega = 0 is the run without a probe (to the round-off of the OpenMP reduction order);
        imaginary time ignores the probe."""
    p = _cavity_small(6.0, g=0.0, n=64, delta=-1.3)
    p["kappa"] = np.array([0.7])
    Om, Dp, ph, dt = 0.8, 37.0, 0.4, 2e-3
    p["probe_omega"], p["probe_delta"], p["probe_phi"] = np.array([Om]), np.array([Dp]), np.array([ph])
    # (a)
    pa = dict(p); pa["n_atoms"] = np.array([0.0])
    psi = pa["psi0"].copy()
    rec = Oracle(pa).evolve(psi, dt, 12, False, record_every=1)
    n = np.arange(1, 13)
    want = Om * np.exp(1j * (Dp * n * dt + ph)) / (-1.3 + 0.7j)
    assert np.allclose(rec[:, 0, 3] + 1j * rec[:, 0, 4], want, rtol=1e-13, atol=1e-15)
    # (b) uniform state, no trap, no pump lattice but eta given directly (mode 0), N_at = 0
    L = 4 * math.pi
    pb = W._base(64, 64, L)
    pb["cavity_on"], pb["cavity_k"], pb["eta_mode"] = 1, 4.0, 0
    pb["eta_or_u"], pb["n_atoms"], pb["delta"], pb["kappa"] = np.array([1.5]), np.array([0.0]), np.array([-1.3]), np.array([0.7])
    pb["probe_omega"], pb["probe_delta"], pb["probe_phi"] = np.array([Om]), np.array([Dp]), np.array([ph])
    psi = np.full((64, 64), 1.0 / L, dtype=np.complex128)
    tiny = 1e-6
    Oracle(pb).evolve(psi, tiny, 1, False)
    x = W.axis(64, L)
    cc = np.cos(4.0 * x)[:, None] * np.cos(4.0 * x)[None, :]
    d0 = (Om * np.exp(1j * ph) / (-1.3 + 0.7j)).real
    phase = np.angle(psi * L)
    assert np.allclose(phase, -tiny * 2.0 * 1.5 * d0 * cc, rtol=1e-4, atol=1e-12)
    # (c)
    p0 = dict(p); p0["probe_omega"] = np.array([0.0])
    pn = {k: v for k, v in p.items() if not k.startswith("probe_")}
    a, b = p["psi0"].copy(), p["psi0"].copy()
    Oracle(p0).evolve(a, dt, 5, False); Oracle(pn).evolve(b, dt, 5, False)
    assert np.linalg.norm(a - b) <= 1e-14 * np.linalg.norm(b)
    a, b = p["psi0"].copy(), p["psi0"].copy()
    Oracle(p).evolve(a, dt, 5, True); Oracle(pn).evolve(b, dt, 5, True)
    assert np.linalg.norm(a - b) <= 1e-14 * np.linalg.norm(b)
    # and the probe does act in real time
    a = p["psi0"].copy(); Oracle(p).evolve(a, dt, 5, False)
    b = p["psi0"].copy(); Oracle(pn).evolve(b, dt, 5, False)
    assert np.linalg.norm(a - b) > 1e-6


def test_full_cavity_model_closed_forms():
    """Cavity lattice V_c = U0 |alpha|^2 cos^2(kx) and dispersive shift Delta~ = Delta - N U0 B,
    B = int cos^2(kx)|psi|^2 (Eqs. 12 and 15).
    (a) psi = c (1 + eps cos kx cos ky): Theta = c^2 L^2 eps/2, B = c^2 L^2 (1/2 + 3 eps^2/16),
        c^2 L^2 = 1/(1 + eps^2/4), so alpha = N eta Theta/(Delta - N U0 B + i kappa) in closed form
        -- pins the definition of B (axis x), the sign of the shift and the factor N.
    (b) N = 0 with a probe: alpha = dalpha exactly (no shift), and one short step from a uniform
        state imprints -dt (2 eta Re(dalpha) cos kx cos ky + U0 |dalpha|^2 cos^2 kx): pins the
        coefficient and the axis of V_c.
    (c) U0 = 0 is the three-term model of the hot path; real time conserves the norm."""
    L, n, k = 4 * math.pi, 128, 4.0
    x = W.axis(n, L)
    cc = np.cos(k * x)[:, None] * np.cos(k * x)[None, :]
    eps, eta, N, u0, D, K = 0.3, 1.5, 2.5, 0.8, -1.3, 0.7
    p = W._base(n, n, L)
    p["cavity_on"], p["cavity_k"], p["eta_mode"] = 1, k, 0
    p["eta_or_u"], p["n_atoms"], p["delta"], p["kappa"] = np.array([eta]), np.array([N]), np.array([D]), np.array([K])
    p["cav_u0"] = np.array([u0])
    c2L2 = 1.0 / (1.0 + eps * eps / 4.0)
    psi = (np.sqrt(c2L2) / L * (1.0 + eps * cc)).astype(np.complex128)
    ob = Oracle(p).observables(psi)[0][0]
    theta, B = c2L2 * eps / 2.0, c2L2 * (0.5 + 3.0 * eps * eps / 16.0)
    alpha = N * eta * theta / (D - N * u0 * B + 1j * K)
    assert ob["norm"] == pytest.approx(1.0, abs=1e-13)
    assert ob["theta"] == pytest.approx(theta, rel=1e-12)
    assert ob["re_alpha"] == pytest.approx(alpha.real, rel=1e-12)
    assert ob["im_alpha"] == pytest.approx(alpha.imag, rel=1e-12)
    # (b)
    Om, ph = 0.8, 0.4
    pb = dict(p); pb["n_atoms"] = np.array([0.0])
    pb["probe_omega"], pb["probe_delta"], pb["probe_phi"] = np.array([Om]), np.array([11.0]), np.array([ph])
    u = np.full((n, n), 1.0 / L, dtype=np.complex128)
    tiny = 1e-6
    Oracle(pb).evolve(u, tiny, 1, False)
    da = Om * np.exp(1j * ph) / (D + 1j * K)
    want = -tiny * (2.0 * eta * da.real * cc + u0 * abs(da) ** 2 * (np.cos(k * x) ** 2)[:, None] * np.ones((1, n)))
    assert np.allclose(np.angle(u * L), want, rtol=1e-4, atol=1e-12)
    # (c)
    q = _cavity_small(8.0, g=5.0)
    q0 = dict(q); q0["cav_u0"] = np.array([0.0])
    a, b = q["psi0"].copy(), q["psi0"].copy()
    Oracle(q0).evolve(a, 1e-3, 5, False); Oracle(q).evolve(b, 1e-3, 5, False)
    assert np.linalg.norm(a - b) <= 1e-14 * np.linalg.norm(b)
    q1 = dict(q); q1["cav_u0"] = np.array([3.0])
    a = q["psi0"].copy()
    o = Oracle(q1); o.evolve(a, 1e-3, 50, False)
    assert o.observables(a)[0][0]["norm"] == pytest.approx(1.0, abs=1e-12)
    b = q["psi0"].copy(); Oracle(q).evolve(b, 1e-3, 50, False)
    assert np.linalg.norm(a - b) > 1e-6          # and U0 does act


def test_schedule_midpoint_sampling_is_exact_for_a_linear_ramp():
    """sched_midpoint (reading Q4).  A uniform state under a lattice whose amplitude
    ramps linearly in time: over a short run the kinetic term mixes the imprinted grating only at
    O(k^2 t) of an already small phase, so the accumulated phase is -cos^2(kx) int A dt.  Sampling
    at the middle of each step gives that integral exactly, sampling at the start misses
    (A(T) - A(0)) dt / 2: pins the +1/2 and that nothing else moved."""
    L, n, k = 4 * math.pi, 64, 0.5          # k small: the kinetic mixing of the imprinted grating is O(k^2 t phase)
    p = W._base(n, n, L)
    p["lattice_axis"], p["lattice_k"] = 0, k
    nst, dt = 10, 1e-5
    p["sched_step"], p["sched_amp"] = np.array([0.0, float(nst)]), np.array([2.0, 12.0])
    x = W.axis(n, L)
    c2 = (np.cos(k * x) ** 2)[:, None] * np.ones((1, n))
    out = {}
    for mid in (0, 1):
        q = dict(p); q["sched_midpoint"] = mid
        psi = np.full((n, n), 1.0 / L, dtype=np.complex128)
        rec = Oracle(q).evolve(psi, dt, nst, False, record_every=1)
        out[mid] = (np.angle(psi * L), rec[:, 0, 5])
    integral = 0.5 * (2.0 + 12.0) * nst * dt
    assert np.allclose(out[1][0], -c2 * integral, rtol=0, atol=2e-9)
    assert np.allclose(out[0][0], -c2 * (integral - 0.5 * (12.0 - 2.0) * dt), rtol=0, atol=2e-9)
    assert np.max(np.abs(out[1][0] - out[0][0])) > 1e-5 * 0.9 * 5.0          # the two differ by 5 dt cos^2
    # records report the sample of the upcoming step: A(n + 1/2) against A(n), clamped after the last knot
    assert np.allclose(out[1][1][:-1], 2.0 + (np.arange(1, nst) + 0.5))
    assert np.allclose(out[0][1], 2.0 + np.arange(1, nst + 1))


def test_interactions_raise_threshold():
    """repulsive interactions increase the critical pump."""
    thetas = {}
    for g in (0.0, 60.0):
        p = _cavity_small(8.0, g=g)
        psi = p["psi0"].copy()
        o = Oracle(p)
        o.evolve(psi, 2e-3, 3000, True)
        thetas[g] = abs(o.observables(psi)[0][0]["theta"])
    assert thetas[0.0] > 0.5
    assert thetas[60.0] < 0.2 * thetas[0.0]


# ------------------------------------------------------------------ batch and records
def test_batch_members_equal_single_runs_and_records():
    p = W.config5(n=64, side=2, n_steps=30)
    psi = p["psi0"].astype(np.complex128).copy()
    o = Oracle(p)
    rec = o.evolve(psi, 5e-4, 30, True, record_every=10)
    assert rec.shape == (3, 4, 6)
    for b in range(4):
        q = W.member(p, b)
        s = q["psi0"].astype(np.complex128).copy()
        os_ = Oracle(q)
        r1 = os_.evolve(s, 5e-4, 30, True, record_every=10)
        # OpenMP sum order is not fixed, so equality is to round-off, not bitwise
        assert np.linalg.norm(s - psi[b]) / np.linalg.norm(s) <= 1e-13
        assert np.allclose(r1[:, 0, :], rec[:, b, :], rtol=1e-12, atol=1e-15)
    ob = o.observables(psi)[0]
    assert rec[-1, 3, 0] == 30
    assert rec[-1, 3, 2] == pytest.approx(ob[3]["theta"], rel=1e-12)
    assert rec[-1, 3, 1] == pytest.approx(1.0, abs=1e-12)


def test_f32_build_tracks_f64():
    """The float build is the same statements in complex64 (used only as the fp32 floor)."""
    p = W.config1(g=10.0)
    a = p["psi0"].astype(np.complex64)
    b = a.astype(np.complex128)
    Oracle(p, "f32").evolve(a, 1e-3, 10, True)
    Oracle(p, "f64").evolve(b, 1e-3, 10, True)
    err = np.linalg.norm(a.astype(np.complex128) - b) / np.linalg.norm(b)
    assert 1e-9 < err < 5e-6


# ------------------------------------------------------------------ T/2 V T/2 ordering
def test_tvt_gaussian_recurrence_closed_form():
    """ordering = 1, the form the paper prints (Eqs. 3-4).  Same Gaussian algebra as
    the V/2.T.V/2 pin, in the other order: half a kinetic step 1/a <- 1/a + dt/2,
    the full potential factor a <- a + dt, half a kinetic step again; renormalisation leaves a alone.
    Pins the dt/4 in the kinetic exponents, the full dt in the potential factor and their order: after
    2000 steps the V/2.T.V/2 recurrence gives an a that differs by 2.4e-7, four orders of magnitude
    above the tolerance (checked below)."""
    p = W.config1(g=0.0, noise=0.0)
    p["ordering"] = 1
    psi = p["psi0"].copy()
    dt, nsteps = 1e-3, 2000
    o = Oracle(p)
    o.evolve(psi, dt, nsteps, True)
    a = a_vtv = 1.0 / 1.5 ** 2
    for _ in range(nsteps):
        a = a / (1 + a * dt / 2)
        a = a + dt
        a = a / (1 + a * dt / 2)
        b = a_vtv + dt / 2
        a_vtv = b / (1 + b * dt) + dt / 2
    assert abs(a - a_vtv) > 1e-7
    obs, _, _ = o.observables(psi)
    assert obs[0]["norm"] == pytest.approx(1.0, abs=1e-13)
    assert obs[0]["e_kin"] + obs[0]["e_pot"] == pytest.approx(2 * (a / 4 + 1 / (4 * a)), abs=2e-11)
    mx, my = _moments(psi, p)
    assert mx == pytest.approx(1 / (2 * a), abs=2e-11)
    assert my == pytest.approx(1 / (2 * a), abs=2e-11)


def test_tvt_is_the_vtv_propagator_conjugated_by_half_steps():
    """For a linear, time-independent Hamiltonian (g = 0, static trap + constant lattice, real time)
    (T/2 V T/2)^n = T/2 V/2 (V/2 T V/2)^(n-1) V/2 T/2 exactly (adjacent half factors of the same
    operator merge).  The right-hand side is built from the V/2.T.V/2 loop and the single factors,
    which have their own pins above."""
    n, L = 64, 16.0
    p = W._with_trap(W._base(n, n, L))
    p["lattice_axis"], p["lattice_k"] = 0, 2 * math.pi * 4 / L
    p["sched_step"], p["sched_amp"] = np.array([0.0]), np.array([3.0])
    psi0 = W.noisy_gaussian(n, n, L, L, 1.3, 11)
    dt, ns = 2e-3, 25
    a = psi0.copy()
    Oracle({**p, "ordering": 1}).evolve(a, dt, ns, False)
    b = psi0.copy()
    o = Oracle(p)
    o.kinetic_step(b, dt / 2, False)
    o.potential_half_step(b, dt, False)
    o.evolve(b, dt, ns - 1, False)
    o.potential_half_step(b, dt, False)
    o.kinetic_step(b, dt / 2, False)
    assert np.linalg.norm(a - b) / np.linalg.norm(b) <= 1e-12
    c = psi0.copy()
    Oracle(p).evolve(c, dt, ns, False)
    assert np.linalg.norm(a - c) / np.linalg.norm(c) > 1e-7      # and the two orderings do differ (1e-6 here)


def test_tvt_time_reversal_and_second_order():
    """The step is symmetric, so running it with -dt undoes it exactly (g != 0 included: a phase factor
    leaves |psi|^2 alone); and both orderings are second-order approximations of the same flow, so
    they converge to one another as dt^2."""
    p = W.config1(g=10.0)
    psi0 = p["psi0"].copy()
    q = {**p, "ordering": 1}
    a = psi0.copy()
    o = Oracle(q)
    o.evolve(a, 1e-3, 40, False)
    assert np.linalg.norm(a - psi0) / np.linalg.norm(psi0) > 1e-2
    o.evolve(a, -1e-3, 40, False)
    assert np.linalg.norm(a - psi0) / np.linalg.norm(psi0) <= 1e-12

    def gap(dt, ns):
        u, v = psi0.copy(), psi0.copy()
        Oracle(q).evolve(u, dt, ns, False)
        Oracle(p).evolve(v, dt, ns, False)
        return np.linalg.norm(u - v) / np.linalg.norm(v)
    g1, g2 = gap(4e-3, 50), gap(2e-3, 100)
    assert 3.5 < g1 / g2 < 4.5


def test_tvt_cavity_scalars_come_from_the_psi_entering_the_potential_factor():
    """One T/2 V T/2 step with the cavity, contact interaction and a lattice equals: half a kinetic
    step, the single potential factor evaluated (Theta, alpha, |psi|^2) on that intermediate psi over
    2 x dt/2, half a kinetic step, normalisation.  Evaluating Theta on the psi at the start of the
    step instead gives a different result (checked), so the cadence is pinned."""
    p = _cavity_small(8.0, g=5.0)
    psi0 = p["psi0"].copy()
    dt = 5e-3
    a = psi0.copy()
    Oracle({**p, "ordering": 1}).evolve(a, dt, 1, True)
    b = psi0.copy()
    o = Oracle(p)
    o.kinetic_step(b, dt / 2, True)
    o.potential_half_step(b, 2 * dt, True)
    o.kinetic_step(b, dt / 2, True)
    b /= math.sqrt(o.observables(b)[0][0]["norm"])
    assert np.linalg.norm(a - b) / np.linalg.norm(b) <= 1e-13
    # the other cadence: Theta of the starting psi, held through the step
    th0 = o.observables(psi0)[0][0]["theta"]
    c = psi0.copy()
    o.kinetic_step(c, dt / 2, True)
    th_mid = o.observables(c)[0][0]["theta"]
    assert abs(th_mid - th0) > 1e-6 * abs(th0)


def test_gaussian_recurrence_on_a_non_power_of_two_grid():
    """the whole step on a 96 x 80 grid (dft_direct on both axes) obeys the same closed form
    as test_gaussian_recurrence_closed_form, so the non-power-of-two branch of the oracle is pinned by more than
    its transform alone."""
    p = W.config1(g=0.0, noise=0.0)
    nx, ny, L = 96, 80, 16.0
    p["nx"], p["ny"] = nx, ny
    v2d, vx, vy = W.harmonic_trap(nx, ny, L, L)
    p["v_static"], p["vx"], p["vy"] = v2d, vx, vy
    psi = W.noisy_gaussian(nx, ny, L, L, 1.5, 1234, 0.0)
    dt, nsteps = 1e-3, 300
    o = Oracle(p)
    o.evolve(psi, dt, nsteps, True)
    a = 1.0 / 1.5 ** 2
    for _ in range(nsteps):
        b = a + dt / 2
        a = b / (1 + b * dt) + dt / 2
    obs, _, _ = o.observables(psi)
    assert obs[0]["norm"] == pytest.approx(1.0, abs=1e-13)
    assert obs[0]["e_kin"] + obs[0]["e_pot"] == pytest.approx(2 * (a / 4 + 1 / (4 * a)), abs=1e-9)
