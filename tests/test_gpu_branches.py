"""GPU parity cases for the kernel branches and boundary paths that the workload-shaped tests of
tests/test_gpu_parity.py never reach ("what's weak" 2): the large-angle tiers of the
potential phase factor, per-member static arrays, the 2-D transform on its own, batched multi-knot
schedules, T/2 V T/2 with the full cavity model and a probe, and the error / asynchrony contract of
include/gpe.h.  Same oracle, same tolerances as tests/test_gpu_parity.py.
"""
import ctypes as C
import math
import time

import numpy as np
import pytest

import workloads as W
from oracle import gpe_oracle
from oracle.gpe_oracle import Oracle
from tests.test_gpu_parity import PER_STEP, _general_workload, _gpu_plan, _oracle_input, _rel, _to_dev, _torch

pytestmark = pytest.mark.gpu


def _lattice_workload(nx, ny, V0, axis=1, g=30.0):
    """Deep lattice across the cloud: the phase w = (V + g|psi|^2) dt/2 is large where psi is large."""
    L = 4 * math.pi
    p = W._base(nx, ny, L)
    v2d, vx, vy = W.harmonic_trap(nx, ny, L, L, 1.0, 0.7)
    p["v_static"], p["vx"], p["vy"] = v2d, vx, vy
    p["g"] = np.array([g])
    p["lattice_axis"], p["lattice_k"] = axis, 4.0
    p["sched_step"], p["sched_amp"] = np.array([0.0]), np.array([V0])
    p["cavity_on"], p["cavity_k"], p["eta_mode"] = 1, 4.0, 0
    p["eta_or_u"], p["delta"], p["kappa"] = np.array([2.0]), np.array([-1.5]), np.array([0.5])
    p["psi0"] = W.noisy_gaussian(nx, ny, L, L, 1.2, 11)
    return p


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("no_pair", [False, True])
@pytest.mark.parametrize("V0,dt,axis", [(800.0, 1e-2, 1), (3000.0, 1e-2, 0), (90.0, 1e-2, 1)])
def test_large_phase_real_time(monkeypatch, V0, dt, axis, no_pair, dtype):
    """|w| = V0 dt/2 = 4, 15 and 0.45 (merged multiply: 8, 30, 0.9): the library-range-reduction tier and
    the degree-9 tier of the phase factor (gpe_pair.cuh potential_pair16, gpe_kernels.cuh
    potential_step16; Eq. 3 has no small-angle restriction), on both kernel families; an
    odd step count per call ends in the k_pending_halfstep epilogue with the same angle."""
    for k in ("GPE_NO_PAIR", "GPE_NO_MERGE"):
        monkeypatch.delenv(k, raising=False)
    if no_pair:
        monkeypatch.setenv("GPE_NO_PAIR", "1")
    p = _lattice_workload(256, 128, V0, axis)
    plan = _gpu_plan(p, dtype)
    psi, ref = _to_dev(p["psi0"], dtype), _oracle_input(p["psi0"], dtype)
    o = Oracle(p)
    done = 0
    for n in (1, 3):
        plan.evolve(psi, dt, n, "real")
        o.evolve(ref, dt, n, False)
        done += n
        e = _rel(psi.cpu().numpy(), ref)
        assert e <= done * PER_STEP[dtype], f"V0 {V0} after {done} steps: {e:.3e}"
    plan.close()


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("no_merge", [False, True])
def test_large_phase_unmerged_and_2d_array(monkeypatch, no_merge, dtype):
    """The same with the static potential as a 2-D array holding a deep lattice (|w| up to 6 from the
    array alone), separate and merged half-steps."""
    for k in ("GPE_NO_PAIR", "GPE_NO_MERGE"):
        monkeypatch.delenv(k, raising=False)
    if no_merge:
        monkeypatch.setenv("GPE_NO_MERGE", "1")
    p = _lattice_workload(128, 256, 40.0)
    y = W.axis(256, p["Ly"])
    p["v_static"] = p["v_static"] + 1200.0 * np.sin(3.0 * y)[None, :] ** 2
    plan = _gpu_plan(p, dtype, use_separable=False)
    psi, ref = _to_dev(p["psi0"], dtype), _oracle_input(p["psi0"], dtype)
    o = Oracle(p)
    plan.evolve(psi, 1e-2, 3, "real")
    o.evolve(ref, 1e-2, 3, False)
    e = _rel(psi.cpu().numpy(), ref)
    assert e <= 3 * PER_STEP[dtype], f"{e:.3e}"
    plan.close()


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("no_pair", [False, True])
def test_large_exponent_imag_time(monkeypatch, no_pair, dtype):
    """Imaginary time with |w| = V0 dtau/2 up to 10: the ex2.approx form of the real factor
    (gpe_pair.cuh GPE_EXPF) and expf / exp of the other kernel family."""
    monkeypatch.delenv("GPE_NO_PAIR", raising=False)
    if no_pair:
        monkeypatch.setenv("GPE_NO_PAIR", "1")
    p = _lattice_workload(128, 128, 4000.0)
    plan = _gpu_plan(p, dtype)
    psi, ref = _to_dev(p["psi0"], dtype), _oracle_input(p["psi0"], dtype)
    o = Oracle(p)
    for done in (1, 3):
        plan.evolve(psi, 5e-3, 1 if done == 1 else 2, "imag")
        o.evolve(ref, 5e-3, 1 if done == 1 else 2, True)
        e = _rel(psi.cpu().numpy(), ref)
        assert e <= done * PER_STEP[dtype], f"after {done} steps: {e:.3e}"
    plan.close()


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("mode", ["real", "imag"])
def test_v_static_batched_distinct_members(mode, dtype):
    """v_static_batched = 1 with a different 2-D array per member (F_V2D_BATCHED), and a batched
    multi-knot schedule (sched_batched with four knots, one of them a jump)."""
    nx, ny, B = 128, 256, 3
    p = _general_workload(nx, ny, batch=B)
    vs = np.stack([W.harmonic_trap(nx, ny, p["Lx"], p["Ly"], 1.0 + 0.5 * b, 0.7 + 0.2 * b)[0] for b in range(B)])
    x = W.axis(nx, p["Lx"])
    vs[1] += 3.0 * np.cos(2.0 * x)[:, None]
    p["v_static"] = vs
    p["sched_step"] = np.array([0.0, 3.0, 3.0, 9.0])
    p["sched_amp"] = np.array([[6.0, 6.0, 9.0, 12.0], [0.0, 4.0, 1.0, 8.0], [10.0, 2.0, 2.0, 0.0]])
    plan = _gpu_plan(p, dtype, use_separable=False)
    psi, ref = _to_dev(p["psi0"], dtype), _oracle_input(p["psi0"], dtype)
    o = Oracle(p)
    rg = plan.evolve(psi, 1e-3, 12, mode, record_every=1).cpu().numpy()
    ro = o.evolve(ref, 1e-3, 12, mode == "imag", record_every=1)
    out = psi.cpu().numpy()
    for b in range(B):
        e = _rel(out[b], ref[b])
        assert e <= 12 * PER_STEP[dtype], (b, e)
    assert np.allclose(rg[:, :, 5], ro[:, :, 5], rtol=1e-14, atol=1e-300)       # A_n of every member and step
    assert len({tuple(ro[:, b, 5]) for b in range(B)}) == B                     # the members really differ
    tol = 1e-5 if dtype == "c64" else 1e-10
    assert np.all(np.abs(rg[:, :, 2] - ro[:, :, 2]) <= tol * np.maximum(np.abs(ro[:, :, 2]), 1e-2))
    # the members' arrays matter: member 1 evolved under member 0's array is far outside the bar
    q = W.member(p, 1)
    q["v_static"] = vs[0]
    other = _oracle_input(q["psi0"], dtype)
    Oracle(q).evolve(other, 1e-3, 12, mode == "imag")
    assert _rel(other, ref[1]) > 100 * PER_STEP["c64"]
    plan.close()


SIZES = [(64, 64), (128, 128), (256, 256), (512, 512), (1024, 1024), (2048, 2048), (64, 256), (1024, 128), (128, 2048)]


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("nx,ny", SIZES)
def test_fft2_forward_alone(nx, ny, dtype):
    """gpe_fft2_forward on its own against the oracle's transform: an impulse at the
    origin (-> all ones), a shifted impulse (-> the plane wave exp(-2 pi i (p i0/nx + q j0/ny)): sign and
    axis order), seeded noise, out of place and in place; Parseval on the noise."""
    import paper_2404_14401_b200 as G
    torch = _torch()
    cd = np.complex64 if dtype == "c64" else np.complex128
    eps = 6e-8 if dtype == "c64" else 1.2e-16
    plan = G.Plan(nx, ny, 1.0, 1.0, dtype, 1)
    rng = np.random.default_rng(nx * 7 + ny)
    i0, j0 = 3 % nx, (ny // 2 + 5) % ny
    imp0 = np.zeros((nx, ny), dtype=cd); imp0[0, 0] = 1.0
    imp1 = np.zeros((nx, ny), dtype=cd); imp1[i0, j0] = 2.0 - 1.0j
    noise = (rng.standard_normal((nx, ny)) + 1j * rng.standard_normal((nx, ny))).astype(cd)
    for name, a in (("impulse", imp0), ("shifted impulse", imp1), ("noise", noise)):
        src = torch.from_numpy(a.copy()).cuda()
        dst = torch.empty_like(src)
        G.gpe_fft2_forward(plan.plan, src.data_ptr(), dst.data_ptr())
        got = dst.cpu().numpy().astype(np.complex128)
        want = gpe_oracle.fft2(a.astype(np.complex128))
        if name == "impulse":
            assert np.max(np.abs(got - 1.0)) <= 16 * eps
        if name == "shifted impulse":
            # phases reduced mod 1 in integers first, so that the reference itself is good to an ulp
            ph = ((np.arange(nx) * i0) % nx)[:, None] / nx + ((np.arange(ny) * j0) % ny)[None, :] / ny
            pw = (2.0 - 1.0j) * np.exp(-2j * np.pi * ph)
            assert np.max(np.abs(got - pw)) <= 64 * eps * abs(2.0 - 1.0j)
        e = _rel(got, want)
        assert e <= 40 * eps, f"{name}: {e:.3e}"
        if name == "noise":
            lhs, rhs = np.sum(np.abs(got) ** 2), nx * ny * np.sum(np.abs(a.astype(np.complex128)) ** 2)
            assert abs(lhs - rhs) <= 200 * eps * rhs
            G.gpe_fft2_forward(plan.plan, src.data_ptr(), src.data_ptr())          # in place
            assert np.array_equal(src.cpu().numpy(), dst.cpu().numpy())
    plan.close()


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("mode", ["real", "imag"])
def test_tvt_with_full_cavity_model_and_probe(mode, dtype):
    """ordering = 1 together with cav_u0 (cavity lattice + dispersive shift, Eqs. 12, 15) and an on-axis
    probe (Eq. 17): psi and the records against the oracle over two calls."""
    p = _general_workload(256, 128, batch=2)
    p["ordering"] = 1
    p["cav_u0"] = np.array([8.0, 0.0])
    p["probe_omega"], p["probe_delta"], p["probe_phi"] = np.array([3.0, 0.5]), np.array([30.0, 5.0]), np.array([0.2, 1.0])
    plan = _gpu_plan(p, dtype)
    psi, ref = _to_dev(p["psi0"], dtype), _oracle_input(p["psi0"], dtype)
    o = Oracle(p)
    rg = np.concatenate([plan.evolve(psi, 1e-3, n, mode, record_every=2).cpu().numpy()[:k] for n, k in ((3, 1), (9, 5))])
    ro = np.concatenate([o.evolve(ref, 1e-3, n, mode == "imag", record_every=2) for n in (3, 9)])
    e = _rel(psi.cpu().numpy(), ref)
    assert e <= 12 * PER_STEP[dtype], f"{e:.3e}"
    tol = 1e-5 if dtype == "c64" else 1e-10
    assert rg.shape == ro.shape
    assert np.array_equal(rg[:, :, 0], ro[:, :, 0])
    for c in (1, 2, 3, 4, 5):
        assert np.all(np.abs(rg[:, :, c] - ro[:, :, c]) <= tol * np.maximum(np.abs(ro[:, :, c]), 1e-2)), c
    plan.close()


def test_negative_step_rejected_and_records_indexing():
    """gpe_set_step(< 0) is GPE_EINVAL (the record index and the T/2 V T/2 chunking use truncating
    division: ADVICE round 1); a start that is not a multiple of record_every writes the right rows."""
    import paper_2404_14401_b200 as G
    p = _general_workload(64, 64)
    plan = _gpu_plan(p, "c64")
    with pytest.raises(G.GpeError) as e:
        plan.step = -5
    assert e.value.status == 1
    assert plan.step == 0
    for ordering in (0, 1):
        q = {**p, "ordering": ordering}
        plan.set_potential(q)
        plan.step = 7
        psi, ref = _to_dev(p["psi0"], "c64"), _oracle_input(p["psi0"], "c64")
        o = Oracle(q)
        o.step = 7
        rg = plan.evolve(psi, 1e-3, 10, "real", record_every=4).cpu().numpy()
        ro = o.evolve(ref, 1e-3, 10, False, record_every=4)
        assert rg.shape == ro.shape == (3, 1, 6)                # steps 8, 12, 16
        assert np.array_equal(rg[:, :, 0], ro[:, :, 0])
        assert np.all(np.abs(rg[:, :, 2] - ro[:, :, 2]) <= 1e-5 * np.maximum(np.abs(ro[:, :, 2]), 1e-2))
    plan.close()


def test_set_potential_is_all_or_nothing():
    """A rejected gpe_set_potential (here: ordering = 2 with a longer schedule) leaves the previous
    potential in force, untouched (sched_len was overwritten before validation ended)."""
    import paper_2404_14401_b200 as G
    p = _general_workload(128, 128)
    outs = []
    for poke in (False, True):
        plan = _gpu_plan(p, "c64")
        if poke:
            bad = {**p, "ordering": 2, "sched_step": np.arange(64.0), "sched_amp": np.linspace(0.0, 50.0, 64),
                   "cavity_on": 0, "lattice_axis": 0}
            with pytest.raises(G.GpeError) as e:
                plan.set_potential(bad)
            assert e.value.status == 1
        psi = _to_dev(p["psi0"], "c64")
        rec = plan.evolve(psi, 1e-3, 6, "real", record_every=1)
        outs.append((psi.cpu().numpy(), rec.cpu().numpy()))
        plan.close()
    assert np.array_equal(outs[0][0], outs[1][0])
    assert np.array_equal(outs[0][1], outs[1][1])


def test_abi_null_descriptor_nomem_and_flag_reset():
    """NULL descriptor -> GPE_EINVAL; an allocation the device cannot satisfy -> GPE_ENOMEM with *out
    untouched; GPE_ENONFINITE is reported once, the output is filled, and the plan is usable again."""
    import paper_2404_14401_b200 as G
    torch = _torch()
    lib = G.load_library()
    plan = G.gpe_plan_create(64, 64, 16.0, 16.0, G.GPE_C64, 1)
    assert lib.gpe_set_potential(plan, None) == 1
    assert b"NULL" in lib.gpe_last_error(plan)
    out = C.c_void_p(0x1234)
    st = lib.gpe_plan_create(C.byref(out), 64, 64, 1.0, 1.0, G.GPE_C64, 2 ** 31 - 1)
    assert st == 3, (st, lib.gpe_last_error(None))
    assert out.value == 0x1234
    G.gpe_set_potential(plan, G.gpe_potential_desc(lattice_axis=-1))
    zero = torch.zeros((64, 64), dtype=torch.complex64, device="cuda")
    G.gpe_evolve(plan, zero.data_ptr(), 1e-3, 2, G.GPE_IMAG_TIME)           # norm 0 -> non-finite scale
    with pytest.raises(G.GpeError) as e:
        G.gpe_observables(plan, zero.data_ptr(), 1)
    assert e.value.status == 6
    good = _to_dev(W.noisy_gaussian(64, 64, 16.0, 16.0), "c64")
    G.gpe_evolve(plan, good.data_ptr(), 1e-3, 2, G.GPE_IMAG_TIME)
    obs = G.gpe_observables(plan, good.data_ptr(), 1)                       # the flag was cleared
    assert obs[0]["norm"] == pytest.approx(1.0, abs=1e-5)
    G.gpe_plan_destroy(plan)


@pytest.mark.parametrize("ordering", [0, 1])
def test_evolve_only_enqueues(ordering):
    """include/gpe.h: gpe_evolve "only ENQUEUES": a first call with a new (dt, mode) -- which has to
    build the kinetic tables -- returns while a long kernel queued before it on the same stream is still
    running, in both time modes and with the second table set of ordering = 1."""
    torch = _torch()
    import paper_2404_14401_b200 as G
    p = _general_workload(256, 256)
    p["ordering"] = ordering
    stream = torch.cuda.Stream()
    plan = G.Plan(256, 256, p["Lx"], p["Ly"], "c64", 1, stream=stream.cuda_stream)
    with torch.cuda.stream(stream):
        plan.set_potential(p)
        psi = _to_dev(p["psi0"], "c64")
        plan.evolve(psi, 2e-3, 2, "real")              # first launches (function attributes, lazy module load)
        plan.evolve(psi, 2e-3, 2, "imag")
    stream.synchronize()
    spin_cycles = int(0.4 * 1.9e9)                     # about 0.4 s at the B200's clock
    for mode, dt in (("real", 1e-3), ("imag", 5e-4), ("real", 7e-4)):
        with torch.cuda.stream(stream):
            torch.cuda._sleep(spin_cycles)
            t0 = time.perf_counter()
            plan.evolve(psi, dt, 3, mode)
            t_call = time.perf_counter() - t0
            done_at_return = stream.query()
        stream.synchronize()
        t_total = time.perf_counter() - t0
        assert not done_at_return, "the spin kernel had already finished: nothing was shown"
        assert t_call < 0.5 * t_total, f"{mode}: gpe_evolve blocked for {t_call:.3f} s of {t_total:.3f} s"
    ref = _oracle_input(p["psi0"], "c64")
    o = Oracle(p)
    for mode, dt, n in (("real", 2e-3, 2), ("imag", 2e-3, 2), ("real", 1e-3, 3), ("imag", 5e-4, 3), ("real", 7e-4, 3)):
        o.evolve(ref, dt, n, mode == "imag")
    assert _rel(psi.cpu().numpy(), ref) <= 13 * PER_STEP["c64"]      # the tables built on the device are right
    plan.close()


def _records_ok(rg, ro, tol):
    """step and A exact; norm and Theta by reading Q17; alpha by Q17's bound on Theta carried through Eq. 14
    (alpha = K Theta + probe: an error dTheta moves alpha by |K| dTheta, and |K| = N eta / |Delta + i kappa|
    is about 7 in these workloads, so a flat 1e-5 max(|alpha|, 1e-2) would be tighter than the Theta bar)."""
    assert rg.shape == ro.shape
    assert np.array_equal(rg[:, :, 0], ro[:, :, 0])
    assert np.allclose(rg[:, :, 5], ro[:, :, 5], rtol=1e-14, atol=1e-300)
    assert np.all(np.abs(rg[:, :, 1] - ro[:, :, 1]) <= tol * np.abs(ro[:, :, 1]))
    th = np.maximum(np.abs(ro[:, :, 2]), 1e-2)
    assert np.all(np.abs(rg[:, :, 2] - ro[:, :, 2]) <= tol * th)
    gain = np.maximum(np.hypot(ro[:, :, 3], ro[:, :, 4]) / np.maximum(np.abs(ro[:, :, 2]), 1e-300), 1.0)
    gain = np.where(np.abs(ro[:, :, 2]) > 1e-12, gain, 1.0)
    for c in (3, 4):
        assert np.all(np.abs(rg[:, :, c] - ro[:, :, c]) <= tol * th * np.maximum(gain, 1.0)), c


def _local_workload(nx, ny, batch=1, g=40.0, v2d=False):
    """No cavity term: static trap (+ optional 2-D array), ramped lattice, contact interaction."""
    p = _general_workload(nx, ny, batch=batch)
    p["cavity_on"] = 0
    p["g"] = np.linspace(g, 1.5 * g, batch)
    return p   # v_static stays: the oracle knows the trap only as a 2-D array (the GPU may take vx + vy instead)


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("nx,ny,batch", [(64, 64, 1), (256, 256, 1), (128, 512, 2), (1024, 128, 1), (2048, 2048, 1)])
def test_two_pass_real_time(monkeypatch, nx, ny, batch, dtype):
    """The 2-pass form (real time with a local potential runs IFFT_y -> full potential factor
    -> FFT_y in one kernel): psi and the records against the oracle for step counts on both sides of the
    CUDA-graph threshold, over two calls, and against the 3-pass form of the same library (GPE_NO_FUSE)."""
    torch = _torch()
    for k in ("GPE_NO_PAIR", "GPE_NO_MERGE", "GPE_NO_FUSE"):
        monkeypatch.delenv(k, raising=False)
    big = nx * ny >= 2048 * 2048
    p = _local_workload(nx, ny, batch, v2d=(nx == 256))
    counts = (2, 5) if big else (3, 40)
    ref = _oracle_input(p["psi0"], dtype)
    o = Oracle(p)
    ro = np.concatenate([o.evolve(ref, 1e-3, n, False, record_every=1) for n in counts])
    outs = []
    for fuse in (True, False):
        if not fuse:
            monkeypatch.setenv("GPE_NO_FUSE", "1")
        plan = _gpu_plan(p, dtype, use_separable=(nx != 256))
        psi = _to_dev(p["psi0"], dtype)
        rg = np.concatenate([plan.evolve(psi, 1e-3, n, "real", record_every=1).cpu().numpy()[:n] for n in counts])
        torch.cuda.synchronize()
        out = psi.cpu().numpy()
        e = _rel(out, ref)
        assert e <= sum(counts) * PER_STEP[dtype], f"fuse={fuse}: {e:.3e}"
        assert np.array_equal(rg[:, :, 0], ro[:, :, 0])
        tol = 1e-5 if dtype == "c64" else 1e-10
        assert np.allclose(rg[:, :, 1], ro[:, :, 1], rtol=tol, atol=0)          # the computed norm, every step
        assert np.allclose(rg[:, :, 5], ro[:, :, 5], rtol=1e-14, atol=1e-300)
        assert plan.step == sum(counts)
        outs.append(out)
        plan.close()
    assert _rel(outs[0], outs[1].astype(np.complex128)) <= (2e-6 if dtype == "c64" else 1e-13)


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("n", [64, 128, 512, 2048])
def test_two_pass_imag_time_linear(monkeypatch, n, dtype):
    """The 2-pass form in imaginary time with g = 0 and no cavity term (the paper's Sec. 4.1 workload,
    PAPER.md:130-132): the lagging lazy scale must not change the result -- psi after a run that ends in the
    plain pass C is the oracle's (renormalised every step), norm 1, same energies."""
    monkeypatch.delenv("GPE_NO_FUSE", raising=False)
    p = W.sweep_s(n, dtype)
    steps = 6 if n == 2048 else 60
    plan = _gpu_plan(p, dtype)
    psi, ref = _to_dev(p["psi0"], dtype), _oracle_input(p["psi0"], dtype)
    o = Oracle(p)
    rec = plan.evolve(psi, 1e-3, steps, "imag", record_every=3).cpu().numpy()
    o.evolve(ref, 1e-3, steps, True)
    e = _rel(psi.cpu().numpy(), ref)
    assert e <= min(steps, 20) * PER_STEP[dtype], f"{e:.3e}"
    assert np.allclose(rec[:, :, 1], 1.0, atol=1e-12)
    go, oo = plan.observables(psi)[0][0], o.observables(ref)[0][0]
    tol = 1e-5 if dtype == "c64" else 1e-10
    assert abs(go["norm"] - 1.0) <= (2e-6 if dtype == "c64" else 1e-13)
    for k in ("e_kin", "e_pot"):
        assert abs(go[k] - oo[k]) <= tol * abs(oo[k]), k
    plan.close()


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("mode", ["real", "imag"])
@pytest.mark.parametrize("n,batch", [(64, 1), (128, 3), (256, 1)])
def test_cluster_kernel_and_multi_launch_path_agree(monkeypatch, n, batch, mode, dtype):
    """Square grids up to 256^2 run all steps of a call in one cluster kernel (gpe_chip.cuh); GPE_NO_CHIP
    forces the multi-launch passes for the same sizes.  Both against the oracle (everything switched on:
    2-D array, lattice ramp, cavity, g; records every step, two calls), and against each other."""
    torch = _torch()
    for k in ("GPE_NO_PAIR", "GPE_NO_MERGE", "GPE_NO_FUSE", "GPE_NO_CHIP"):
        monkeypatch.delenv(k, raising=False)
    p = _general_workload(n, n, batch=batch)
    ref = _oracle_input(p["psi0"], dtype)
    o = Oracle(p)
    counts = (1, 24)
    ro = np.concatenate([o.evolve(ref, 1e-3, c, mode == "imag", record_every=1) for c in counts])
    outs = []
    for chip in (True, False):
        if not chip:
            monkeypatch.setenv("GPE_NO_CHIP", "1")
        plan = _gpu_plan(p, dtype, use_separable=False)
        psi = _to_dev(p["psi0"], dtype)
        rg = np.concatenate([plan.evolve(psi, 1e-3, c, mode, record_every=1).cpu().numpy()[:c] for c in counts])
        torch.cuda.synchronize()
        out = psi.cpu().numpy()
        e = _rel(out, ref)
        assert e <= 25 * PER_STEP[dtype], f"chip={chip}: {e:.3e}"
        _records_ok(rg, ro, 1e-5 if dtype == "c64" else 1e-10)
        assert plan.step == 25
        outs.append(out)
        plan.close()
    assert _rel(outs[0], outs[1].astype(np.complex128)) <= (5e-6 if dtype == "c64" else 1e-13)


def test_measure_roofs_is_sane():
    """gpe_measure_roofs (the denominators bench.py reports against): positive, ordered as the memory hierarchy
    is (L2-resident >= 0.8 x HBM-resident), fp32 FMA rate above fp64's, and the call leaves no error behind."""
    import paper_2404_14401_b200 as G
    r = G.gpe_measure_roofs(_torch().cuda.current_stream().cuda_stream)
    assert 1000.0 < r["hbm_rw_1GiB_gbs"] < 20000.0
    assert r["l2_rw_32MiB_gbs"] >= 0.8 * r["hbm_rw_1GiB_gbs"] and r["l2_rw_64MiB_gbs"] >= 0.8 * r["hbm_rw_1GiB_gbs"]
    assert 10.0 < r["fp64_fma_tflops"] < r["fp32_fma_tflops"] < 400.0
    p = _general_workload(64, 64)
    plan = _gpu_plan(p, "c64")
    plan.evolve(_to_dev(p["psi0"], "c64"), 1e-3, 2, "real")
    plan.close()


@pytest.mark.parametrize("dtype", ["c64", "c128"])
def test_two_pass_with_midpoint_schedule_and_batch(monkeypatch, dtype):
    """The fused C+A kernel takes A_{n+1} from the coefficients pass B prepared: with mid-step sampling of a ramp
    (sched_midpoint) and a different schedule per member, on a non-square grid (multi-launch 2-pass path)."""
    monkeypatch.delenv("GPE_NO_FUSE", raising=False)
    p = _local_workload(256, 128, batch=2)
    p["sched_midpoint"] = 1
    p["sched_step"] = np.array([0.0, 5.0, 5.0, 30.0])
    p["sched_amp"] = np.array([[6.0, 6.0, 9.0, 12.0], [0.0, 10.0, 3.0, 0.0]])
    plan = _gpu_plan(p, dtype)
    psi, ref = _to_dev(p["psi0"], dtype), _oracle_input(p["psi0"], dtype)
    o = Oracle(p)
    rg = plan.evolve(psi, 1e-3, 33, "real", record_every=1).cpu().numpy()
    ro = o.evolve(ref, 1e-3, 33, False, record_every=1)
    e = _rel(psi.cpu().numpy(), ref)
    assert e <= 33 * PER_STEP[dtype], f"{e:.3e}"
    assert np.allclose(rg[:, :, 5], ro[:, :, 5], rtol=1e-14, atol=1e-300)
    assert np.allclose(rg[:, :, 1], ro[:, :, 1], rtol=1e-5 if dtype == "c64" else 1e-10, atol=0)
    plan.close()
