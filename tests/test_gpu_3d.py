"""Parity of the 3-D CUDA path (gpe3_*, csrc/gpe3_kernels.cuh) with the 3-D oracle (oracle/gpe3_oracle.c),
element by element on the same seeded inputs, through the C ABI.  SURVEY.md 8(f) f4 (second half).

Tolerances (DESIGN.md section 9 carried to three axes): complex128 relative L2 <= 1e-11 after tens of steps (three
transforms of <= 512 points per axis, rounding ~ log2(P) eps per step); complex64 <= 2e-6 * sqrt(steps) + 2e-6 against
the complex128 oracle on the same fp32-rounded input, the potential array rounded to fp32 as the library holds it.
Observables: 1e-10 relative (complex128), 2e-5 (complex64).
"""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu


def _rel(a, b):
    a = np.asarray(a, dtype=np.complex128).ravel()
    b = np.asarray(b, dtype=np.complex128).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def _run_both(p, dtype, mode, dt, n_steps, record_every=0, chunks=1):
    import torch
    import paper_2404_14401_b200 as G
    from oracle.gpe3_oracle import Oracle3
    cd = np.complex64 if dtype == "c64" else np.complex128
    psi0 = p["psi0"].astype(cd)
    q = dict(p)
    if dtype == "c64" and p.get("v_static") is not None:   # the library holds V in the plan's real type
        q["v_static"] = p["v_static"].astype(np.float32).astype(np.float64)
    for k in ("vx", "vy", "vz"):
        if dtype == "c64" and p.get(k) is not None:
            q[k] = p[k].astype(np.float32).astype(np.float64)
    q["g"] = float(np.float32(p["g"])) if dtype == "c64" else p["g"]
    o = Oracle3(q)
    ref = np.ascontiguousarray(psi0.astype(np.complex128))
    plan = G.Plan3(p["nx"], p["ny"], p["nz"], p["Lx"], p["Ly"], p["Lz"], dtype)
    plan.set_potential(p)
    psi = torch.from_numpy(psi0).cuda()
    recs_o, recs_g = [], []
    per = n_steps // chunks
    for c in range(chunks):
        n = per if c < chunks - 1 else n_steps - per * (chunks - 1)
        ro = o.evolve(ref, dt, n, mode == "imag", record_every)
        rg = plan.evolve(psi, dt, n, mode, record_every)
        if ro is not None and len(ro):
            recs_o.append(ro); recs_g.append(rg.cpu().numpy()[:len(ro)])
    plan.synchronize()
    out = psi.cpu().numpy()
    obs_g = plan.observables(psi)
    obs_o = o.observables(ref)
    plan.close()
    return out, ref, (np.concatenate(recs_g) if recs_g else None), (np.concatenate(recs_o) if recs_o else None), obs_g, obs_o


def _tol(dtype, steps):
    return 1e-11 if dtype == "c128" else 2e-6 * np.sqrt(steps) + 2e-6


def _check_obs(obs_g, obs_o, dtype):
    rt = 1e-10 if dtype == "c128" else 2e-5
    scale = abs(obs_o["e_kin"]) + abs(obs_o["e_pot"]) + abs(obs_o["e_int"])
    for k in ("norm", "x2", "y2", "z2"):
        assert obs_g[k] == pytest.approx(obs_o[k], rel=rt), k
    for k in ("e_kin", "e_pot", "e_int"):
        assert abs(obs_g[k] - obs_o[k]) <= rt * scale, k


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("mode", ["real", "imag"])
def test_cube_64(dtype, mode):
    p = W.config3d(64, g=50.0)
    out, ref, _, _, og, oo = _run_both(p, dtype, mode, 1e-3, 20)
    assert _rel(out, ref) <= _tol(dtype, 20)
    _check_obs(og, oo, dtype)


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("shape", [(128, 64, 64), (64, 128, 64), (64, 64, 128), (128, 256, 64), (64, 128, 512)])
def test_every_axis_length(dtype, shape):
    """each axis takes each template size at least once (512 and 256 on the two strided axes and on the rows);
    three different lengths catch any mix-up of nx / ny / nz in the strides"""
    nx, ny, nz = shape
    for mode in ("real", "imag"):
        p = W.config3d(nx, ny, nz, g=40.0, seed=3)
        out, ref, _, _, og, oo = _run_both(p, dtype, mode, 1e-3, 6)
        assert _rel(out, ref) <= _tol(dtype, 6), mode
        _check_obs(og, oo, dtype)


@pytest.mark.parametrize("dtype", ["c64", "c128"])
def test_lengths_256_and_512_on_x_and_rows(dtype):
    for shape in ((256, 64, 64), (512, 64, 64), (64, 512, 64), (64, 64, 256)):
        p = W.config3d(*shape, g=30.0, seed=4)
        out, ref, _, _, _, _ = _run_both(p, dtype, "real", 1e-3, 3)
        assert _rel(out, ref) <= _tol(dtype, 3), shape


@pytest.mark.parametrize("dtype", ["c64", "c128"])
def test_elongated_grids_1024(dtype):
    """1024 points along each axis in turn (cigar-shaped traps): the longest line the 3-D passes take"""
    for shape in ((1024, 64, 64), (64, 1024, 64), (64, 64, 1024)):
        for mode in ("real", "imag"):
            p = W.config3d(*shape, g=30.0, seed=6)
            out, ref, _, _, og, oo = _run_both(p, dtype, mode, 1e-3, 4)
            assert _rel(out, ref) <= _tol(dtype, 4), (shape, mode)
            _check_obs(og, oo, dtype)


@pytest.mark.parametrize("dtype", ["c64", "c128"])
def test_records_and_chunked_calls(dtype):
    """records of both time modes, and a run split over several calls equals one call (step counter, merged
    half-steps across the call boundary, lazy scale applied at the end of every imaginary-time call)"""
    for mode in ("real", "imag"):
        p = W.config3d(64, 64, 128, g=60.0, seed=5)
        out, ref, rg, ro, _, _ = _run_both(p, dtype, mode, 2e-3, 12, record_every=4, chunks=3)
        assert _rel(out, ref) <= _tol(dtype, 12)
        assert rg.shape == ro.shape == (3, 3)
        assert np.array_equal(rg[:, 0], ro[:, 0])
        rt = 1e-11 if dtype == "c128" else 5e-6
        assert np.abs(rg[:, 1] - ro[:, 1]).max() <= rt
        assert np.abs(rg[:, 2] / ro[:, 2] - 1).max() <= rt


def test_potential_forms_agree():
    """the separable arrays and the same potential handed in as one 3-D array give the same result (c128: both exact
    in double up to the order of the additions)"""
    a = _run_both(W.config3d(64, 128, 64, g=25.0, separable=True), "c128", "real", 1e-3, 5)[0]
    b = _run_both(W.config3d(64, 128, 64, g=25.0, separable=False), "c128", "real", 1e-3, 5)[0]
    assert _rel(a, b) <= 1e-13


def test_no_potential_no_interaction_is_free_expansion():
    """g = 0, V = 0: closed form <x^2>(t) = s0^2/2 + t^2/(2 s0^2) per axis, through the library alone"""
    import torch
    import paper_2404_14401_b200 as G
    nx, ny, nz, L = 64, 128, 64, 40.0
    s0 = (1.6, 1.2, 2.0)
    x = W.axis(nx, L)[None, :, None]; y = W.axis(ny, L)[None, None, :]; z = W.axis(nz, L)[:, None, None]
    psi = np.exp(-x * x / (2 * s0[0] ** 2) - y * y / (2 * s0[1] ** 2) - z * z / (2 * s0[2] ** 2)).astype(np.complex128)
    psi /= np.sqrt(np.sum(np.abs(psi) ** 2) * (L / nx) * (L / ny) * (L / nz))
    plan = G.Plan3(nx, ny, nz, L, L, L, "c128")
    plan.set_potential(dict(g=0.0))
    t = torch.from_numpy(np.ascontiguousarray(psi)).cuda()
    plan.evolve(t, 0.05, 40, "real")
    ob = plan.observables(t)
    for k, s in zip(("x2", "y2", "z2"), s0):
        assert ob[k] == pytest.approx(s * s / 2 + 4.0 / (2 * s * s), rel=1e-8)
    assert ob["norm"] == pytest.approx(1.0, abs=1e-12)
    plan.close()


def test_boundary_errors():
    import torch
    import paper_2404_14401_b200 as G
    for bad in ((96, 64, 64), (64, 32, 64), (64, 64, 2048)):
        with pytest.raises(G.GpeError, match="GPE_EUNSUPPORTED"):
            G.Plan3(*bad, 1.0, 1.0, 1.0)
    with pytest.raises(G.GpeError, match="GPE_EINVAL"):
        G.Plan3(64, 64, 64, 1.0, -1.0, 1.0)
    plan = G.Plan3(64, 64, 64, 8.0, 8.0, 8.0, "c64")
    psi = torch.zeros((64, 64, 64), dtype=torch.complex64, device="cuda")
    with pytest.raises(G.GpeError, match="GPE_ESTATE"):
        plan.evolve(psi, 1e-3, 1, "real")
    plan.set_potential(dict(g=1.0))
    with pytest.raises(G.GpeError, match="GPE_EINVAL"):
        plan.evolve(psi, -1e-3, 1, "imag")
    with pytest.raises(G.GpeError, match="GPE_EINVAL"):
        plan.evolve(psi, float("nan"), 1, "real")
    with pytest.raises(G.GpeError, match="GPE_EINVAL"):
        G.gpe3_set_potential(plan.plan, None, np.full(64, np.inf), None, None, 0.0)
    # a zero wavefunction in imaginary time: the norm is zero -> reported once by the next synchronize
    plan.evolve(psi, 1e-3, 1, "imag")
    with pytest.raises(G.GpeError, match="GPE_ENONFINITE"):
        plan.synchronize()
    plan.synchronize()
    with pytest.raises(G.GpeError, match="GPE_EINVAL"):
        plan.step = -1
    plan.close()


@pytest.mark.parametrize("dtype", ["c64", "c128"])
def test_full_size_256_cubed(dtype):
    """the bench workload (256^3, the launch configuration bench.py times), whole array against the oracle"""
    p = W.config3d(256, g=50.0)
    out, ref, _, _, og, oo = _run_both(p, dtype, "imag", 1e-3, 3)
    assert _rel(out, ref) <= _tol(dtype, 3)
    _check_obs(og, oo, dtype)
    out, ref, _, _, _, _ = _run_both(p, dtype, "real", 1e-3, 3)
    assert _rel(out, ref) <= _tol(dtype, 3)


def test_largest_grid_properties():
    """512^3 complex64 (1 GiB of wavefunction, the largest grid the boundary takes): what holds at any size --
    norm conservation in real time, time reversal (the symmetric splitting is its own inverse under dt -> -dt), and
    sampled lines of the kinetic factor against the closed form for a plane wave"""
    import torch
    import paper_2404_14401_b200 as G
    n, L = 512, 20.0
    plan = G.Plan3(n, n, n, L, L, L, "c64")
    x = torch.linspace(-L / 2, L / 2 - L / n, n, device="cuda", dtype=torch.float32)
    g = torch.Generator(device="cuda").manual_seed(3)
    psi = torch.exp(-(x[None, :, None] ** 2 / 8 + x[None, None, :] ** 2 / 6 + x[:, None, None] ** 2 / 10)).to(torch.complex64)
    psi = psi * (1 + 0.05 * torch.randn((n, n, n), device="cuda", generator=g))
    dV = (L / n) ** 3
    psi /= torch.sqrt((psi.real ** 2 + psi.imag ** 2).sum(dtype=torch.float64) * dV).to(torch.float32)
    start = psi.clone()
    xs = np.asarray(W.axis(n, L))
    G.gpe3_set_potential(plan.plan, None, 0.5 * xs ** 2, 0.7 * xs ** 2, 0.4 * xs ** 2, 80.0)
    rec = plan.evolve(psi, 1e-3, 4, "real", record_every=2).cpu().numpy()
    assert np.abs(rec[:, 1] - 1.0).max() <= 2e-6
    assert float((psi - start).abs().max()) > 1e-4          # it moved
    plan.evolve(psi, -1e-3, 4, "real")
    plan.synchronize()
    err = torch.sqrt(((psi - start).abs() ** 2).sum(dtype=torch.float64) / (start.abs() ** 2).sum(dtype=torch.float64))
    assert float(err) <= 1e-5
    # a plane wave with mode numbers (3, -7, 5) on (x, y, z), V = 0, g = 0: one step multiplies it by e^{-i |k|^2 dt/2}
    G.gpe3_set_potential(plan.plan, None, None, None, None, 0.0)
    k = 2 * np.pi / L * np.array([3.0, -7.0, 5.0])
    ph = (k[0] * x.double()[None, :, None] + k[1] * x.double()[None, None, :] + k[2] * x.double()[:, None, None])
    wave = torch.complex(torch.cos(ph), torch.sin(ph)).to(torch.complex64)
    del ph, start
    ref_line = wave[17, 33, :].cpu().numpy().astype(np.complex128) * np.exp(-0.5j * float(k @ k) * 1e-2)
    plan.evolve(wave, 1e-2, 1, "real")
    got = wave[17, 33, :].cpu().numpy().astype(np.complex128)
    assert np.abs(got - ref_line).max() <= 5e-6
    plan.close()


@pytest.mark.parametrize("mode", ["real", "imag"])
def test_graph_replay_with_records(mode):
    """small grids replay eight plain steps from a CUDA graph; records, the first and the last step of a call stay
    outside it: 45 steps with a record every 10, then a second call that continues the count"""
    p = W.config3d(64, g=40.0, seed=8)
    out, ref, rg, ro, og, oo = _run_both(p, "c128", mode, 1e-3, 45 + 27, record_every=10, chunks=2)
    assert _rel(out, ref) <= 1e-11
    assert rg.shape == ro.shape and np.array_equal(rg[:, 0], ro[:, 0]) and len(rg) == 7
    assert np.abs(rg[:, 1:] / ro[:, 1:] - 1).max() <= 1e-11
    _check_obs(og, oo, "c128")


def test_graph_survives_a_new_potential_a_new_dt_and_a_user_stream():
    """the graph of plain steps holds g, dt/2 and the potential pointers as kernel arguments: a second
    gpe3_set_potential, another dt and another wavefunction buffer must each rebuild it; all work on a user stream"""
    import torch
    import paper_2404_14401_b200 as G
    from oracle.gpe3_oracle import Oracle3
    p = W.config3d(64, g=30.0, seed=12)
    q = W.config3d(64, g=75.0, seed=12, w2=(0.5, 2.0, 1.0), dimple=-1.0)
    stream = torch.cuda.Stream()
    plan = G.Plan3(64, 64, 64, p["Lx"], p["Ly"], p["Lz"], "c128", stream=stream.cuda_stream)
    ref = p["psi0"].copy()
    with torch.cuda.stream(stream):
        psi = torch.from_numpy(p["psi0"].copy()).cuda()
        plan.set_potential(p)
        plan.evolve(psi, 1e-3, 20, "real")
        plan.evolve(psi, 2e-3, 20, "real")          # another dt
        plan.set_potential(q)                         # another potential and g
        plan.evolve(psi, 2e-3, 20, "real")
        psi2 = psi.clone()                            # another buffer
        plan.evolve(psi2, 2e-3, 20, "imag")
        plan.evolve(psi2, 2e-3, 20, "imag")
    plan.synchronize()
    o = Oracle3(p)
    o.evolve(ref, 1e-3, 20, False); o.evolve(ref, 2e-3, 20, False)
    o2 = Oracle3(q)
    o2.evolve(ref, 2e-3, 20, False)
    assert _rel(psi.cpu().numpy(), ref) <= 1e-11
    o2.evolve(ref, 2e-3, 40, True)
    assert _rel(psi2.cpu().numpy(), ref) <= 1e-11
    plan.close()


def test_graph_with_large_tiles_first_in_a_fresh_plan():
    """64 x 64 x 512 in complex128 is small enough for the step graph while its 512-point passes need more than 48 KB of
    shared memory: the opt-in attribute must be set by a direct launch before the capture"""
    p = W.config3d(64, 64, 512, g=20.0, seed=13)
    out, ref, _, _, _, _ = _run_both(p, "c128", "imag", 1e-3, 20)
    assert _rel(out, ref) <= 1e-11
    p = W.config3d(512, 64, 64, g=20.0, seed=14)
    out, ref, _, _, _, _ = _run_both(p, "c128", "real", 1e-3, 20)
    assert _rel(out, ref) <= 1e-11
