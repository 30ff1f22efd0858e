"""Writes tests/golden/oracle_regression.json: values of the CPU oracle on small seeded workloads,
to guard the oracle's arithmetic against accidental changes (a later deliberate change re-runs this
script and says why in its commit message).  Calls only oracle/ and the seeded input generators
(workloads/); nothing here comes from the CUDA path.

    python tests/golden/make_golden.py
"""
from __future__ import annotations

import json
import math
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import workloads as W                      # noqa: E402
from oracle.gpe_oracle import Oracle       # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.json")


def cases():
    """name -> (params, [(dt, n_steps, imag_time)], record_every)"""
    out = {}
    for g in (0.0, 10.0):            # BASELINE.json configs[0]
        p = W.config1(g=g)
        out[f"config1_g{g:g}"] = (p, [(1e-3, 2000, True)], 0)
    L = 4 * math.pi                  # cavity with every term on, both time modes
    p = W._cavity(W._with_trap(W._base(64, 64, L)), 1, 8.0, -1.0, 5.0)
    p["sched_step"], p["sched_amp"] = np.array([0.0, 40.0]), np.array([6.0, 10.0])
    p["psi0"] = W.noisy_gaussian(64, 64, L, L, 1.2, 7)
    out["cavity64_imag_then_real"] = (p, [(5e-4, 24, True), (1e-3, 24, False)], 8)
    q = dict(p)                      # SURVEY.md 8(f) f1 + f2: full cavity model and probe
    q["cav_u0"] = np.array([2.0])
    q["probe_omega"], q["probe_delta"], q["probe_phi"] = np.array([0.5]), np.array([20.0]), np.array([0.1])
    out["cavity64_full_model_probe"] = (q, [(5e-4, 16, True), (1e-3, 32, False)], 8)
    return out


def run(p, phases, record_every):
    psi = p["psi0"].astype(np.complex128).copy()
    o = Oracle(p)
    recs = []
    for dt, n, imag in phases:
        r = o.evolve(psi, dt, n, imag, record_every=record_every)
        if r is not None:
            recs.append(r)
    ob = o.observables(psi)[0][0]
    res = {k: float(ob[k]) for k in ("norm", "e_kin", "e_pot", "e_int", "e_cav", "theta", "re_alpha", "im_alpha")}
    idx = np.arange(psi.size, dtype=np.float64).reshape(psi.shape)
    res["psi_checksum"] = [float(np.sum(psi.real * np.cos(0.37 * idx))), float(np.sum(psi.imag * np.sin(0.11 * idx))),
                           float(np.sum(np.abs(psi) ** 4))]
    if recs:
        res["records"] = np.concatenate(recs)[:, 0, :].tolist()
    return res


def main():
    data = {name: run(*c) for name, c in cases().items()}
    with open(OUT, "w") as f:
        json.dump(data, f, indent=1, sort_keys=True)
    print("wrote", OUT)


if __name__ == "__main__":
    main()
