"""Full-size parity report (not collected by pytest): runs BASELINE.json's configs at their full grid
sizes on the GPU through the C ABI and on the CPU oracle, checkpoint by checkpoint, and prints a
markdown table: relative L2 error of psi, error of the order parameter Theta, and -- for complex64 --
the method's own fp32 floor (the oracle's statements in complex64 against complex128 on the same
input) next to them.

    python tests/full_size_report.py [--quick] [--only 3,4c64] > gpurun_out/full_size_parity.md

Needs a B200 and the host cores for the oracle (about an hour without --quick).
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import workloads as W                      # noqa: E402
from oracle.gpe_oracle import Oracle       # noqa: E402


def rel(a, b):
    return float(np.linalg.norm(a.astype(np.complex128).ravel() - b.ravel()) / np.linalg.norm(b.ravel()))


def run(name, p, dtype, mode, dt, checkpoints, floor=True):
    """Evolve GPU, oracle (complex128) and, for complex64, the fp32 build of the oracle from the same
    input; compare at every checkpoint (cumulative step counts)."""
    import torch
    import paper_2404_14401_b200 as G
    cd = np.complex64 if dtype == "c64" else np.complex128
    plan = G.Plan(p["nx"], p["ny"], p["Lx"], p["Ly"], dtype, p.get("batch", 1))
    plan.set_potential(p)
    psi = torch.from_numpy(np.ascontiguousarray(p["psi0"].astype(cd))).cuda()
    ref = np.ascontiguousarray(p["psi0"].astype(cd).astype(np.complex128))
    o = Oracle(p)
    fl = of = None
    if floor and dtype == "c64":
        fl = np.ascontiguousarray(p["psi0"].astype(np.complex64))
        of = Oracle(p, "f32")
    imag = mode == "imag"
    done = 0
    for c in checkpoints:
        n = c - done
        t0 = time.perf_counter()
        plan.evolve(psi, dt, n, mode)
        torch.cuda.synchronize()
        tg = time.perf_counter() - t0
        t0 = time.perf_counter()
        o.evolve(ref, dt, n, imag)
        to = time.perf_counter() - t0
        if of is not None:
            of.evolve(fl, dt, n, imag)
        done = c
        got = psi.cpu().numpy()
        og, oo = plan.observables(psi)[0], o.observables(ref)[0]
        th_g = np.array([x["theta"] for x in og]); th_o = np.array([x["theta"] for x in oo])
        e_g = np.array([x["e_kin"] + x["e_pot"] + x["e_int"] + x["e_cav"] for x in og])
        e_o = np.array([x["e_kin"] + x["e_pot"] + x["e_int"] + x["e_cav"] for x in oo])
        row = [name, dtype, mode, str(c), f"{rel(got, ref):.2e}"]
        row.append(f"{rel(fl, ref):.2e}" if of is not None else "—")
        k = int(np.argmax(np.abs(th_g - th_o)))
        row.append(f"{abs(th_g[k] - th_o[k]):.2e} (Theta = {th_o[k]:+.4e})")
        if of is not None:
            th_f = np.array([x["theta"] for x in of.observables(fl)[0]])
            row.append(f"{np.max(np.abs(th_f - th_o)):.2e}")
        else:
            row.append("—")
        row.append(f"{np.max(np.abs(e_g - e_o) / np.abs(e_o)):.2e}")
        row.append(f"{tg:.2f} / {to:.1f}")
        print("| " + " | ".join(row) + " |", flush=True)
    plan.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--quick", action="store_true", help="a tenth of the steps")
    ap.add_argument("--only", default="1,2,3,5,4c128,4c64", help="comma-separated subset of 1,2,3,5,4c128,4c64")
    a = ap.parse_args()
    s = 10 if a.quick else 1
    only = set(a.only.split(","))
    print("| config | dtype | mode | steps | rel L2 err of psi (GPU vs oracle) | fp32 floor of the method | max abs err of Theta | "
          "fp32 floor of Theta | max rel err of the energy | wall s GPU / oracle |")
    print("|---|---|---|---|---|---|---|---|---|---|", flush=True)
    if "1" in only:
        for g in (0.0, 10.0):
            run(f"1 (g={g:g})", W.config1(g=g), "c128", "imag", 1e-3, [1, 2000 // s])
    if "2" in only:
        for dtype in ("c64", "c128"):
            p = W.config2(V0=10.0, dtype=dtype)
            p["sched_step"], p["sched_amp"] = None, None           # the ground-state phase has no lattice
            run("2 ground state", p, dtype, "imag", 1e-3, [1, 1000 // s, 5000 // s])
    if "3" in only:
        p = W.config3()
        run("3", p, "c64", "imag", 5e-4, [1, 10, 100, 1000 // s, 5000 // s] if s == 1 else [1, 10, 100, 500])
    if "5" in only:
        p = W.config5(n_steps=1)
        run("5 (64 x 512^2)", p, "c64", "imag", 5e-4, [1, 100, 1000 // s])
    if "4c128" in only:
        p = W.config4(dtype="c128")
        run("4", p, "c128", "real", 1e-4, [1, 100, 1000 // s])
    if "4c64" in only:
        p = W.config4()
        run("4", p, "c64", "real", 1e-4, [1, 10, 100, 1000, 5000, 10000] if s == 1 else [1, 10, 100, 1000])

if __name__ == "__main__":
    main()
