"""Writes the cached oracle checkpoints of BASELINE.json's configs 3, 4 and 5 at their FULL sizes
("the oracle's outputs cached on disk keyed by (config, seed), checkpointed
parity"), which tests/test_gpu_fullsize.py compares the CUDA path against.

Calls ONLY oracle/ and workloads/ (never the CUDA package): every stored value is the oracle's.

    python tests/golden/make_fullsize_cache.py --only c3,c3_floor [--out DIR] [--threads N]

Items (one .npz each under tests/golden/fullsize/, keyed by config, input dtype and seed):
  c3        config 3: 1024^2, complex64 input, imaginary time dt=5e-4 x 5000, seed 7
  c4_c64    config 4: 2048^2, complex64 input (the fp32-rounded psi0, up-cast), real time dt=1e-4 x 10000
  c4_c128   config 4: 2048^2, complex128 input, same run
  c5        config 5: 64 x 512^2, complex64 input, imaginary time dt=5e-4 x 3000 -- the oracle runs EIGHT of the 64
            members (C5_MEMBERS: the four corners of the (V_p, Delta) sweep and four points of its diagonal; members
            never interact, so member b of the batch is the single-grid run with its parameters); the GPU test runs
            all 64 and compares these eight
  <item>_floor   the same run with the oracle's statements compiled in complex64 (-DREAL=float): the
            fp32 round-off floor OF THE METHOD, never used as a reference.
            Needs <item>.npz (it stores its distance to it).

What is stored per checkpoint (cumulative step count c):
  psi_<c>   the oracle's wavefunction on the sample lattice [:, ::stride, ::stride] (complex64 for a
            complex64-input run -- rounding the reference adds 6e-8 relative, three orders below the
            tightest bar it is used for -- complex128 for the complex128-input run)
  obs_<c>   [batch][8] the oracle's observables on the FULL grid (norm, e_kin, e_pot, e_int, e_cav,
            theta, re_alpha, im_alpha): every grid point enters these
  records   [n_rec][batch][6] every record of the run (config 4: the order parameter every 100 steps)
A 2048^2 complex128 array is 64 MiB, so whole checkpoints cannot live in the repository; the sample
lattice is an unbiased estimator of the relative L2 error and the full-grid sums catch anything local.
"""
from __future__ import annotations

import argparse
import hashlib
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import workloads as W                                  # noqa: E402
from oracle.gpe_oracle import Oracle, OBS_NAMES        # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
CACHE = os.path.join(HERE, "fullsize")

C5_MEMBERS = (0, 7, 18, 27, 36, 45, 56, 63)   # member index 8 b + a: V_p = 20 a / 7, Delta = -3 + 2.8 b / 7

ITEMS = {
    # name: (workload factory, input dtype, mode, dt, checkpoints, record_every, sample stride)
    "c3": (lambda: W.config3(), "c64", "imag", 5e-4, (1, 10, 100, 1000, 5000), 100, 4),
    "c4_c64": (lambda: W.config4(), "c64", "real", 1e-4, (1, 10, 100, 1000, 5000, 10000), 100, 8),
    "c4_c128": (lambda: W.config4(dtype="c128"), "c128", "real", 1e-4, (1, 100, 1000, 10000), 100, 8),
    "c5": (lambda: W.select_members(W.config5(), C5_MEMBERS), "c64", "imag", 5e-4, (1, 100, 1000, 3000), 500, 8),
}


def oracle_input(psi0: np.ndarray, dtype: str) -> np.ndarray:
    """The values the CUDA path receives: for a complex64 run the fp32-rounded array, up-cast."""
    cd = np.complex64 if dtype == "c64" else np.complex128
    return np.ascontiguousarray(psi0.astype(cd).astype(np.complex128))


def sample(psi: np.ndarray, stride: int) -> np.ndarray:
    return np.ascontiguousarray(psi[..., ::stride, ::stride])


def rel(a: np.ndarray, b: np.ndarray) -> float:
    a = np.asarray(a, dtype=np.complex128).ravel()
    b = np.asarray(b, dtype=np.complex128).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def obs_array(o: Oracle, psi: np.ndarray) -> np.ndarray:
    return np.array([[ob[k] for k in OBS_NAMES] for ob in o.observables(psi)[0]], dtype=np.float64)


def oracle_sha() -> str:
    with open(os.path.join(ROOT, "oracle", "gpe_oracle.c"), "rb") as f:
        return hashlib.sha256(f.read()).hexdigest()[:16]


def run_item(name: str, out_dir: str, scale: int = 1) -> str:
    floor = name.endswith("_floor")
    base = name[:-6] if floor else name
    make, dtype, mode, dt, checkpoints, record_every, stride = ITEMS[base]
    if scale > 1:   # smoke run of the generator itself (not a cache anyone reads)
        checkpoints = tuple(sorted({max(1, c // scale) for c in checkpoints}))
        record_every = max(1, record_every // scale)
    p = make()
    imag = mode == "imag"
    ref_file = os.path.join(out_dir, base + ".npz")
    out = {"members": np.array(C5_MEMBERS if base == "c5" else range(p.get("batch", 1)), dtype=np.int64),
           "stride": np.int64(stride), "steps": np.array(checkpoints, dtype=np.int64), "dt": np.float64(dt),
           "imag": np.int64(imag), "record_every": np.int64(record_every),
           "oracle_sha16": np.array(oracle_sha()), "item": np.array(name)}
    if floor:
        ref = np.load(ref_file)
        assert [int(c) for c in ref["steps"]] == list(checkpoints), "reference cache has other checkpoints"
        psi = np.ascontiguousarray(p["psi0"].astype(np.complex64))
        o = Oracle(p, "f32")
    else:
        psi = oracle_input(p["psi0"], dtype)
        o = Oracle(p)
    recs = []
    done = 0
    t0 = time.perf_counter()
    for c in checkpoints:
        r = o.evolve(psi, dt, c - done, imag, record_every=record_every)
        if r is not None and len(r):
            recs.append(r)
        done = c
        ob = obs_array(o, psi)
        if floor:
            out[f"floor_rel_{c}"] = np.float64(rel(sample(psi, stride), ref[f"psi_{c}"]))
            out[f"floor_obs_{c}"] = ob
        else:
            s = sample(psi, stride)
            out[f"psi_{c}"] = s.astype(np.complex64) if dtype == "c64" else s
            out[f"obs_{c}"] = ob
        print(f"[{name}] step {c}: theta[0] = {ob[0, 5]:+.10e}  E[0] = {ob[0, 1:5].sum():.10e}  "
              f"({time.perf_counter() - t0:.0f} s)", flush=True)
    out["floor_records" if floor else "records"] = (np.concatenate(recs) if recs
                                                    else np.zeros((0, p.get("batch", 1), 6)))
    os.makedirs(out_dir, exist_ok=True)
    path = os.path.join(out_dir, name + ".npz")
    tmp = path + ".tmp.npz"
    np.savez(tmp, **out)
    os.replace(tmp, path)
    return path


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--only", default=",".join(list(ITEMS) + [k + "_floor" for k in ITEMS if k != "c4_c128"]))
    ap.add_argument("--out", default=CACHE)
    ap.add_argument("--scale", type=int, default=1, help="divide the step counts (generator smoke test only)")
    ap.add_argument("--skip-existing", action="store_true")
    a = ap.parse_args()
    for name in a.only.split(","):
        if a.skip_existing and os.path.exists(os.path.join(a.out, name + ".npz")):
            print(f"[{name}] exists, skipped", flush=True)
            continue
        t0 = time.perf_counter()
        path = run_item(name, a.out, a.scale)
        print(f"[{name}] wrote {path} ({os.path.getsize(path) / 1e6:.2f} MB) in {time.perf_counter() - t0:.0f} s",
              flush=True)


if __name__ == "__main__":
    main()
