#!/usr/bin/env python
"""Writes the stored full-size oracle results under tests/golden/ (SURVEY.md 8(d) "Oracle timing": run the full
oracle once and keep its output keyed by a hash of inputs + oracle source).

    python tests/golden/make_golden.py config3 [config4 config5 ...]      (CPU only; minutes to hours)

Calls ONLY oracle/ (its bit-identical blocked loop arrangement, dos_oracle_blocked.c) and the seeded input
generators. Nothing here touches the CUDA path; no stored value comes from it.

What is stored per case (float32 unless noted), tests/golden/<case>.npz:
    key            sha256 over every input array / scalar of the problem and the text of oracle/*.c
    cells          int64 [Ns]   seeded sample of voxels: half drawn among voxels inside the beam, half uniform
    phi_u, phi_c, phi_c_abs, phi_total   [G][Ns] at those voxels (phi_c_abs = sum_n w_n |psi_n|, reading R15b)
    peak_*         [G] float64  max |field| over ALL voxels (the 1e-6-of-peak threshold of the parity measure)
    dose_cells     int64 [Nd], dose [Nd], dose_peak    a larger seeded uniform sample of the dose map
The relative L2 error of a parity test is then taken over the sample (a seeded uniform subset estimates the
all-voxel ratio of mean squares without bias); max-rel uses the true peaks.
"""
from __future__ import annotations

import hashlib
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

# case -> (config, make_problem overrides, source index, text)
CASES = {
    "config3": ("config3", {}, 0, "config 3 in full: 128x128x64, 19 groups x 20 iterations, S16/P5"),
    "config4_pos5": ("config4", {}, 5, "config 4, source position 5 of 36 in full: 256x256x64, 19 groups x 15 iterations, S8/P3"),
    "config5_top6": ("config5", {"top_groups": 6}, 0,
                     "config 5 mesh (256^3, S16/P5), the 6 highest-energy groups of its 19 x 20 iterations"),
    "config5_top3x6": ("config5", {"top_groups": 3, "n_iter": 6}, 0,
                       "config 5 mesh (256^3, S16/P5), the 3 highest-energy groups x 6 iterations"),
    # small case of the same machinery, run by the CPU test suite in seconds
    "selftest": ("config3", dict(nx=26, ny=20, nz=9, voxel=1.5, n_group=4, n_iter=3), 0, "reduced config 3 (self-test of this script)"),
}
N_SAMPLE = 10240
N_DOSE = 262144


def problem_key(p, source_index):
    import oracle
    h = hashlib.sha256()
    for path in oracle.source_files():
        with open(path, "rb") as f:
            h.update(f.read())
    for k in ("material", "sigma_t", "sigma_s", "kerma", "spectrum"):
        a = np.ascontiguousarray(p[k])
        h.update(k.encode()); h.update(str(a.dtype).encode()); h.update(str(a.shape).encode()); h.update(a.tobytes())
    for k in ("mu", "eta", "xi", "w"):
        h.update(np.ascontiguousarray(p["quadrature"][k]).tobytes())
    h.update(json.dumps({"mesh": p["mesh"], "P_L": p["P_L"], "n_iter": p["n_iter"], "n_group": p["n_group"],
                         "source": p["sources"][source_index]}, sort_keys=True).encode())
    return h.hexdigest()


def sample_cells(phi_u0, seed):
    """Half of the sample among voxels inside the beam (phi_u > 0), half uniform over the mesh; sorted, unique."""
    rng = np.random.default_rng(seed)
    flat = np.asarray(phi_u0).reshape(-1)
    inside = np.flatnonzero(flat > 0)
    a = rng.choice(inside, min(N_SAMPLE // 2, inside.size), replace=False)
    b = rng.choice(flat.size, min(N_SAMPLE - a.size, flat.size), replace=False)
    return np.unique(np.concatenate([a, b])).astype(np.int64)


def make(case, out_dir=HERE):
    import oracle
    from paper_1811_12391_b200.inputs import make_problem
    config, ov, sidx, text = CASES[case]
    p = make_problem(config, **ov)
    key = problem_key(p, sidx)
    t0 = time.time()
    r = oracle.run_problem(p, source_index=sidx, blocked=True)
    secs = time.time() - t0
    G = p["n_group"]
    cells = sample_cells(r["phi_u"][0], seed=1234 + sum(map(ord, case)))
    nv = r["dose"].size
    dcells = np.sort(np.random.default_rng(99).choice(nv, min(N_DOSE, nv), replace=False)).astype(np.int64)
    out = {"key": np.array(key), "cells": cells, "dose_cells": dcells,
           "dose": r["dose"].reshape(-1)[dcells].astype(np.float32), "dose_peak": np.array(np.abs(r["dose"]).max())}
    for f in ("phi_u", "phi_c", "phi_c_abs", "phi_total"):
        a = np.asarray(r[f]).reshape(G, -1)
        out[f] = a[:, cells].astype(np.float32)
        out["peak_" + f] = np.abs(a).max(axis=1)
    out["meta"] = np.array(json.dumps({"case": case, "config": config, "overrides": ov, "source_index": sidx, "text": text,
                                       "oracle_seconds": round(secs, 1), "threads": os.cpu_count(),
                                       "variant": "dos_oracle_blocked.c (bit-identical to dos_oracle.c: test_blocked_variant_is_bit_identical)"}))
    path = os.path.join(out_dir, case + ".npz")
    np.savez_compressed(path, **out)
    print(f"{case}: {secs:.0f} s of oracle, {os.path.getsize(path) / 1e6:.2f} MB -> {path}", flush=True)
    return path


if __name__ == "__main__":
    for c in sys.argv[1:] or ["selftest"]:
        make(c)
