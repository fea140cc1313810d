"""Writes tests/golden/oracle_small.json: forces, energies and a 10-step trajectory of three tiny
seeded cases, computed by the ORACLE ONLY (oracle/ref.py -> oracle/lrmd_ref.cpp).

    python tests/golden/make_golden.py

The paper prints no worked numerical example (its figures are absent from the reference
and its tables are timings), so there is no paper value to store; what pins the oracle itself are the
mathematical checks in tests/test_oracle_*.py (mpmath gradients of the printed Hamiltonians, closed
forms, invariants).  This file freezes the pinned oracle's output on fixed inputs so that
  * a later change to the oracle's arithmetic shows up as a diff of stored numbers (regression), and
  * the CUDA path is also compared with stored values written by the oracle alone (tests/test_golden.py); they were
    committed after the first kernels existed, which is harmless: no value in them comes from the CUDA path.
Nothing here imports or calls the CUDA path.  Inputs are written into the file (hex floats, exact).
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import ref  # noqa: E402

HMF, RING, GRAV2D = 0, 1, 2
CASES = [("hmf_n37", HMF, 37, 0.0, 0.05), ("ring_n41", RING, 41, 0.01, 0.01), ("grav2d_n29", GRAV2D, 29, 1e-3, 0.005)]


def hexlist(a):
    return [float(v).hex() for v in np.asarray(a, dtype=np.float64)]


def state(model, N, seed):
    rng = np.random.default_rng(seed)
    if model == GRAV2D:
        r, ph = np.sqrt(rng.random(N)), 2 * np.pi * rng.random(N)
        px, py = 0.1 * rng.standard_normal(N), 0.1 * rng.standard_normal(N)
        return [r * np.cos(ph), r * np.sin(ph), px - px.mean(), py - py.mean()]
    a = 1.5 if model == HMF else 1.0
    return [rng.uniform(-a, a, N), rng.uniform(-0.5, 0.5, N)]


def main():
    out = {"written_by": "tests/golden/make_golden.py (oracle only)", "cases": {}}
    for k, (name, model, N, eps, dt) in enumerate(CASES):
        st = state(model, N, 20121202 + k)
        two = model == GRAV2D
        q0, q1 = (st[0], st[1]) if two else (st[0], None)
        p0, p1 = (st[2], st[3]) if two else (st[1], None)
        f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=0, nthreads=1)
        e, eabs = ref.energy(model, eps, q0, q1, p0, p1, nthreads=1)
        fin = [a.copy() for a in st]
        fq0, fq1 = (fin[0], fin[1]) if two else (fin[0], None)
        fp0, fp1 = (fin[2], fin[3]) if two else (fin[1], None)
        ref.step(model, eps, fq0, fq1, fp0, fp1, 10, dt, form=0, nthreads=1)
        e10, _ = ref.energy(model, eps, fq0, fq1, fp0, fp1, nthreads=1)
        out["cases"][name] = {
            "model": model, "N": N, "eps": eps, "dt": dt, "steps": 10,
            "state0": [hexlist(a) for a in st],
            "forces": [hexlist(f0)] + ([hexlist(f1)] if two else []),
            "abs_force_sums": [hexlist(A0)] + ([hexlist(A1)] if two else []),
            "energy0": hexlist(e), "energy0_abs": hexlist(eabs),
            "state10": [hexlist(a) for a in fin], "energy10": hexlist(e10),
        }
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_small.json")
    with open(path, "w") as fh:
        json.dump(out, fh, indent=0)
    print("wrote", path)


if __name__ == "__main__":
    main()
