"""Paper-shaped runs: the initial conditions of the paper's section 4 and Figs. 3-6
 advanced on the GPU with K(t), V(t) and the relative energy error
|(E - E0)/E0| recorded through ``lrmd_step_observe``.

    python -m paper_1212_0262_b200.paper_runs [--model hmf|ring|grav2d|all] [--N N] [--steps S] [--every E]

The paper does not state N for its figures and the images are absent from the reference, so there are
no numbers to match: the runs reproduce the set-up (homogeneous at rest, dt = 0.1 for HMF; eps = 1e-3,
dt = 0.005 for Ring; annulus 1.0 <= r <= 1.5 at rest, eps = 1e-3, dt = 0.005 for 2D gravity) and print
the curves as JSON lines.  All arithmetic of the method runs in the CUDA kernels behind the C ABI.
"""
from __future__ import annotations

import argparse
import json

from . import inputs, lrmd

SETUPS = {
    "hmf": dict(model=inputs.HMF, eps=0.0, dt=0.1, N=100_000),
    "ring": dict(model=inputs.RING, eps=1e-3, dt=0.005, N=16_384),
    "grav2d": dict(model=inputs.GRAV2D, eps=1e-3, dt=0.005, N=16_384),
}


def initial_state(name: str, N: int, seed: int = 20121203):
    if name == "grav2d":
        return inputs.annulus_at_rest(N, 1.0, 1.5, seed)
    return inputs.homogeneous_at_rest(N, seed)


def run(name: str, N: int | None = None, steps: int = 200, every: int = 10, device="cuda:0"):
    """Returns {"t": [...], "K": [...], "V": [...], "energy_error": [...]} (host lists)."""
    su = SETUPS[name]
    N = int(N or su["N"])
    ctx = lrmd.Context(su["model"], N, su["eps"], device=device)
    ctx.set_state(*initial_state(name, N))
    rec = ctx.step_observe(steps, su["dt"], every).cpu().numpy()
    ctx.close()
    E = rec[:, 0] + rec[:, 1]
    # E0 can be ~0 only for a degenerate input; the paper's error is |(E - E0)/E0|
    err = abs((E - E[0]) / E[0])
    return {"run": name, "N": N, "eps": su["eps"], "dt": su["dt"], "t": [su["dt"] * every * k for k in range(len(E))],
            "K": rec[:, 0].tolist(), "V": rec[:, 1].tolist(), "a": rec[:, 2].tolist(), "b": rec[:, 3].tolist(),
            "energy_error": err.tolist()}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--model", default="all", choices=["all", *SETUPS])
    ap.add_argument("--N", type=int, default=None)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--every", type=int, default=10)
    args = ap.parse_args()
    for name in (SETUPS if args.model == "all" else [args.model]):
        print(json.dumps(run(name, args.N, args.steps, args.every)))


if __name__ == "__main__":
    main()
