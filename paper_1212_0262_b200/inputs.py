"""Seeded synthetic initial conditions (numpy only, fp64).

This module is the ONLY code shared by the CUDA path and the oracle: it draws
the initial positions and momenta and holds none of the method's arithmetic
(no forces, no energies, no integrator).  The same host arrays go to both
sides bit-identically.

The paper measures on no public dataset: its workloads are synthetic initial
conditions (section 4).  The five workloads below take the
shapes BASELINE.json's ``configs`` state; the draw order and seeds follow
SURVEY.md section 8(d): ``numpy.random.default_rng(12120262 + k)``.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

HMF, RING, GRAV2D = 0, 1, 2
MODEL_NAMES = {HMF: "hmf", RING: "ring", GRAV2D: "grav2d"}

SEED_BASE = 12120262


def waterbag(N: int, theta_half_width: float, p_half_width: float, seed: int):
    """theta ~ U[-a, a), p ~ U[-b, b) (waterbag; BASELINE.json configs 1, 2, 4).

    Draw order: all N angles first, then all N momenta.
    """
    rng = np.random.default_rng(seed)
    a, b = float(theta_half_width), float(p_half_width)
    theta = -a + (2.0 * a) * rng.random(N)
    p = -b + (2.0 * b) * rng.random(N)
    return theta, p


def disk2d(N: int, sigma_p: float, seed: int):
    """Positions uniform in the unit disk, momenta N(0, sigma_p^2) with the mean
    removed (BASELINE.json configs 3, 5).

    Draw order: U1[N], U2[N], then N(0,1)[N] for px and N(0,1)[N] for py.
    r = sqrt(U1), phi = 2 pi U2 (no rejection); the mean of each momentum
    component is an exactly rounded sum (math.fsum) divided by N.
    """
    rng = np.random.default_rng(seed)
    u1 = rng.random(N)
    u2 = rng.random(N)
    r = np.sqrt(u1)
    phi = (2.0 * math.pi) * u2
    x = r * np.cos(phi)
    y = r * np.sin(phi)
    px = sigma_p * rng.standard_normal(N)
    py = sigma_p * rng.standard_normal(N)
    px = px - math.fsum(px) / N
    py = py - math.fsum(py) / N
    return x, y, px, py


def annulus_at_rest(N: int, r1: float, r2: float, seed: int):
    """Paper-shaped 2D input: uniform on the shell r1 <= r <= r2, at rest
    (section 4)."""
    rng = np.random.default_rng(seed)
    u1 = rng.random(N)
    u2 = rng.random(N)
    r = np.sqrt(r1 * r1 + (r2 * r2 - r1 * r1) * u1)
    phi = (2.0 * math.pi) * u2
    return r * np.cos(phi), r * np.sin(phi), np.zeros(N), np.zeros(N)


def homogeneous_at_rest(N: int, seed: int):
    """Paper-shaped HMF/Ring input: theta uniform on [-pi, pi), p = 0
    (section 4)."""
    rng = np.random.default_rng(seed)
    theta = -math.pi + (2.0 * math.pi) * rng.random(N)
    return theta, np.zeros(N)


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config: model, size, parameters and run length."""
    key: str
    k: int          # config number 1..5 (BASELINE.json configs[k-1])
    model: int
    N: int
    eps: float
    dt: float
    steps: int
    theta_hw: float = 0.0
    p_hw: float = 0.0
    sigma_p: float = 0.0

    @property
    def seed(self) -> int:
        return SEED_BASE + self.k

    def state(self, N: int | None = None):
        """Arrays (theta, p) or (x, y, px, py); ``N`` overrides the size for
        reduced-size parity cases with the same distribution."""
        n = self.N if N is None else int(N)
        if self.model == GRAV2D:
            return disk2d(n, self.sigma_p, self.seed)
        return waterbag(n, self.theta_hw, self.p_hw, self.seed)


WORKLOADS = {
    "hmf_1e4": Workload("hmf_1e4", 1, HMF, 10_000, 0.0, 0.05, 1000, theta_hw=1.5, p_hw=0.5),
    "ring_16k": Workload("ring_16k", 2, RING, 16_384, 0.01, 0.01, 100, theta_hw=1.0, p_hw=0.3),
    "grav2d_64k": Workload("grav2d_64k", 3, GRAV2D, 65_536, 1e-3, 0.005, 50, sigma_p=0.1),
    "hmf_5e7": Workload("hmf_5e7", 4, HMF, 50_000_000, 0.0, 0.05, 100, theta_hw=1.5, p_hw=0.5),
    "grav2d_1m": Workload("grav2d_1m", 5, GRAV2D, 1_048_576, 1e-3, 0.005, 5, sigma_p=0.1),
}

# HMF sizes of the paper's Table 1 (N = 1e5 .. 1e8) that are not BASELINE.json configs: same waterbag
# as configs 1 and 4, own seeds.  bench.py reports them beside the configs so that the three HMF regimes of the
# library (cluster-resident, graph replay of the register-prefetch kernel, TMA-staged) each have a measured entry.
TABLE1_WORKLOADS = {
    "hmf_1e5": Workload("hmf_1e5", 6, HMF, 100_000, 0.0, 0.05, 1000, theta_hw=1.5, p_hw=0.5),
    "hmf_1e6": Workload("hmf_1e6", 7, HMF, 1_000_000, 0.0, 0.05, 500, theta_hw=1.5, p_hw=0.5),
    "hmf_1e7": Workload("hmf_1e7", 8, HMF, 10_000_000, 0.0, 0.05, 200, theta_hw=1.5, p_hw=0.5),
}

# Pair-model sizes of the paper's Tables 2 and 3 beyond BASELINE.json's configs: the largest Ring
# run (N = 512,000) and the N = 102,400 rows of both tables; same distributions as configs 2 and 3, own seeds.
TABLE23_WORKLOADS = {
    "ring_102k": Workload("ring_102k", 9, RING, 102_400, 0.01, 0.01, 10, theta_hw=1.0, p_hw=0.3),
    "ring_512k": Workload("ring_512k", 10, RING, 512_000, 0.01, 0.01, 3, theta_hw=1.0, p_hw=0.3),
    "grav2d_102k": Workload("grav2d_102k", 11, GRAV2D, 102_400, 1e-3, 0.005, 10, sigma_p=0.1),
}
# seconds per time step the paper reports on one GK104 of a GTX 690 (Tables 1-3; context only, other hardware)
PAPER_SECONDS_PER_STEP = {"hmf_1e5": 6.3e-4, "hmf_1e6": 4.0e-3, "hmf_1e7": 3.7e-2, "hmf_5e7": 1.81e-1,
                          "ring_102k": 3.9, "ring_512k": 97.5, "grav2d_102k": 0.99}
