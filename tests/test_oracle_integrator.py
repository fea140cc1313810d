"""Pins of the oracle's 4th-order symplectic step (eq.(4) and the 12-step listing)
against what the paper and the mathematics fix: Yoshida's order conditions (ref. [33]),
the O(dt^5) local error ("+ O(dt^5)") seen as a 16x drop of the energy error per
halving of dt, time reversibility ("The approximation in eq. (4) is time reversible",
PAPER.md:52), the exact conservation laws of the composition (momentum, 2D angular momentum),
closed-form two-body motion (pendulum period 4K(k); circular orbit), and force reuse
(reading G3: 3n+1 force evaluations).
"""
import math

import numpy as np
import pytest
from scipy.special import ellipk

HMF, RING, GRAV2D = 0, 1, 2


def _state(model, N, seed):
    rng = np.random.default_rng(seed)
    if model == GRAV2D:
        u1, u2 = rng.random(N), rng.random(N)
        r, ph = np.sqrt(u1), 2 * math.pi * u2
        px, py = 0.1 * rng.standard_normal(N), 0.1 * rng.standard_normal(N)
        return r * np.cos(ph), r * np.sin(ph), px - px.mean(), py - py.mean()
    th = rng.uniform(-1.5, 1.5, N)
    p = rng.uniform(-0.5, 0.5, N)
    return th, None, p, None


def _energy(ref, model, eps, s):
    e, _ = ref.energy(model, eps, s[0], s[1], s[2], s[3], form=0)
    return e[0] + e[1]


def test_yoshida_coefficients_satisfy_order_conditions(ref):
    """Reading G4.  Triple-jump weights w1, w0, w1 must satisfy 2 w1 + w0 = 1 (consistency) and
    2 w1^3 + w0^3 = 0 (cancels the dt^3 error term of the leapfrog) - Yoshida 1990, ref. [33];
    eq.(4)'s arrangement gives D0 = w1, D1 = w0, B0 = w1/2, B1 = (w0 + w1)/2."""
    B0, B1, D0, D1 = ref.coefficients()
    assert abs(2 * D0 + D1 - 1) < 1e-15 and abs(2 * B0 + 2 * B1 - 1) < 1e-15
    assert abs(2 * D0 ** 3 + D1 ** 3) < 1e-14
    assert abs(B0 - D0 / 2) < 1e-16 and abs(B1 - (D0 + D1) / 2) < 1e-16
    assert B1 < 0 and D1 < 0 and B0 > 0 and D0 > 0
    # printed to 16 digits in SURVEY.md section 8
    assert abs(B0 - 0.6756035959798289) < 1e-15 and abs(D1 + 1.7024143839193153) < 1e-15


@pytest.mark.parametrize("model,eps,N,dt0", [(HMF, 0.0, 64, 0.1), (GRAV2D, 1e-3, 128, 0.02), (RING, 0.01, 64, 0.02)])
def test_fourth_order_energy_error_scaling(ref, model, eps, N, dt0):
    """Global error of a 4th-order scheme ~ dt^4: max relative energy error over a fixed time
    falls ~16x per halving of dt.  (With listing step 11 read literally - f^(I) - the ratio is 2;
    with eq.(8)'s printed sign the Ring error does not fall at all: readings G1, G2.)"""
    T = 2.0 if model != RING else 1.0
    errs = []
    for k in range(4):
        dt = dt0 / 2 ** k
        s = list(_state(model, N, 100 + model))
        E0 = _energy(ref, model, eps, s)
        f0 = f1 = None
        nsteps = int(round(T / dt))
        worst = 0.0
        chunk = max(1, nsteps // 16)
        done = 0
        valid = False
        while done < nsteps:
            n = min(chunk, nsteps - done)
            f0, f1 = ref.step(model, eps, s[0], s[1], s[2], s[3], n, dt, f0, f1, force_valid=valid, form=1)
            valid = True
            done += n
            worst = max(worst, abs((_energy(ref, model, eps, s) - E0) / E0))
        errs.append(worst)
    ratios = [errs[i] / errs[i + 1] for i in range(3)]
    assert all(10.0 < r < 26.0 for r in ratios[1:]), (errs, ratios)
    assert errs[-1] < errs[0] / 1000


@pytest.mark.parametrize("model,eps", [(HMF, 0.0), (RING, 0.01), (GRAV2D, 1e-3)])
def test_time_reversibility(ref, model, eps):
    """Integrate, flip p, integrate back (equivalently: integrate with -dt) -> start, to rounding."""
    N = 64
    s = list(_state(model, N, 5))
    s0 = [None if a is None else a.copy() for a in s]
    ref.step(model, eps, s[0], s[1], s[2], s[3], 100, 0.01, form=1)
    moved = np.max(np.abs(s[0] - s0[0]))
    assert moved > 1e-2
    for k in (2, 3):
        if s[k] is not None:
            s[k] *= -1.0
    ref.step(model, eps, s[0], s[1], s[2], s[3], 100, 0.01, form=1)
    for k in (2, 3):
        if s[k] is not None:
            s[k] *= -1.0
    for a, b in zip(s, s0):
        if a is not None:
            assert np.max(np.abs(a - b)) < 1e-11
    # negative dt is the same thing
    t = [None if a is None else a.copy() for a in s0]
    ref.step(model, eps, t[0], t[1], t[2], t[3], 50, 0.01, form=1)
    ref.step(model, eps, t[0], t[1], t[2], t[3], 50, -0.01, form=1)
    for a, b in zip(t, s0):
        if a is not None:
            assert np.max(np.abs(a - b)) < 1e-11


@pytest.mark.parametrize("model,eps", [(HMF, 0.0), (RING, 0.01), (GRAV2D, 1e-3)])
def test_momentum_and_angular_momentum_conservation(ref, model, eps):
    N = 100
    s = list(_state(model, N, 8))
    P0 = math.fsum(s[2])
    L0 = math.fsum(s[0] * s[3] - s[1] * s[2]) if model == GRAV2D else 0.0
    ref.step(model, eps, s[0], s[1], s[2], s[3], 200, 0.01, form=1)
    scale = math.fsum(np.abs(s[2]))
    assert abs(math.fsum(s[2]) - P0) < 1e-13 * scale
    if model == GRAV2D:
        assert abs(math.fsum(s[3])) < 1e-13 * scale
        assert abs(math.fsum(s[0] * s[3] - s[1] * s[2]) - L0) < 1e-13 * scale


def test_hmf_two_body_pendulum_period(ref):
    """N = 2 HMF: phi = th1 - th2 obeys phi'' = -sin phi; released at rest from phi0 it returns
    after T = 4 K(k), k = sin(phi0/2) (phi0 = 1 -> T = 6.69997566437...)."""
    phi0 = 1.0
    T = 4 * ellipk(math.sin(phi0 / 2) ** 2)
    assert abs(T - 6.6999756643704527) < 1e-12
    n = 2000
    th = np.array([0.5 * phi0, -0.5 * phi0]); p = np.zeros(2)
    ref.step(HMF, 0.0, th, None, p, None, n, T / n)
    assert abs((th[0] - th[1]) - phi0) < 1e-10 and np.max(np.abs(p)) < 1e-9
    # half period: mirror image
    th = np.array([0.5 * phi0, -0.5 * phi0]); p = np.zeros(2)
    ref.step(HMF, 0.0, th, None, p, None, n // 2, T / n)
    assert abs((th[0] - th[1]) + phi0) < 1e-10


def test_grav2d_two_body_circular_orbit(ref):
    """N = 2, separation R: relative acceleration = -2 r/(r^2 + eps) => circular orbit with
    omega^2 = 2/(R^2 + eps); after one period both bodies are back."""
    R, eps = 0.8, 1e-3
    w = math.sqrt(2.0 / (R * R + eps))
    x = np.array([R / 2, -R / 2]); y = np.zeros(2)
    px = np.zeros(2); py = np.array([w * R / 2, -w * R / 2])
    n = 2000
    ref.step(GRAV2D, eps, x, y, px, py, n, (2 * math.pi / w) / n)
    assert np.max(np.abs(x - np.array([R / 2, -R / 2]))) < 1e-9 and np.max(np.abs(y)) < 1e-9
    # quarter period: rotated by 90 degrees
    x = np.array([R / 2, -R / 2]); y = np.zeros(2)
    px = np.zeros(2); py = np.array([w * R / 2, -w * R / 2])
    ref.step(GRAV2D, eps, x, y, px, py, n // 4, (2 * math.pi / w) / n)
    assert np.max(np.abs(y - np.array([R / 2, -R / 2]))) < 1e-9 and np.max(np.abs(x)) < 1e-9


def test_free_drift_and_listing_structure(ref):
    """With a single particle the force is zero: one step is a pure drift q += (2 D0 + D1) dt p = dt p.
    With forces: n steps in one call == n calls of one step reusing the force (reading G3),
    bit for bit; and the returned force is f(q(t + n dt))."""
    th = np.array([0.3]); p = np.array([0.7])
    ref.step(HMF, 0.0, th, None, p, None, 10, 0.1)
    assert abs(th[0] - (0.3 + 0.7)) < 1e-15 and p[0] == 0.7
    s = list(_state(RING, 50, 12))
    t = [None if a is None else a.copy() for a in s]
    fa, _ = ref.step(RING, 0.01, s[0], None, s[2], None, 5, 0.01, form=1)
    fb = None
    for k in range(5):
        fb, _ = ref.step(RING, 0.01, t[0], None, t[2], None, 1, 0.01, fb, None, force_valid=(k > 0), form=1)
    assert np.array_equal(s[0], t[0]) and np.array_equal(s[2], t[2]) and np.array_equal(fa, fb)
    assert np.array_equal(fa, ref.forces(RING, 0.01, s[0], form=1))


def test_one_step_matches_listing_written_out(ref):
    """The 12-step listing (readings G2/G3) written out with numpy for HMF N = 3,
    forces taken from the (separately pinned) oracle force routine."""
    B0, B1, D0, D1 = ref.coefficients()
    dt = 0.07
    r = np.array([0.1, -0.9, 1.4]); p = np.array([0.3, -0.2, 0.05])
    F = lambda q: ref.forces(HMF, 0.0, q)
    f1 = F(r)                                   # 1
    p1 = p + B0 * dt * f1; r1 = r + D0 * dt * p1          # 2, 3
    f2 = F(r1)                                  # 4
    p2 = p1 + B1 * dt * f2; r2 = r1 + D1 * dt * p2        # 5, 6
    f3 = F(r2)                                  # 7
    p3 = p2 + B1 * dt * f3; r3 = r2 + D0 * dt * p3        # 8, 9
    f4 = F(r3)                                  # 10
    p4 = p3 + B0 * dt * f4                      # 11 (G2)
    q = r.copy(); pp = p.copy()
    ref.step(HMF, 0.0, q, None, pp, None, 1, dt)
    assert np.max(np.abs(q - r3)) < 1e-15 and np.max(np.abs(pp - p4)) < 1e-15
