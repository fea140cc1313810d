"""Pins of the oracle's forces and energies against what the paper and the mathematics fix.

None of these re-type the oracle's force formulas: forces are pinned to a 50-digit mpmath
*numerical derivative* of the Hamiltonians as printed (eq.(1), eq.(2),
PAPER.md:40 eq.(3)), to closed forms (regular polygon, two bodies, equal/equally-spaced angles),
to the identities the paper states (eqs.(5)-(7), eq.(8) == eq.(9), large-eps Ring -> HMF,
PAPER.md:32), and to invariants (sum_i f_i = 0, 2 pi periodicity).
"""
import math

import mpmath as mp
import numpy as np
import pytest

HMF, RING, GRAV2D = 0, 1, 2


# ---- the Hamiltonians' potential energies exactly as printed, in mpmath ----------------------

def V_mp(model, eps, q0, q1=None):
    N = len(q0)
    s = mp.mpf(0)
    for i in range(N):
        for j in range(i + 1, N):
            if model == HMF:        # eq.(2): +(1/N) sum_{i<j} [1 - cos(ti - tj)]
                s += 1 - mp.cos(q0[i] - q0[j])
            elif model == RING:     # eq.(1): -(1/N) sum_{i<j} 1/(sqrt2 sqrt(1 - cos(ti-tj) + eps))
                s -= 1 / (mp.sqrt(2) * mp.sqrt(1 - mp.cos(q0[i] - q0[j]) + eps))
            else:                   # eq.(3): +(1/N) sum_{i<j} log[(xi-xj)^2 + (yi-yj)^2 + eps]
                s += mp.log((q0[i] - q0[j]) ** 2 + (q1[i] - q1[j]) ** 2 + eps)
    return s / N


def force_mp(model, eps, q0, q1, i, comp=0):
    """-dV/dq_i by mpmath numerical differentiation (no analytic formula typed here)."""
    q0 = [mp.mpf(float(v)) for v in q0]
    q1 = None if q1 is None else [mp.mpf(float(v)) for v in q1]
    eps = mp.mpf(float(eps))

    def fun(z):
        a = list(q0)
        b = None if q1 is None else list(q1)
        if comp == 0:
            a[i] = z
        else:
            b[i] = z
        return V_mp(model, eps, a, b)

    z0 = q0[i] if comp == 0 else q1[i]
    return -mp.diff(fun, z0)


@pytest.fixture(autouse=True)
def _mp_precision():
    old = mp.mp.dps
    mp.mp.dps = 50
    yield
    mp.mp.dps = old


def _rand_state(model, N, seed):
    rng = np.random.default_rng(seed)
    if model == GRAV2D:
        return rng.uniform(-1, 1, N), rng.uniform(-1, 1, N)
    return rng.uniform(-3, 3, N), None


@pytest.mark.parametrize("model,eps,form", [(HMF, 0.0, 0), (HMF, 0.0, 1), (RING, 0.01, 0), (RING, 0.01, 1),
                                            (RING, 1e-3, 1), (GRAV2D, 1e-3, 0), (GRAV2D, 0.0, 0)])
def test_force_is_minus_gradient_of_printed_hamiltonian(ref, model, eps, form):
    """Pins sign (reading G1), prefactors 1/N, 1/(2 sqrt2 N), 2/N, and the exponent 3/2."""
    N = 6
    q0, q1 = _rand_state(model, N, 7 + model)
    f = ref.forces(model, eps, q0, q1, form=form)
    f0, f1 = (f if model == GRAV2D else (f, None))
    for i in range(N):
        e0 = float(force_mp(model, eps, q0, q1, i, 0))
        assert abs(f0[i] - e0) <= 2e-14 * max(1.0, abs(e0)), (i, f0[i], e0)
        if model == GRAV2D:
            e1 = float(force_mp(model, eps, q0, q1, i, 1))
            assert abs(f1[i] - e1) <= 2e-14 * max(1.0, abs(e1))


@pytest.mark.parametrize("model,eps,form", [(HMF, 0.0, 0), (HMF, 0.0, 1), (RING, 0.01, 0), (GRAV2D, 1e-3, 0)])
def test_potential_energy_matches_printed_hamiltonian(ref, model, eps, form):
    N = 7
    q0, q1 = _rand_state(model, N, 11 + model)
    p = np.linspace(-1, 1, N)
    out4, out_abs = ref.energy(model, eps, q0, q1, p, p if model == GRAV2D else None, form=form)
    Vx = float(V_mp(model, mp.mpf(eps), [mp.mpf(float(v)) for v in q0],
                    None if q1 is None else [mp.mpf(float(v)) for v in q1]))
    assert abs(out4[1] - Vx) <= 1e-14 * max(1.0, abs(Vx))
    Kx = 0.5 * math.fsum(float(v) ** 2 for v in p) * (2 if model == GRAV2D else 1)
    assert abs(out4[0] - Kx) <= 1e-15 * Kx
    if model != HMF:   # (a, b) = total momentum
        assert abs(out4[2] - math.fsum(p)) < 1e-15
    assert out_abs[1] >= abs(out4[1]) * (1 - 1e-15)


def test_hmf_pair_sum_equals_mean_field_identity(ref):
    """eqs.(5)-(7): O(N^2) pair sum == O(N) identity, forces and V."""
    rng = np.random.default_rng(3)
    N = 257
    th = rng.uniform(-4, 4, N)
    f_id = ref.forces(HMF, 0.0, th, form=0)
    f_pair, _, A, _ = ref.forces_abs(HMF, 0.0, th, form=1)
    assert np.all(np.abs(f_id - f_pair) <= 1e-14 * A + 1e-17)
    z = np.zeros(N)
    e_id, _ = ref.energy(HMF, 0.0, th, None, z, None, form=0)
    e_pair, ab = ref.energy(HMF, 0.0, th, None, z, None, form=1)
    assert abs(e_id[1] - e_pair[1]) <= 1e-13 * ab[1]
    # (a, b) = (Mx, My), eq.(7)
    assert abs(e_id[2] - math.fsum(np.cos(th)) / N) < 1e-15
    assert abs(e_id[3] - math.fsum(np.sin(th)) / N) < 1e-15


def test_hmf_special_configurations(ref):
    N = 64
    z = np.zeros(N)
    same = np.full(N, 0.83)
    assert np.max(np.abs(ref.forces(HMF, 0.0, same))) < 1e-15          # M = 1 along theta: f = 0
    e, _ = ref.energy(HMF, 0.0, same, None, z, None)
    assert abs(e[1]) < 1e-12 and abs(math.hypot(e[2], e[3]) - 1.0) < 1e-15
    spaced = 2 * math.pi * np.arange(N) / N
    assert np.max(np.abs(ref.forces(HMF, 0.0, spaced))) < 1e-15        # M = 0
    e, _ = ref.energy(HMF, 0.0, spaced, None, z, None)
    assert abs(e[1] - N / 2) < 1e-12 and math.hypot(e[2], e[3]) < 1e-15


def test_ring_direct_form_equals_precomputed_form(ref):
    """eq.(8) == eq.(9)."""
    rng = np.random.default_rng(5)
    N = 300
    th = rng.uniform(-math.pi, math.pi, N)
    for eps in (1e-3, 0.01, 1.0):
        f8, _, A, _ = ref.forces_abs(RING, eps, th, form=0)
        f9 = ref.forces(RING, eps, th, form=1)
        # eq.(9)'s denominator 1 - cc - ss + eps cancels to ~eps for close pairs: relative
        # rounding 2^-53/eps per term in d, x1.5 in d^-3/2
        assert np.all(np.abs(f8 - f9) <= (4e-16 / eps + 4e-16) * 1.5 * A)


def test_ring_equally_spaced_is_force_free(ref):
    N = 48
    th = 2 * math.pi * np.arange(N) / N + 0.3
    f, _, A, _ = ref.forces_abs(RING, 0.01, th, form=0)
    assert np.max(np.abs(f)) <= 1e-14 * np.max(A)


def test_ring_large_eps_limit_is_hmf(ref):
    """'the limit for large values of eps' of the Ring model is the HMF model.
    f_ring * 2 sqrt2 eps^(3/2) -> f_HMF with relative deviation <= 3/eps."""
    rng = np.random.default_rng(9)
    th = rng.uniform(-2, 2, 200)
    fh = ref.forces(HMF, 0.0, th)
    prev = None
    for eps in (1e2, 1e4, 1e6):
        fr = ref.forces(RING, eps, th, form=0) * (2 * math.sqrt(2) * eps ** 1.5)
        dev = np.max(np.abs(fr - fh)) / np.max(np.abs(fh))
        assert dev <= 3.0 / eps
        if prev is not None:
            assert dev < prev / 50      # first-order in 1/eps
        prev = dev


@pytest.mark.parametrize("N,R", [(3, 1.0), (7, 1.3), (32, 0.4)])
def test_grav2d_regular_polygon_closed_form(ref, N, R):
    """Regular N-gon of radius R, eps = 0: every pair's radial component is 1/(2R), so
    F_i = -((N-1)/(N R)) r_hat_i exactly (a property of eq.(3))."""
    phi = 2 * math.pi * np.arange(N) / N + 0.2
    x, y = R * np.cos(phi), R * np.sin(phi)
    fx, fy = ref.forces(GRAV2D, 0.0, x, y)
    mag = (N - 1) / (N * R)
    assert np.max(np.abs(fx + mag * np.cos(phi))) < 1e-13 * mag * N
    assert np.max(np.abs(fy + mag * np.sin(phi))) < 1e-13 * mag * N


def test_two_body_closed_forms(ref):
    """N = 2: HMF V = (1/2)(1 - cos D), f_1 = -(1/2) sin D; Ring V = -1/(2 sqrt2 sqrt(1-cos D+eps));
    2D V = (1/2) log(r^2 + eps), F_1 = -(r1 - r2)/(r^2 + eps)."""
    D = 0.9
    th = np.array([0.2 + D, 0.2]); z = np.zeros(2)
    f = ref.forces(HMF, 0.0, th)
    assert abs(f[0] + 0.5 * math.sin(D)) < 1e-15 and abs(f[0] + f[1]) < 1e-15
    assert abs(ref.energy(HMF, 0.0, th, None, z, None)[0][1] - 0.5 * (1 - math.cos(D))) < 1e-15
    eps = 0.05
    d = 1 - math.cos(D) + eps
    f = ref.forces(RING, eps, th)
    assert abs(f[0] + math.sin(D) / (4 * math.sqrt(2) * d ** 1.5)) < 1e-15
    assert abs(ref.energy(RING, eps, th, None, z, None)[0][1] + 1 / (2 * math.sqrt(2) * math.sqrt(d))) < 1e-15
    x = np.array([0.3, -0.4]); y = np.array([0.1, 0.6])
    r2 = 0.7 ** 2 + 0.5 ** 2 + eps
    fx, fy = ref.forces(GRAV2D, eps, x, y)
    assert abs(fx[0] + 0.7 / r2) < 1e-15 and abs(fy[0] - 0.5 / r2) < 1e-15
    assert abs(fx[0] + fx[1]) < 1e-15 and abs(fy[0] + fy[1]) < 1e-15
    assert abs(ref.energy(GRAV2D, eps, x, y, z, z)[0][1] - 0.5 * math.log(r2)) < 1e-15


@pytest.mark.parametrize("model,eps", [(HMF, 0.0), (RING, 0.01), (GRAV2D, 1e-3)])
def test_pair_forces_are_antisymmetric_total_force_zero(ref, model, eps):
    N = 500
    q0, q1 = _rand_state(model, N, 21)
    f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=1)
    assert abs(math.fsum(f0)) <= 1e-15 * math.fsum(A0)
    if model == GRAV2D:
        assert abs(math.fsum(f1)) <= 1e-15 * math.fsum(A1)
        # central forces: zero total torque
        assert abs(math.fsum(q0 * f1 - q1 * f0)) <= 1e-14 * math.fsum(A0 + A1)


def test_forces_are_2pi_periodic(ref):
    rng = np.random.default_rng(1)
    th = rng.uniform(-1, 1, 100)
    k = rng.integers(-3, 4, 100)
    for model, eps in ((HMF, 0.0), (RING, 0.01)):
        a = ref.forces(model, eps, th, form=0)
        b, _, A, _ = ref.forces_abs(model, eps, th + 2 * math.pi * k, form=0)
        tol = 1e-13 * np.max(A) if model == HMF else 1e-11 * np.max(A)   # Ring: |df/dth| ~ eps^-1
        assert np.max(np.abs(a - b)) <= max(tol, 1e-13)


def test_abs_sums_rows_and_threads(ref):
    """A_i = sum_{j != i} |f_ij| by brute force; sampled rows == full rows; bit-identical for any
    thread count (every row keeps its serial j order)."""
    N = 40
    x, y = _rand_state(GRAV2D, N, 2)
    eps = 1e-3
    f0, f1, A0, A1 = ref.forces_abs(GRAV2D, eps, x, y)
    for i in (0, 17, 39):
        ax = math.fsum(abs((x[i] - x[j]) / ((x[i] - x[j]) ** 2 + (y[i] - y[j]) ** 2 + eps))
                       for j in range(N) if j != i) * 2 / N
        assert abs(A0[i] - ax) <= 1e-14 * ax
        assert A0[i] >= abs(f0[i]) and A1[i] >= abs(f1[i])
    rows = np.array([39, 0, 17, 17])
    g0, g1 = ref.forces_rows(GRAV2D, eps, x, y, rows)
    assert np.array_equal(g0, f0[rows]) and np.array_equal(g1, f1[rows])
    th, _ = _rand_state(RING, 300, 4)
    a = ref.forces(RING, 0.01, th, form=1, nthreads=1)
    b = ref.forces(RING, 0.01, th, form=1, nthreads=4)
    assert np.array_equal(a, b)
    # HMF O(N) bound S_i >= A_i
    thh, _ = _rand_state(HMF, 200, 6)
    _, _, S, _ = ref.forces_abs(HMF, 0.0, thh, form=0)
    _, _, A, _ = ref.forces_abs(HMF, 0.0, thh, form=1)
    assert np.all(S >= A * (1 - 1e-12) - 1.0 / 200)


def _pair_potential_mp(model, eps, ai, bi, aj, bj, N):
    """One term of the printed double sums (eq.(1), :36 eq.(2), :40 eq.(3)), with its 1/N."""
    if model == HMF:
        return (1 - mp.cos(ai - aj)) / N
    if model == RING:
        return -1 / (mp.sqrt(2) * mp.sqrt(1 - mp.cos(ai - aj) + eps)) / N
    return mp.log((ai - aj) ** 2 + (bi - bj) ** 2 + eps) / N


@pytest.mark.parametrize("model,eps,form", [(HMF, 0.0, 1), (RING, 0.01, 0), (RING, 0.01, 1), (RING, 1e-3, 1),
                                            (GRAV2D, 1e-3, 0)])
def test_abs_force_sums_every_branch(ref, model, eps, form):
    """Pins lrmd_ref_abs_force_sums, the scale A_i = sum_{j != i} |f_ij| of every force tolerance
    (north_star: |f_gpu - f_ref|_i <= 1e-12 A_i), for every branch that computes it: each |f_ij| is the
    absolute value of the mpmath numerical derivative of ONE printed pair-potential term with respect to
    particle i's coordinate — no force formula is typed here, so a dropped fabs, a wrong prefactor or a
    swapped component in the oracle fails."""
    N = 9
    q0, q1 = _rand_state(model, N, 31 + model)
    f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=form)
    e = mp.mpf(float(eps))
    a = [mp.mpf(float(v)) for v in q0]
    b = [mp.mpf(0)] * N if q1 is None else [mp.mpf(float(v)) for v in q1]
    for i in range(N):
        ex = mp.mpf(0)
        ey = mp.mpf(0)
        for j in range(N):
            if j == i:
                continue
            ex += abs(mp.diff(lambda z: _pair_potential_mp(model, e, z, b[i], a[j], b[j], N), a[i]))
            if model == GRAV2D:
                ey += abs(mp.diff(lambda z: _pair_potential_mp(model, e, a[i], z, a[j], b[j], N), b[i]))
        assert abs(A0[i] - float(ex)) <= 1e-13 * float(ex), (i, A0[i], float(ex))
        assert A0[i] >= abs(f0[i]) * (1 - 1e-15)
        if model == GRAV2D:
            assert abs(A1[i] - float(ey)) <= 1e-13 * float(ey), (i, A1[i], float(ey))
            assert A1[i] >= abs(f1[i]) * (1 - 1e-15)
    # sampled rows return the same A_i as the full call
    rows = np.array([N - 1, 0, 4])
    out = ref.forces_rows(model, eps, q0, q1, rows, form=form, with_abs=True)
    assert np.array_equal(out[2], A0[rows])
    if model == GRAV2D:
        assert np.array_equal(out[3], A1[rows])


def test_hmf_force_bound_is_pinned_from_both_sides(ref):
    """The O(N) scale used at N = 5e7 (config 4), S_i = |cos t_i| <|sin|> + |sin t_i| <|cos|>:
    (a) it equals that expression evaluated independently with math.fsum, to rounding — so it cannot be
    over-generous; (b) it bounds the true A_i = (1/N) sum_{j != i} |sin(t_i - t_j)| from above (triangle
    inequality on sin(a - b) = sin a cos b - cos a sin b), and is not far above it (<= sqrt2 A_i + 1/N for
    angles spread over the circle)."""
    N = 300
    th, _ = _rand_state(HMF, N, 6)
    _, _, S, _ = ref.forces_abs(HMF, 0.0, th, form=0)
    mean_abs_sin = math.fsum(abs(math.sin(t)) for t in th) / N
    mean_abs_cos = math.fsum(abs(math.cos(t)) for t in th) / N
    for i in range(N):
        want = abs(math.cos(th[i])) * mean_abs_sin + abs(math.sin(th[i])) * mean_abs_cos
        assert abs(S[i] - want) <= 4e-16 * want
        A = math.fsum(abs(math.sin(th[i] - t)) for j, t in enumerate(th) if j != i) / N
        assert S[i] >= A * (1 - 1e-14)
        assert S[i] <= 2.0 * A + 1.0 / N
    # sampled rows carry the same bound
    rows = np.array([7, 299, 0])
    out = ref.forces_rows(HMF, 0.0, th, None, rows, form=0, with_abs=True)
    assert np.array_equal(out[2], S[rows])


def test_waterbag_magnetisation_statistics(ref):
    """Config-1 shaped input: theta ~ U[-1.5, 1.5) => E[M] = sin(1.5)/1.5 = 0.66500."""
    from paper_1212_0262_b200 import inputs
    th, p = inputs.WORKLOADS["hmf_1e4"].state()
    e, _ = ref.energy(HMF, 0.0, th, None, p, None)
    assert abs(e[2] - math.sin(1.5) / 1.5) < 0.02 and abs(e[3]) < 0.02
    assert abs(e[0] / 1e4 - 0.5 / 12) < 0.002          # <p^2>/2 = (1/2)(1/12) for U[-.5,.5)


def test_invalid_arguments_are_rejected(ref):
    with pytest.raises(ValueError):
        ref.forces(3, 0.0, np.zeros(4))
    with pytest.raises(ValueError):
        ref.forces(RING, -1.0, np.zeros(4))
    with pytest.raises(ValueError):
        ref.forces_rows(HMF, 0.0, np.zeros(4), None, np.array([4]))
