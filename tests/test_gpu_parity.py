"""Parity of the CUDA path (through the C ABI, include/lrmd.h) with the oracle (oracle/lrmd_ref.cpp)
on the same seeded inputs.  Tolerances are BASELINE.json's north_star:
    forces      |f_gpu - f_ref|_i <= 1e-12 * A_i,  A_i = sum_{j != i} |f_ij|
    trajectory  positions and momenta within 1e-9 (absolute) after 10 steps
    energies    K, V within 1e-12 * sum |terms|        (proposed addition)
    long run    max relative energy error of the same order of magnitude as the oracle's
Several summation orders are correct (reading G15): the GPU result is additionally required to be
bitwise reproducible run to run.
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

HMF, RING, GRAV2D = 0, 1, 2
FTOL = 1e-12
XTOL = 1e-9


@pytest.fixture(scope="module")
def torch():
    import torch as _torch
    assert _torch.cuda.is_available(), "GPU tests need a CUDA device"
    return _torch


def _state(model, N, seed):
    rng = np.random.default_rng(seed)
    if model == GRAV2D:
        u1, u2 = rng.random(N), rng.random(N)
        r, ph = np.sqrt(u1), 2 * math.pi * u2
        px, py = 0.1 * rng.standard_normal(N), 0.1 * rng.standard_normal(N)
        return [r * np.cos(ph), r * np.sin(ph), px - px.mean(), py - py.mean()]
    a = 1.5 if model == HMF else 1.0
    return [rng.uniform(-a, a, N), rng.uniform(-0.5, 0.5, N)]


def _eps(model):
    return {HMF: 0.0, RING: 0.01, GRAV2D: 1e-3}[model]


def _q(model, st):
    return (st[0], st[1]) if model == GRAV2D else (st[0], None)


def _p(model, st):
    return (st[2], st[3]) if model == GRAV2D else (st[1], None)


def _gpu_forces(lrmd, model, eps, st, options=None):
    ctx = lrmd.Context(model, len(st[0]), eps, options=options)
    ctx.set_state(*st)
    f = ctx.forces()
    out = tuple(t.cpu().numpy() for t in f) if model == GRAV2D else (f.cpu().numpy(), None)
    n_launch = ctx.launch_count()
    ctx.close()
    assert n_launch > 0
    return out


def _check_forces(model, got, want, A):
    for g, w, a in zip(got, want, A):
        if g is None:
            continue
        err = np.abs(g - w)
        # HMF goes through the identity eq.(6): its two O(1) products cos*My, sin*Mx cancel the self term
        # only to rounding, so a floor of a few 2^-53 applies (matters only where A_i ~ 0, e.g. N = 1)
        tol = FTOL * a + (4e-16 if model == HMF else 1e-300)
        bad = np.nonzero(err > tol)[0]
        assert bad.size == 0, (model, bad[:5], err[bad[:5]], tol[bad[:5]], float((err / tol).max()))


HMF_FULL_A_MAX_N = 20_480


def _hmf_true_A(ref, theta, nsample=1024, seed=0):
    """A_i = sum_{j != i} |f_ij| of eq.(2)'s pair terms (oracle form=1, O(N^2)): the scale north_star states for the force
    tolerance.  Every row up to N = 20,480.  Beyond, it is computed exactly on `nsample` seeded rows (plus the rows of the
    smallest and largest angle) and interpolated linearly in theta for the others — A is a smooth function of theta_i
    alone, |dA/dtheta| <= 1 — with 2 % taken off as a margin.  Returns (A on all rows, sampled rows or None, the
    oracle's pair-sum forces on the sampled rows or None, exact A on the sampled rows or None)."""
    N = theta.size
    if N <= HMF_FULL_A_MAX_N:
        _, _, A, _ = ref.forces_abs(HMF, 0.0, theta, None, form=1)
        return A, None, None, None
    rows = np.random.default_rng(seed).choice(N, min(nsample, N), replace=False)
    rows = np.unique(np.concatenate([rows, [int(np.argmin(theta)), int(np.argmax(theta))]]))
    fr, _, Ar, _ = ref.forces_rows(HMF, 0.0, theta, None, rows, form=1, with_abs=True)
    order = np.argsort(theta[rows])
    A = 0.98 * np.interp(theta, theta[rows][order], Ar[order])
    return A, rows, fr, Ar


def _check_hmf_forces(ref, theta, got, what=None, nsample=1024):
    """HMF forces `got` at angles `theta` against the oracle within 1e-12 * A_i, A_i the TRUE pair-term sum (not the
    O(N) bound S_i >= A_i, which is up to twice as loose): every row against the oracle's eq.(6)-(7) path, the sampled
    rows (N > 20,480) also against its O(N^2) pair sum with their exact A_i.  The 4e-16 floor is _check_forces's."""
    f_ref = ref.forces(HMF, 0.0, theta, None, form=0)
    A, rows, fr, Ar = _hmf_true_A(ref, theta, nsample=nsample)
    err = np.abs(got - f_ref)
    tol = FTOL * A + 4e-16
    bad = np.nonzero(err > tol)[0]
    assert bad.size == 0, (what, bad[:5], err[bad[:5]], tol[bad[:5]])
    if rows is not None:
        err = np.abs(got[rows] - fr)
        tol = FTOL * Ar + 4e-16
        bad = np.nonzero(err > tol)[0]
        assert bad.size == 0, (what, rows[bad[:5]], err[bad[:5]], tol[bad[:5]])


# ---- forces: sizes that span several i-tiles / j-tiles, ragged tails, degenerate sizes ----------------

@pytest.mark.parametrize("model", [HMF, RING, GRAV2D])
@pytest.mark.parametrize("N", [1, 2, 3, 5, 255, 256, 257, 511, 512, 513, 1000, 1024, 4099])
def test_forces_match_oracle_small_and_ragged(lrmd, ref, torch, model, N):
    eps = _eps(model)
    st = _state(model, N, 1000 + N)
    q0, q1 = _q(model, st)
    f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=(1 if model == HMF else 0))
    got = _gpu_forces(lrmd, model, eps, st)
    _check_forces(model, got, (f0, f1), (A0, A1))


@pytest.mark.parametrize("model", [RING, GRAV2D])
@pytest.mark.parametrize("S", [1, 2, 3, 7, 16, 148, 1000, 12500])
def test_forces_any_partition(lrmd, ref, torch, model, S):
    """Any number of CTAs over the flattened (i-tile, j) space; partial-force rows summed in slot order (row a-U1)."""
    eps = _eps(model)
    N = 2500
    st = _state(model, N, 77)
    q0, q1 = _q(model, st)
    f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=0)
    got = _gpu_forces(lrmd, model, eps, st, options={lrmd.OPT_PAIR_SYMMETRIC: 0, lrmd.OPT_PAIR_CTAS: S})
    _check_forces(model, got, (f0, f1), (A0, A1))


@pytest.mark.parametrize("grid", [1, 3, 148, 1184])
def test_hmf_forces_any_grid(lrmd, ref, torch, grid):
    N = 100_003
    st = _state(HMF, N, 5)
    got = _gpu_forces(lrmd, HMF, 0.0, st, options={lrmd.OPT_HMF_GRID: grid})
    _check_hmf_forces(ref, st[0], got[0], grid)


@pytest.mark.parametrize("variant", [1, 2])
@pytest.mark.parametrize("N", [1, 2, 7, 2047, 2048, 2049, 300_001])
def test_hmf_tma_variants_match_oracle(lrmd, ref, torch, variant, N):
    """TMA-staged fused substage (persistent CTAs, smem ring, bulk loads and stores): forces and a
    3-step trajectory against the oracle; odd N exercises the scalar tail, N < chunk the short copies."""
    st = _state(HMF, N, 700 + N % 97)
    ctx = lrmd.Context(HMF, N, 0.0, options={lrmd.OPT_HMF_VARIANT: variant, lrmd.OPT_GRAPH: 0})
    ctx.set_state(*st)
    got = ctx.forces().cpu().numpy()
    _check_hmf_forces(ref, st[0], got, (variant, N))
    ctx.step(3, 0.05)
    e = ctx.energy().cpu().numpy()
    out = ctx.state_numpy()
    ctx.close()
    th, p = st[0].copy(), st[1].copy()
    ref.step(HMF, 0.0, th, None, p, None, 3, 0.05, form=0)
    assert np.max(np.abs(out[0] - th)) <= XTOL and np.max(np.abs(out[1] - p)) <= XTOL
    er, ea = ref.energy(HMF, 0.0, th, None, p, None)
    assert abs(e[0] - er[0]) <= 1e-12 * ea[0] + 1e-300
    assert abs(e[1] - er[1]) <= 1e-12 * max(ea[1], 0.5 * N) + 1e-300


@pytest.mark.parametrize("N", [1, 2, 31, 640, 2559, 2560, 2561, 5121, 10_000, 10_241, 20_480])
def test_hmf_cluster_resident_kernel_matches_oracle(lrmd, ref, torch, N):
    """Cluster-resident HMF kernel (variant 3; 1, 2, 4 or 8 particles per thread): 7-step trajectory, the
    cached sums it leaves behind (forces, energy) and step(n) == n x step(1) bit for bit."""
    st = _state(HMF, N, 300 + N % 11)
    ctx = lrmd.Context(HMF, N, 0.0, options={lrmd.OPT_HMF_VARIANT: 3})
    assert ctx.get_option(lrmd.OPT_HMF_VARIANT) == 3
    ctx.set_state(*st)
    ctx.step(7, 0.05)
    out = ctx.state_numpy()
    f = ctx.forces().cpu().numpy()
    e = ctx.energy().cpu().numpy()
    assert ctx.launch_count() <= 1 + 1 + 2      # one launch for the 7 steps, one for forces, two for the energy
    ctx.close()
    th, p = st[0].copy(), st[1].copy()
    ref.step(HMF, 0.0, th, None, p, None, 7, 0.05, form=0)
    assert np.max(np.abs(out[0] - th)) <= XTOL and np.max(np.abs(out[1] - p)) <= XTOL
    _check_hmf_forces(ref, out[0], f, N)      # at the GPU's own final angles
    er, ea = ref.energy(HMF, 0.0, out[0], None, out[1], None)
    assert abs(e[0] - er[0]) <= 1e-12 * ea[0] + 1e-300 and abs(e[1] - er[1]) <= 1e-12 * max(ea[1], 0.5 * N) + 1e-300
    b = lrmd.Context(HMF, N, 0.0, options={lrmd.OPT_HMF_VARIANT: 3})
    b.set_state(*st)
    for _ in range(7):
        b.step(1, 0.05)
    for x, y in zip(out, b.state_numpy()):
        assert np.array_equal(x, y)
    b.close()


def test_hmf_cluster_of_16_ctas_same_trajectory(lrmd, torch):
    """The non-portable cluster size (LRMD_OPT_HMF_GRID = 16) changes the summation tree only."""
    N = 10_000
    st = _state(HMF, N, 77)
    outs = []
    for g in (8, 16):
        ctx = lrmd.Context(HMF, N, 0.0, options={lrmd.OPT_HMF_VARIANT: 3, lrmd.OPT_HMF_GRID: g})
        ctx.set_state(*st)
        ctx.step(25, 0.05)
        assert ctx.get_option(lrmd.OPT_HMF_GRID) == g
        outs.append(ctx.state_numpy())
        ctx.close()
    for x, y in zip(*outs):
        assert np.max(np.abs(x - y)) <= 1e-11


def test_hmf_cluster_variant_falls_back_above_its_size(lrmd, torch):
    ctx = lrmd.Context(HMF, 20_481, 0.0, options={lrmd.OPT_HMF_VARIANT: 3})
    assert ctx.get_option(lrmd.OPT_HMF_VARIANT) == 0
    ctx.close()


@pytest.mark.parametrize("N", [1, 2, 147, 149, 20_481, 100_000, 300_001, 1_070_336])
def test_hmf_grid_resident_kernel_matches_oracle(lrmd, ref, torch, N):
    """LRMD_OPT_HMF_VARIANT = 4: the whole state in shared memory, one cooperative launch per lrmd_step call, a grid
    barrier per substage.  Fewer particles than CTAs, ragged shares, the largest size that fits; forces before and
    after, 10-step trajectory, energies; step(10) == 10 x step(1) bit for bit; run-to-run reproducible."""
    st = _state(HMF, N, 2_000 + N % 11)
    outs = []
    for single in (False, True, False):
        ctx = lrmd.Context(HMF, N, 0.0, options={lrmd.OPT_HMF_VARIANT: 4})
        assert ctx.get_option(lrmd.OPT_HMF_VARIANT) == 4
        ctx.set_state(*st)
        if single:
            for _ in range(10):
                ctx.step(1, 0.05)
        else:
            ctx.step(10, 0.05)
        outs.append(ctx.state_numpy())
        f = ctx.forces().cpu().numpy()
        e = ctx.energy().cpu().numpy()
        assert ctx.get_option(lrmd.OPT_HMF_VARIANT) == 4          # no fallback happened
        ctx.close()
    for other in outs[1:]:
        assert np.array_equal(outs[0][0], other[0]) and np.array_equal(outs[0][1], other[1])
    th, p = st[0].copy(), st[1].copy()
    ref.step(HMF, 0.0, th, None, p, None, 10, 0.05, form=0)
    assert np.max(np.abs(outs[0][0] - th)) <= XTOL and np.max(np.abs(outs[0][1] - p)) <= XTOL
    _check_hmf_forces(ref, outs[0][0], f, N)
    er, ea = ref.energy(HMF, 0.0, outs[0][0], None, outs[0][1], None)
    assert abs(e[0] - er[0]) <= 1e-12 * max(ea[0], 1e-300) and abs(e[1] - er[1]) <= 1e-12 * max(ea[1], 0.5 * N)


def test_hmf_grid_resident_kernel_default_range_and_limits(lrmd, torch):
    a = lrmd.Context(HMF, 20_480, 0.0)
    b = lrmd.Context(HMF, 20_481, 0.0)
    c = lrmd.Context(HMF, 1_000_000, 0.0)
    d = lrmd.Context(HMF, 1_070_337, 0.0, options={lrmd.OPT_HMF_VARIANT: 4})      # does not fit: TMA-staged kernel
    assert a.get_option(lrmd.OPT_HMF_VARIANT) == 3 and b.get_option(lrmd.OPT_HMF_VARIANT) == 4
    assert c.get_option(lrmd.OPT_HMF_VARIANT) == 4 and d.get_option(lrmd.OPT_HMF_VARIANT) == 1
    for x in (a, b, c, d):
        x.close()


@pytest.mark.parametrize("variant", [1, 2])
def test_hmf_tma_variant_graph_and_grid(lrmd, torch, variant):
    """Graph replay and a non-default grid give the same bits as plain launches of the same variant and grid."""
    N = 40_001
    st = _state(HMF, N, 3)
    outs = []
    for graph in (0, 1):
        ctx = lrmd.Context(HMF, N, 0.0, options={lrmd.OPT_HMF_VARIANT: variant, lrmd.OPT_GRAPH: graph, lrmd.OPT_HMF_GRID: 5})
        ctx.set_state(*st)
        ctx.step(20, 0.05)
        outs.append(ctx.state_numpy())
        ctx.close()
    for x, y in zip(*outs):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("model", [RING, GRAV2D])
@pytest.mark.parametrize("variant", [0, 1, 2])
@pytest.mark.parametrize("symmetric", [0, 1])
def test_pair_variants_match_oracle(lrmd, ref, torch, model, variant, symmetric):
    """Every compiled launch shape of the ORDERED pair kernels (PairCfg0/1/2: pair_force_kernel, pair_energy_kernel;
    LRMD_OPT_PAIR_SYMMETRIC pinned to 0) and, as its twin, of the symmetric kernels: forces and potential energy
    against the oracle."""
    if symmetric and variant == 2:
        pytest.skip("the symmetric kernels have two tile sizes (variants 0 and 1)")
    eps = _eps(model)
    N = 3333
    st = _state(model, N, 55)
    q0, q1 = _q(model, st)
    p0, p1 = _p(model, st)
    f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=0)
    ctx = lrmd.Context(model, N, eps, options={lrmd.OPT_PAIR_VARIANT: variant, lrmd.OPT_PAIR_SYMMETRIC: symmetric})
    assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == symmetric
    ctx.set_state(*st)
    f = ctx.forces()
    got = tuple(t.cpu().numpy() for t in f) if model == GRAV2D else (f.cpu().numpy(), None)
    e = ctx.energy().cpu().numpy()
    ctx.close()
    _check_forces(model, got, (f0, f1), (A0, A1))
    e_ref, e_abs = ref.energy(model, eps, q0, q1, p0, p1)
    assert abs(e[1] - e_ref[1]) <= 1e-12 * e_abs[1]


@pytest.mark.parametrize("model,eps", [(RING, 1e-3), (RING, 1.0), (RING, 1e4), (GRAV2D, 1e-6), (GRAV2D, 10.0)])
def test_forces_other_softenings(lrmd, ref, torch, model, eps):
    N = 1500
    st = _state(model, N, 31)
    q0, q1 = _q(model, st)
    f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=0)
    if model == RING and eps < 0.01:
        # eq.(9)'s denominator cancels to ~eps for close pairs: relative rounding 2^-53/eps per pair,
        # x1.5 in d^(-3/2) (same allowance as the oracle's own eq.(8)-vs-eq.(9) pin)
        A0 = A0 * max(1.0, 1.5 * 4e-16 / eps / FTOL)
    for sym in (0, 1):     # the ordered kernel and the symmetric one
        got = _gpu_forces(lrmd, model, eps, st, options={lrmd.OPT_PAIR_SYMMETRIC: sym})
        _check_forces(model, got, (f0, f1), (A0, A1))


def test_forces_coincident_particles(lrmd, ref, torch):
    """Degenerate input: pairs of particles at identical positions (d_ij = eps exactly)."""
    for model in (RING, GRAV2D):
        eps = _eps(model)
        st = _state(model, 600, 3)
        for a in st:
            a[300:] = a[:300]
        q0, q1 = _q(model, st)
        f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=0)
        for sym in (0, 1):
            got = _gpu_forces(lrmd, model, eps, st, options={lrmd.OPT_PAIR_SYMMETRIC: sym})
            _check_forces(model, got, (f0, f1), (A0, A1))


# ---- the BASELINE.json configs at full size -----------------------------------------------------------

def test_config1_hmf_1e4_forces_and_energy(lrmd, ref, torch, inputs):
    w = inputs.WORKLOADS["hmf_1e4"]
    th, p = w.state()
    f_pair, _, A, _ = ref.forces_abs(HMF, 0.0, th, None, form=1)      # O(N^2) pair sum of eq.(2)
    ctx = lrmd.Context(HMF, w.N)
    ctx.set_state(th, p)
    f = ctx.forces().cpu().numpy()
    assert np.all(np.abs(f - f_pair) <= FTOL * A)
    e = ctx.energy().cpu().numpy()
    e_ref, e_abs = ref.energy(HMF, 0.0, th, None, p, None, form=0)
    assert abs(e[0] - e_ref[0]) <= 1e-12 * e_abs[0] and abs(e[1] - e_ref[1]) <= 1e-12 * e_abs[1]
    assert abs(e[2] - e_ref[2]) <= 1e-15 * 2 and abs(e[3] - e_ref[3]) <= 1e-15 * 2
    ctx.close()


@pytest.mark.parametrize("key", ["hmf_1e4", "ring_16k", "grav2d_64k"])
def test_trajectory_10_steps_full_configs(lrmd, ref, torch, inputs, key):
    """Configs 1-3 at full N: 10 steps, every position and momentum within 1e-9."""
    w = inputs.WORKLOADS[key]
    st = [a.copy() for a in w.state()]
    ctx = lrmd.Context(w.model, w.N, w.eps)
    ctx.set_state(*st)
    ctx.step(10, w.dt)
    got = ctx.state_numpy()
    f_gpu = ctx.forces()
    ctx.close()
    q0, q1 = _q(w.model, st)
    p0, p1 = _p(w.model, st)
    rf0, rf1 = ref.step(w.model, w.eps, q0, q1, p0, p1, 10, w.dt, form=(0 if w.model == HMF else 1))
    for g, r in zip(got, st):
        assert np.max(np.abs(g - r)) <= XTOL
    # the cached force after the step is f(q(t + 10 dt))
    fg = f_gpu if w.model == GRAV2D else (f_gpu, None)
    for g, r in zip(fg, (rf0, rf1)):
        if g is not None:
            assert np.max(np.abs(g.cpu().numpy() - r)) <= 1e-9 * max(1.0, np.max(np.abs(r)))


def test_config2_ring_forces_and_energy_full(lrmd, ref, torch, inputs):
    w = inputs.WORKLOADS["ring_16k"]
    th, p = w.state()
    f0, _, A0, _ = ref.forces_abs(RING, w.eps, th, None, form=0)
    ctx = lrmd.Context(RING, w.N, w.eps)
    ctx.set_state(th, p)
    f = ctx.forces().cpu().numpy()
    assert np.all(np.abs(f - f0) <= FTOL * A0)
    e = ctx.energy().cpu().numpy()
    e_ref, e_abs = ref.energy(RING, w.eps, th, None, p, None)
    assert abs(e[0] - e_ref[0]) <= 1e-12 * e_abs[0]
    assert abs(e[1] - e_ref[1]) <= 1e-12 * e_abs[1]
    assert abs(e[2] - e_ref[2]) <= 1e-12 * np.sum(np.abs(p)) and e[3] == 0.0
    ctx.close()


def test_config3_grav2d_forces_and_energy_full(lrmd, ref, torch, inputs):
    w = inputs.WORKLOADS["grav2d_64k"]
    x, y, px, py = w.state()
    rows = np.random.default_rng(9).choice(w.N, 2048, replace=False)
    f0, f1, A0, A1 = ref.forces_rows(GRAV2D, w.eps, x, y, rows, with_abs=True)
    ctx = lrmd.Context(GRAV2D, w.N, w.eps)
    ctx.set_state(x, y, px, py)
    fx, fy = (t.cpu().numpy() for t in ctx.forces())
    assert np.all(np.abs(fx[rows] - f0) <= FTOL * A0) and np.all(np.abs(fy[rows] - f1) <= FTOL * A1)
    e = ctx.energy().cpu().numpy()
    e_ref, e_abs = ref.energy(GRAV2D, w.eps, x, y, px, py)
    assert abs(e[0] - e_ref[0]) <= 1e-12 * e_abs[0]
    assert abs(e[1] - e_ref[1]) <= 1e-12 * e_abs[1]
    assert abs(e[2] - e_ref[2]) <= 1e-12 * np.sum(np.abs(px)) and abs(e[3] - e_ref[3]) <= 1e-12 * np.sum(np.abs(py))
    ctx.close()


def test_config4_hmf_5e7_sampled_and_invariants(lrmd, ref, torch, inputs):
    """Config 4 at full size in bench.py's launch configuration: forces on all rows at t = 0 against
    the oracle's eq.(6)-(7) path (tolerance scaled by the O(N) bound S_i >= A_i — the one size where SURVEY.md 8(c)
    item 4 allows it, the O(N^2) sum over all rows being impossible — and by the TRUE A_i on 256 sampled rows),
    then 10 GPU steps and (i) every position and momentum against 10 oracle steps, (ii) forces at the GPU's
    final angles on sampled rows, (iii) energy and momentum conservation, the relative energy error beside the
    oracle's own over the same 10 steps (north_star: "same order of magnitude as the oracle's")."""
    w = inputs.WORKLOADS["hmf_5e7"]
    th, p = w.state()
    ctx = lrmd.Context(HMF, w.N)
    ctx.set_state(th, p)
    f = ctx.forces().cpu().numpy()
    f_ref, _, S, _ = ref.forces_abs(HMF, 0.0, th, None, form=0)
    assert np.all(np.abs(f - f_ref) <= FTOL * S)
    rows_a = np.random.default_rng(40).choice(w.N, 256, replace=False)
    fa, _, Aa, _ = ref.forces_rows(HMF, 0.0, th, None, rows_a, form=1, with_abs=True)      # O(N^2) pair sum, true A_i
    assert np.all(np.abs(f[rows_a] - fa) <= FTOL * Aa)
    e0 = ctx.energy().cpu().numpy()
    e_ref, e_abs = ref.energy(HMF, 0.0, th, None, p, None, form=0)
    assert abs(e0[0] - e_ref[0]) <= 1e-12 * e_abs[0] and abs(e0[1] - e_ref[1]) <= 1e-12 * e_abs[1]
    P0 = float(ctx.state[1].sum())
    ctx.step(10, w.dt)
    e1 = ctx.energy().cpu().numpy()
    thg, pg = ctx.state_numpy()
    # north_star: positions and momenta within 1e-9 after 10 steps, at the full N = 5e7 (listing PAPER.md:54-62);
    # the oracle's eq.(6)-(7) path is O(N) per force evaluation
    rth, rp = th.copy(), p.copy()
    ref.step(HMF, 0.0, rth, None, rp, None, 10, w.dt, form=0)
    assert np.max(np.abs(thg - rth)) <= XTOL and np.max(np.abs(pg - rp)) <= XTOL
    e_ref1, _ = ref.energy(HMF, 0.0, rth, None, rp, None, form=0)
    del rth, rp
    rows = np.random.default_rng(4).choice(w.N, 4096, replace=False)
    fr, _, Sr, _ = ref.forces_rows(HMF, 0.0, thg, None, rows, with_abs=True)
    fg = ctx.forces().cpu().numpy()
    assert np.all(np.abs(fg[rows] - fr) <= FTOL * Sr)
    E0, E1 = e0[0] + e0[1], e1[0] + e1[1]
    assert abs((E1 - E0) / E0) < 1e-7                 # dt = 0.05, 4th order: ~1e-9 expected
    dE_gpu = abs((E1 - E0) / E0)
    dE_ref = abs((e_ref1[0] + e_ref1[1] - e_ref[0] - e_ref[1]) / (e_ref[0] + e_ref[1]))
    assert dE_ref > 1e-12 and 0.1 <= dE_gpu / dE_ref <= 10.0, (dE_gpu, dE_ref)      # well above the 1e-16-level rounding of the sums
    assert abs(float(ctx.state[1].sum()) - P0) <= 1e-12 * float(np.sum(np.abs(pg)))
    ctx.close()


@pytest.mark.parametrize("symmetric", [-1, 0])
def test_config5_grav2d_1m_sampled_rows(lrmd, ref, torch, inputs, symmetric):
    """Config 5 at full size, in the launch configuration bench.py times (default: the band kernel, one launch per
    force evaluation) and with the ordered kernel: forces on sampled rows (each against all N) at t = 0 and at
    the GPU's positions after one step."""
    w = inputs.WORKLOADS["grav2d_1m"]
    x, y, px, py = w.state()
    rows = np.random.default_rng(6).choice(w.N, 4096, replace=False)      # >= 4,096 sampled rows
    ctx = lrmd.Context(GRAV2D, w.N, w.eps, options={lrmd.OPT_PAIR_SYMMETRIC: symmetric})
    assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == (2 if symmetric else 0)     # default at this N: the band kernel
    ctx.set_state(x, y, px, py)
    fx, fy = (t.cpu().numpy() for t in ctx.forces())
    f0, f1, A0, A1 = ref.forces_rows(GRAV2D, w.eps, x, y, rows, with_abs=True)
    assert np.all(np.abs(fx[rows] - f0) <= FTOL * A0) and np.all(np.abs(fy[rows] - f1) <= FTOL * A1)
    assert abs(math.fsum(fx)) <= 1e-13 * math.fsum(np.abs(fx)) + 1e-12   # antisymmetry: total force 0
    ctx.step(1, w.dt)
    xg, yg, pxg, pyg = ctx.state_numpy()
    fx, fy = (t.cpu().numpy() for t in ctx.forces())
    f0, f1, A0, A1 = ref.forces_rows(GRAV2D, w.eps, xg, yg, rows, with_abs=True)
    assert np.all(np.abs(fx[rows] - f0) <= FTOL * A0) and np.all(np.abs(fy[rows] - f1) <= FTOL * A1)
    scale = math.fsum(np.abs(pxg))
    assert abs(math.fsum(pxg)) <= 1e-12 * scale and abs(math.fsum(pyg)) <= 1e-12 * scale
    ctx.close()


def test_config5_energy_full_size_properties(lrmd, ref, torch, inputs):
    """Rows a-E1 / a-E3 at config 5's size (N = 2^20: N^2 exceeds 2^32 here and at no smaller config).  The oracle's V
    takes 5.5e11 log terms (about ten minutes on the box's 16 cores), so at this size V is checked through properties
    ("config 5 energies"):
      (1) exact closed form: all particles placed on 5 points, cluster membership drawn per particle, so every tile
          of every kernel mixes all clusters.  Then V = (1/N) [sum_a n_a (n_a - 1) / 2 log(eps) + sum_{a<b} n_a n_b
          log(d_ab^2 + eps)] (eq.(3)): a tile visited twice, skipped, or an index wrapped at 2^32 changes
          the pair counts and with them V by far more than 1e-12 x sum |terms|.  The same formula is first checked
          against the oracle at N = 3,001, so that the formula itself is pinned by the oracle;
      (2) on the config's own input the three V kernels, which share no index arithmetic (symmetric sweep, ordered
          sweep, the band force kernel's fused V), agree within 1e-12 |V|, K equals 1/2 sum p^2 summed exactly, and the
          total energy is conserved over one step."""
    w = inputs.WORKLOADS["grav2d_1m"]
    eps = w.eps
    centres = np.array([[0.11, 0.23], [-0.52, 0.31], [0.77, -0.18], [-0.05, -0.81], [0.40, 0.66]])

    def clustered(N, seed):
        m = np.random.default_rng(seed).integers(0, len(centres), N)
        x, y = centres[m, 0].copy(), centres[m, 1].copy()
        cnt = np.bincount(m, minlength=len(centres)).astype(object)      # python ints: exact pair counts
        terms = []
        for a in range(len(centres)):
            terms.append((cnt[a] * (cnt[a] - 1) // 2, math.log(eps)))
            for b in range(a + 1, len(centres)):
                d2 = (centres[a, 0] - centres[b, 0]) ** 2 + (centres[a, 1] - centres[b, 1]) ** 2
                terms.append((cnt[a] * cnt[b], math.log(d2 + eps)))
        V = math.fsum(float(c) * t for c, t in terms) / N
        Vabs = math.fsum(float(c) * abs(t) for c, t in terms) / N
        return x, y, V, Vabs

    def gpu_energy(N, x, y, px, py, symmetric):
        ctx = lrmd.Context(GRAV2D, N, eps, options={lrmd.OPT_PAIR_SYMMETRIC: symmetric})
        ctx.set_state(x, y, px, py)
        e = ctx.energy().cpu().numpy()
        ctx.close()
        return e

    # the closed form against the oracle at a size it finishes at once
    x, y, V, Vabs = clustered(3001, 50)
    z = np.zeros_like(x)
    er, ea = ref.energy(GRAV2D, eps, x, y, z, z)
    assert abs(V - er[1]) <= 1e-13 * ea[1] and abs(Vabs - ea[1]) <= 1e-13 * ea[1]
    # (1) full size, both sweeps
    x, y, V, Vabs = clustered(w.N, 51)
    z = np.zeros_like(x)
    for symmetric in (-1, 0):
        e = gpu_energy(w.N, x, y, z, z, symmetric)
        assert abs(e[1] - V) <= 1e-12 * Vabs, (symmetric, e[1], V)
        assert e[0] == 0.0 and e[2] == 0.0 and e[3] == 0.0
    # (2) the config's own input
    x, y, px, py = w.state()
    ctx = lrmd.Context(GRAV2D, w.N, eps)
    assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 2
    ctx.set_state(x, y, px, py)
    rec = ctx.step_observe(1, w.dt, every=1).cpu().numpy()      # rec[0]: symmetric sweep at t = 0; rec[1]: fused V after the step
    ctx.set_state(*ctx.state_numpy())                            # drops the cached V: the next call sweeps
    sweep1 = ctx.energy().cpu().numpy()
    xg, yg, pxg, pyg = ctx.state_numpy()
    ctx.close()
    K0 = 0.5 * math.fsum(px * px + py * py)
    K1 = 0.5 * math.fsum(pxg * pxg + pyg * pyg)
    assert abs(rec[0, 0] - K0) <= 1e-12 * K0 and abs(rec[1, 0] - K1) <= 1e-12 * K1
    assert abs(rec[1, 1] - sweep1[1]) <= 1e-12 * abs(sweep1[1])          # fused V == symmetric sweep at the same state
    ordered0 = gpu_energy(w.N, x, y, px, py, 0)
    assert abs(ordered0[1] - rec[0, 1]) <= 1e-12 * abs(rec[0, 1])        # ordered sweep == symmetric sweep at t = 0
    E0, E1 = rec[0, 0] + rec[0, 1], rec[1, 0] + rec[1, 1]
    assert abs((E1 - E0) / E0) < 1e-8                                     # one 4th-order step, dt = 0.005


# ---- energies ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("model", [HMF, RING, GRAV2D])
@pytest.mark.parametrize("N", [1, 2, 3, 513, 4099])
def test_energy_matches_oracle(lrmd, ref, torch, model, N):
    eps = _eps(model)
    st = _state(model, N, 200 + N)
    q0, q1 = _q(model, st)
    p0, p1 = _p(model, st)
    e_ref, e_abs = ref.energy(model, eps, q0, q1, p0, p1, form=(1 if model == HMF else 0))
    ctx = lrmd.Context(model, N, eps)
    ctx.set_state(*st)
    e = ctx.energy().cpu().numpy()
    ctx.close()
    assert abs(e[0] - e_ref[0]) <= 1e-12 * e_abs[0] + 1e-300
    assert abs(e[1] - e_ref[1]) <= 1e-12 * max(e_abs[1], 0.5 * N if model == HMF else 0.0) + 1e-300
    assert abs(e[2] - e_ref[2]) <= 1e-12 * max(1.0, np.sum(np.abs(p0)))
    assert abs(e[3] - e_ref[3]) <= 1e-12 * max(1.0, np.sum(np.abs(p1)) if p1 is not None else 1.0)


@pytest.mark.parametrize("S", [1, 5, 333])
@pytest.mark.parametrize("symmetric", [0, 1])
def test_energy_any_partition(lrmd, ref, torch, S, symmetric):
    """Potential energy with any number of CTAs (ordered pair_energy_kernel, LRMD_OPT_PAIR_SYMMETRIC pinned to 0) or
    workers (symmetric twin)."""
    for model in (RING, GRAV2D):
        eps = _eps(model)
        st = _state(model, 3000, 41)
        q0, q1 = _q(model, st)
        p0, p1 = _p(model, st)
        e_ref, e_abs = ref.energy(model, eps, q0, q1, p0, p1)
        ctx = lrmd.Context(model, 3000, eps, options={lrmd.OPT_PAIR_CTAS: S, lrmd.OPT_PAIR_SYMMETRIC: symmetric})
        assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == symmetric
        ctx.set_state(*st)
        e = ctx.energy().cpu().numpy()
        ctx.close()
        assert abs(e[1] - e_ref[1]) <= 1e-12 * e_abs[1]


@pytest.mark.parametrize("model", [RING, GRAV2D])
@pytest.mark.parametrize("variant", [0, 1, 2])
@pytest.mark.parametrize("ctas", [0, 3, 148, 1000])
def test_ordered_energy_kernel_multi_tile_multi_cta(lrmd, ref, torch, model, variant, ctas):
    """The ordered pair_energy_kernel in the shapes a sharded context or an N > 8e6 context takes: N = 5,003 spans
    several i-tiles and ~20 j-tiles of every PairCfg, with one CTA range crossing tile boundaries (ctas = 3), one
    wave (148) and more CTAs than i-tiles (1000); the j = i mask sits in a different j-tile for every i-tile."""
    eps = _eps(model)
    N = 5003
    st = _state(model, N, 4100 + variant)
    q0, q1 = _q(model, st)
    p0, p1 = _p(model, st)
    e_ref, e_abs = ref.energy(model, eps, q0, q1, p0, p1)
    ctx = lrmd.Context(model, N, eps, options={lrmd.OPT_PAIR_SYMMETRIC: 0, lrmd.OPT_PAIR_VARIANT: variant,
                                                lrmd.OPT_PAIR_CTAS: ctas})
    assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 0 and ctx.get_option(lrmd.OPT_PAIR_VARIANT) == variant
    ctx.set_state(*st)
    e = ctx.energy().cpu().numpy()
    e2 = ctx.energy().cpu().numpy()
    ctx.close()
    assert abs(e[1] - e_ref[1]) <= 1e-12 * e_abs[1], (e[1], e_ref[1])
    assert abs(e[0] - e_ref[0]) <= 1e-12 * e_abs[0]
    assert np.array_equal(e, e2)


@pytest.mark.parametrize("model", [RING, GRAV2D])
@pytest.mark.parametrize("N", [2047, 2048])
def test_pair_default_path_switch(lrmd, ref, torch, model, N):
    """Either side of the default-kernel switch (ordered below N = 2048, symmetric from there): default options,
    forces, energy and a 3-step trajectory against the oracle."""
    eps = _eps(model)
    st = _state(model, N, 2040 + N)
    q0, q1 = _q(model, st)
    p0, p1 = _p(model, st)
    f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=0)
    e_ref, e_abs = ref.energy(model, eps, q0, q1, p0, p1)
    ctx = lrmd.Context(model, N, eps)
    assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == (1 if N >= 2048 else 0)
    ctx.set_state(*st)
    f = ctx.forces()
    got = tuple(t.cpu().numpy() for t in f) if model == GRAV2D else (f.cpu().numpy(), None)
    _check_forces(model, got, (f0, f1), (A0, A1))
    e = ctx.energy().cpu().numpy()
    assert abs(e[1] - e_ref[1]) <= 1e-12 * e_abs[1] and abs(e[0] - e_ref[0]) <= 1e-12 * e_abs[0]
    ctx.step(3, 0.01)
    out = ctx.state_numpy()
    ctx.close()
    r = [a.copy() for a in st]
    ref.step(model, eps, *_q(model, r), *_p(model, r), 3, 0.01, form=1)
    for g, w in zip(out, r):
        assert np.max(np.abs(g - w)) <= XTOL


@pytest.mark.parametrize("N", [1_070_335, 1_070_336, 1_070_337])
def test_hmf_default_path_switch(lrmd, ref, torch, N):
    """Either side of the HMF default-kernel switch at N = 1,070,336 = 148 x 7232 (grid-resident kernel while the state
    fits the shared memory of one CTA per SM, TMA-staged persistent kernel beyond), default options: forces at t = 0, a 10-step trajectory (9 steady
    steps: one graph replay of 8 below the switch), forces and energies at the end, against the oracle."""
    st = _state(HMF, N, 1_000 + N % 7)
    ctx = lrmd.Context(HMF, N, 0.0)
    assert ctx.get_option(lrmd.OPT_HMF_VARIANT) == (1 if N > 1_070_336 else 4)
    assert ctx.get_option(lrmd.OPT_GRAPH) == (1 if N > 1_070_336 else 0)      # substage kernels: graph replay of 8 steps
    ctx.set_state(*st)
    f = ctx.forces().cpu().numpy()
    _check_hmf_forces(ref, st[0], f, N)
    ctx.step(10, 0.05)
    out = ctx.state_numpy()
    f = ctx.forces().cpu().numpy()
    e = ctx.energy().cpu().numpy()
    ctx.close()
    th, p = st[0].copy(), st[1].copy()
    ref.step(HMF, 0.0, th, None, p, None, 10, 0.05, form=0)
    assert np.max(np.abs(out[0] - th)) <= XTOL and np.max(np.abs(out[1] - p)) <= XTOL
    _check_hmf_forces(ref, out[0], f, N)
    er, ea = ref.energy(HMF, 0.0, out[0], None, out[1], None)
    assert abs(e[0] - er[0]) <= 1e-12 * ea[0] and abs(e[1] - er[1]) <= 1e-12 * max(ea[1], 0.5 * N)


# ---- symmetric (Newton's third law) force kernel ---------------------

@pytest.mark.parametrize("model", [RING, GRAV2D])
@pytest.mark.parametrize("N", [1, 2, 3, 31, 32, 33, 127, 128, 129, 255, 257, 1000, 4099, 10_007])
@pytest.mark.parametrize("variant", [0, 1])
def test_symmetric_force_kernel_matches_oracle(lrmd, ref, torch, model, N, variant):
    """Every unordered pair once, +f / -f to both particles; i-tiles of 128 (variant 0) or 256 (variant 1) rows,
    ragged last tile and last chunk, any number of workers."""
    eps = _eps(model)
    st = _state(model, N, 4000 + N)
    q0, q1 = _q(model, st)
    f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=0)
    for workers in (0, 1, 5, 1000):
        opts = {lrmd.OPT_PAIR_SYMMETRIC: 1, lrmd.OPT_PAIR_VARIANT: variant, lrmd.OPT_PAIR_CTAS: workers}
        ctx = lrmd.Context(model, N, eps, options=opts)
        assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 1
        ctx.set_state(*st)
        f = ctx.forces()
        got = tuple(t.cpu().numpy() for t in f) if model == GRAV2D else (f.cpu().numpy(), None)
        ctx.close()
        _check_forces(model, got, (f0, f1), (A0, A1))


@pytest.mark.parametrize("model", [RING, GRAV2D])
@pytest.mark.parametrize("tiles", [1, 3, 7])
def test_symmetric_kernel_in_batches_of_tiles(lrmd, ref, torch, model, tiles):
    """Several launches per force evaluation (the j-side scratch rows of one launch are bounded): each batch's
    fold adds to the force row in tile order."""
    eps = _eps(model)
    N = 3001
    st = _state(model, N, 4242)
    q0, q1 = _q(model, st)
    f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=0)
    ctx = lrmd.Context(model, N, eps, options={lrmd.OPT_PAIR_SYMMETRIC: 1, lrmd.OPT_PAIR_SYM_TILES: tiles})
    assert ctx.get_option(lrmd.OPT_PAIR_SYM_TILES) == tiles
    ctx.set_state(*st)
    f = ctx.forces()
    got = tuple(t.cpu().numpy() for t in f) if model == GRAV2D else (f.cpu().numpy(), None)
    _check_forces(model, got, (f0, f1), (A0, A1))
    ctx.step(4, 0.01)
    out = ctx.state_numpy()
    ctx.close()
    r = [a.copy() for a in st]
    rq0, rq1 = _q(model, r)
    rp0, rp1 = _p(model, r)
    ref.step(model, eps, rq0, rq1, rp0, rp1, 4, 0.01, form=1)
    for g, w in zip(out, r):
        assert np.max(np.abs(g - w)) <= XTOL


@pytest.mark.parametrize("model", [RING, GRAV2D])
def test_symmetric_kernel_trajectory_momentum_and_reproducibility(lrmd, ref, torch, model):
    eps = _eps(model)
    N = 5001
    st = _state(model, N, 88)
    outs = []
    for _ in range(2):
        ctx = lrmd.Context(model, N, eps, options={lrmd.OPT_PAIR_SYMMETRIC: 1})
        ctx.set_state(*st)
        ctx.step(10, 0.01)
        outs.append(ctx.state_numpy())
        ctx.close()
    for x, y in zip(*outs):
        assert np.array_equal(x, y)
    r = [a.copy() for a in st]
    q0, q1 = _q(model, r)
    p0, p1 = _p(model, r)
    ref.step(model, eps, q0, q1, p0, p1, 10, 0.01, form=1)
    for g, w in zip(outs[0], r):
        assert np.max(np.abs(g - w)) <= XTOL
    pk = (2, 3) if model == GRAV2D else (1,)
    for k in pk:     # antisymmetric pair forces: total momentum conserved to rounding
        assert abs(math.fsum(outs[0][k]) - math.fsum(st[k])) <= 1e-13 * math.fsum(np.abs(st[k]))


def test_symmetric_default_choice(lrmd, torch):
    a = lrmd.Context(RING, 16_384, 0.01)
    b = lrmd.Context(GRAV2D, 65_536, 1e-3)
    c = lrmd.Context(GRAV2D, 1_048_576, 1e-3)
    d = lrmd.Context(GRAV2D, 65_536, 1e-3, options={lrmd.OPT_PAIR_SYMMETRIC: 0})
    e = lrmd.Context(GRAV2D, 1000, 1e-3)
    b1 = lrmd.Context(GRAV2D, 65_536, 1e-3, options={lrmd.OPT_PAIR_SYMMETRIC: 1})
    c1 = lrmd.Context(GRAV2D, 1_048_576, 1e-3, options={lrmd.OPT_PAIR_PRECISION: 1})
    # 2048 <= N < 49,152: warp-level symmetric kernel; beyond: band kernel (one launch, any N)
    assert a.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 1 and b.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 2
    assert c.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 2 and c.get_option(lrmd.OPT_PAIR_FUSE_UPDATE) == 1
    assert b1.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 1
    assert b1.get_option(lrmd.OPT_PAIR_SYM_TILES) == 256    # all 256 tiles in one launch (268 MB of j-side rows)
    # fp32 pair arithmetic (2D) has its own band kernel; the warp-level one would take 64 launches of 64 tiles here
    assert c1.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 2
    c2 = lrmd.Context(GRAV2D, 1_048_576, 1e-3, options={lrmd.OPT_PAIR_PRECISION: 1, lrmd.OPT_PAIR_SYMMETRIC: 1})
    assert c2.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 1 and c2.get_option(lrmd.OPT_PAIR_SYM_TILES) == 64
    c2.close()
    assert d.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 0 and e.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 0
    for x in (a, b, c, d, e, b1, c1):
        x.close()


@pytest.mark.parametrize("model", [RING, GRAV2D])
@pytest.mark.parametrize("N", [2, 33, 257, 1000, 4099, 10_007])
def test_symmetric_energy_kernel_matches_oracle(lrmd, ref, torch, model, N):
    """V from the symmetric walk (every unordered pair once, j > i inside a tile's own chunks), in one and in
    several launches, both tile sizes."""
    eps = _eps(model)
    st = _state(model, N, 5000 + N)
    q0, q1 = _q(model, st)
    p0, p1 = _p(model, st)
    e_ref, e_abs = ref.energy(model, eps, q0, q1, p0, p1)
    for opts in ({lrmd.OPT_PAIR_VARIANT: 0}, {lrmd.OPT_PAIR_VARIANT: 1}, {lrmd.OPT_PAIR_SYM_TILES: 2, lrmd.OPT_PAIR_CTAS: 5}):
        ctx = lrmd.Context(model, N, eps, options={lrmd.OPT_PAIR_SYMMETRIC: 1, **opts})
        ctx.set_state(*st)
        e = ctx.energy().cpu().numpy()
        e2 = ctx.energy().cpu().numpy()
        ctx.close()
        assert abs(e[1] - e_ref[1]) <= 1e-12 * e_abs[1] + 1e-300, (opts, e[1], e_ref[1])
        assert abs(e[0] - e_ref[0]) <= 1e-12 * e_abs[0] + 1e-300
        assert np.array_equal(e, e2)


# ---- fp32 pair arithmetic -----------------------------------------

F32TOL = 1e-5    # north_star: 1e-5 * sum_j |f_ij| for the fp32 variant


@pytest.mark.parametrize("N", [1, 2, 3, 255, 257, 1023, 4099, 20_011])
@pytest.mark.parametrize("variant", [0, 1, 2])
def test_f32_pair_variant_forces(lrmd, ref, torch, N, variant):
    """2D forces with fp32 pair terms summed in fp32 over <= 32 j, then in fp64 (reading G16), against the
    fp64 oracle; odd j-range boundaries exercise the 16-byte alignment of the fp32 tile copies."""
    st = _state(GRAV2D, N, 900 + N % 13)
    f0, f1, A0, A1 = ref.forces_abs(GRAV2D, 1e-3, st[0], st[1], form=0)
    for sym in (0, 1):          # every ordered pair (PAPER.md:110 as is) / every unordered pair once (N1 + N4)
        for ctas in (0, 7):
            if sym and variant == 2:
                continue
            got = _gpu_forces(lrmd, GRAV2D, 1e-3, st, options={lrmd.OPT_PAIR_PRECISION: 1, lrmd.OPT_PAIR_VARIANT: variant,
                                                              lrmd.OPT_PAIR_CTAS: ctas, lrmd.OPT_PAIR_SYMMETRIC: sym})
            for g, w, a in ((got[0], f0, A0), (got[1], f1, A1)):
                err = np.abs(g - w)
                assert np.all(err <= F32TOL * a + 1e-300), (sym, float((err / np.maximum(a, 1e-300)).max()))


def test_f32_pair_variant_is_not_the_fp64_path_and_is_reproducible(lrmd, ref, torch):
    N = 6000
    st = _state(GRAV2D, N, 4)
    a = _gpu_forces(lrmd, GRAV2D, 1e-3, st, options={lrmd.OPT_PAIR_PRECISION: 1})
    b = _gpu_forces(lrmd, GRAV2D, 1e-3, st, options={lrmd.OPT_PAIR_PRECISION: 1})
    c = _gpu_forces(lrmd, GRAV2D, 1e-3, st)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    rel = np.max(np.abs(a[0] - c[0])) / np.max(np.abs(c[0]))
    assert 1e-12 < rel < 1e-5       # differs from fp64 at the fp32 level, not more


def test_f32_pair_variant_trajectory_and_energy(lrmd, ref, torch):
    """10 steps with fp32 pair forces stay within 1e-6 of the fp64 oracle trajectory; the energies
    (always fp64 kernels) match the oracle evaluated at the GPU's own final state."""
    N = 3001
    st = _state(GRAV2D, N, 21)
    ctx = lrmd.Context(GRAV2D, N, 1e-3, options={lrmd.OPT_PAIR_PRECISION: 1})
    ctx.set_state(*st)
    ctx.step(10, 0.005)
    got = ctx.state_numpy()
    e = ctx.energy().cpu().numpy()
    ctx.close()
    r = [a.copy() for a in st]
    ref.step(GRAV2D, 1e-3, r[0], r[1], r[2], r[3], 10, 0.005, form=1)
    for g, w in zip(got, r):
        assert np.max(np.abs(g - w)) <= 1e-6
    er, ea = ref.energy(GRAV2D, 1e-3, got[0], got[1], got[2], got[3])
    assert abs(e[0] - er[0]) <= 1e-12 * ea[0] and abs(e[1] - er[1]) <= 1e-12 * ea[1]


@pytest.mark.parametrize("eps", [1e-2, 1e-3])
@pytest.mark.parametrize("N", [1, 2, 3, 257, 1023, 4099, 16_384])
def test_ring_f32_pair_variant_forces(lrmd, ref, torch, N, eps):
    """Ring with fp32 pair arithmetic, half-angle form: 1e-5 A_i at eps = 0.01 and 1e-3,
    on the waterbag of config 2 and on angles over the full circle (paper-shaped)."""
    for seed, full_circle in ((900 + N % 13, False), (901 + N % 13, True)):
        st = _state(RING, N, seed)
        if full_circle:
            st[0] = np.random.default_rng(seed).uniform(-math.pi, math.pi, N)
        f0, _, A0, _ = ref.forces_abs(RING, eps, st[0], None, form=0)
        for variant, ctas in ((0, 0), (1, 7), (2, 0)):
            ctx = lrmd.Context(RING, N, eps, options={lrmd.OPT_PAIR_PRECISION: 1, lrmd.OPT_PAIR_VARIANT: variant,
                                                       lrmd.OPT_PAIR_CTAS: ctas})
            assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 0 and ctx.get_option(lrmd.OPT_PAIR_PRECISION) == 1
            ctx.set_state(*st)
            g = ctx.forces().cpu().numpy()
            ctx.close()
            err = np.abs(g - f0)
            assert np.all(err <= F32TOL * A0 + 1e-300), (eps, full_circle, float((err / np.maximum(A0, 1e-300)).max()))
    if N == 1:
        assert g[0] == 0.0          # j = i contributes exactly 0


def test_ring_f32_pair_variant_trajectory_energy_and_reproducibility(lrmd, ref, torch):
    N = 3001
    st = _state(RING, N, 23)
    outs = []
    for _ in range(2):
        ctx = lrmd.Context(RING, N, 0.01, options={lrmd.OPT_PAIR_PRECISION: 1})
        ctx.set_state(*st)
        ctx.step(10, 0.01)
        outs.append(ctx.state_numpy())
        e = ctx.energy().cpu().numpy()
        ctx.close()
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    r = [a.copy() for a in st]
    ref.step(RING, 0.01, r[0], None, r[1], None, 10, 0.01, form=1)
    for g, w in zip(outs[0], r):
        assert np.max(np.abs(g - w)) <= 1e-6
    er, ea = ref.energy(RING, 0.01, outs[0][0], None, outs[0][1], None)
    assert abs(e[0] - er[0]) <= 1e-12 * ea[0] and abs(e[1] - er[1]) <= 1e-12 * ea[1]
    c = lrmd.Context(RING, N, 0.01)
    c.set_state(*st)
    f64 = c.forces().cpu().numpy()
    c.close()
    c = lrmd.Context(RING, N, 0.01, options={lrmd.OPT_PAIR_PRECISION: 1})
    c.set_state(*st)
    f32 = c.forces().cpu().numpy()
    c.close()
    rel = np.max(np.abs(f32 - f64)) / np.max(np.abs(f64))
    assert 1e-12 < rel < 1e-5       # differs from fp64 at the fp32 level, not more


# ---- integrator properties on the GPU ---------------------------------------------------------------

@pytest.mark.parametrize("model", [HMF, RING, GRAV2D])
def test_trajectory_small_ragged(lrmd, ref, torch, model):
    eps = _eps(model)
    N = 1337
    st = _state(model, N, 12)
    ctx = lrmd.Context(model, N, eps)
    ctx.set_state(*st)
    ctx.step(10, 0.01)
    got = ctx.state_numpy()
    ctx.close()
    q0, q1 = _q(model, st)
    p0, p1 = _p(model, st)
    ref.step(model, eps, q0, q1, p0, p1, 10, 0.01, form=(0 if model == HMF else 1))
    for g, r in zip(got, st):
        assert np.max(np.abs(g - r)) <= XTOL


@pytest.mark.parametrize("model", [HMF, RING, GRAV2D])
@pytest.mark.parametrize("graph", [0, 1])
def test_n_steps_equals_n_single_steps_bitwise(lrmd, torch, model, graph):
    """Force reuse (reading G3) and the merged closing+opening kick: step(n) == n x step(1), bit for bit;
    with and without CUDA-graph replay."""
    eps = _eps(model)
    N = 3001
    st = _state(model, N, 8)
    a = lrmd.Context(model, N, eps, options={lrmd.OPT_GRAPH: graph})
    a.set_state(*st)
    a.step(20, 0.01)
    b = lrmd.Context(model, N, eps, options={lrmd.OPT_GRAPH: 0})
    b.set_state(*st)
    for _ in range(20):
        b.step(1, 0.01)
    for x, y in zip(a.state_numpy(), b.state_numpy()):
        assert np.array_equal(x, y)
    a.close(); b.close()


@pytest.mark.parametrize("model", [HMF, RING, GRAV2D])
def test_bitwise_reproducible_run_to_run(lrmd, torch, model):
    eps = _eps(model)
    N = 20_011
    st = _state(model, N, 99)
    outs = []
    for _ in range(2):
        ctx = lrmd.Context(model, N, eps)
        ctx.set_state(*st)
        ctx.step(3, 0.01)
        e = ctx.energy().cpu().numpy()
        outs.append(tuple(ctx.state_numpy()) + (e,))
        ctx.close()
    for x, y in zip(*outs):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("model", [HMF, RING, GRAV2D])
def test_time_reversibility_and_momentum_on_gpu(lrmd, torch, model):
    """PAPER.md:52 'The approximation in eq. (4) is time reversible'; sum_i f_i = 0."""
    eps = _eps(model)
    N = 2048
    st = _state(model, N, 15)
    ctx = lrmd.Context(model, N, eps)
    ctx.set_state(*st)
    ctx.step(50, 0.01)
    mid = ctx.state_numpy()
    assert np.max(np.abs(mid[0] - st[0])) > 1e-3
    pk = (2, 3) if model == GRAV2D else (1,)
    scale = math.fsum(np.abs(mid[pk[0]]))
    for k in pk:
        assert abs(math.fsum(mid[k]) - math.fsum(st[k])) <= 1e-13 * scale
    if model == GRAV2D:   # angular momentum
        L0 = math.fsum(st[0] * st[3] - st[1] * st[2])
        L1 = math.fsum(mid[0] * mid[3] - mid[1] * mid[2])
        assert abs(L1 - L0) <= 1e-13 * scale
    ctx.step(50, -0.01)
    back = ctx.state_numpy()
    ctx.close()
    for g, r in zip(back, st):
        assert np.max(np.abs(g - r)) < 1e-11


def test_long_run_energy_error_same_order_as_oracle(lrmd, ref, torch, inputs):
    """Config 1 in full (1,000 steps, N = 1e4): max_t |(E - E0)/E0| sampled every 50 steps, GPU vs oracle
    ('of the same order of magnitude as for the CPU code')."""
    w = inputs.WORKLOADS["hmf_1e4"]
    th, p = w.state()
    ctx = lrmd.Context(HMF, w.N)
    ctx.set_state(th, p)
    rth, rp = th.copy(), p.copy()
    e = ctx.energy().cpu().numpy()
    E0g = e[0] + e[1]
    er, _ = ref.energy(HMF, 0.0, rth, None, rp, None)
    E0r = er[0] + er[1]
    worst_g = worst_r = 0.0
    f0 = None
    for k in range(w.steps // 50):
        ctx.step(50, w.dt)
        e = ctx.energy().cpu().numpy()
        worst_g = max(worst_g, abs((e[0] + e[1] - E0g) / E0g))
        f0, _ = ref.step(HMF, 0.0, rth, None, rp, None, 50, w.dt, f0, None, force_valid=(k > 0))
        er, _ = ref.energy(HMF, 0.0, rth, None, rp, None)
        worst_r = max(worst_r, abs((er[0] + er[1] - E0r) / E0r))
    ctx.close()
    assert worst_r > 0 and 0.1 <= worst_g / worst_r <= 10.0, (worst_g, worst_r)
    assert worst_g < 1e-6


@pytest.mark.parametrize("key,steps,ref_steps", [("ring_16k", 100, 100), ("grav2d_64k", 50, 20)])
def test_pair_models_energy_error_level(lrmd, ref, torch, inputs, key, steps, ref_steps):
    """Configs 2 and 3 in full on the GPU against the oracle stepped alongside ('relative error in
    the total energy ... same order of magnitude as for the CPU code'): max_t |(E - E0)/E0| sampled every 10 steps
    over the WHOLE run of config 2 (100 steps) and over the first 20 of config 3's 50 steps, GPU and oracle within a
    factor 10 of each other at every sample and in the maximum; the GPU run is completed and stays at that level."""
    w = inputs.WORKLOADS[key]
    st = w.state()
    ctx = lrmd.Context(w.model, w.N, w.eps)
    ctx.set_state(*st)
    rec = ctx.step_observe(steps, w.dt, 10).cpu().numpy()          # K, V at steps 0, 10, 20, ...
    ctx.close()
    Eg = rec[:, 0] + rec[:, 1]
    err_g = np.abs((Eg - Eg[0]) / Eg[0])
    rs = [a.copy() for a in st]
    q0, q1 = _q(w.model, rs)
    p0, p1 = _p(w.model, rs)
    er0, _ = ref.energy(w.model, w.eps, q0, q1, p0, p1)
    E0r = er0[0] + er0[1]
    assert abs(Eg[0] - E0r) <= 1e-11 * abs(E0r)
    err_r = [0.0]
    f0 = f1 = None
    for k in range(ref_steps // 10):
        f0, f1 = ref.step(w.model, w.eps, q0, q1, p0, p1, 10, w.dt, f0, f1, force_valid=(k > 0), form=1)
        er, _ = ref.energy(w.model, w.eps, q0, q1, p0, p1)
        err_r.append(abs((er[0] + er[1] - E0r) / E0r))
    err_r = np.array(err_r)
    for k in range(1, len(err_r)):
        a, b = max(err_g[k], 1e-15), max(err_r[k], 1e-15)
        assert 0.1 <= a / b <= 10.0, (k, err_g[k], err_r[k])
    n = len(err_r)
    assert 0.1 <= max(err_g[1:n].max(), 1e-15) / max(err_r[1:].max(), 1e-15) <= 10.0
    assert err_g.max() < 1e-5 and err_g.max() <= 10.0 * max(err_r.max(), 1e-12)


# ---- the end-to-end entry point and error paths -------------------------------------------------------

@pytest.mark.parametrize("model", [HMF, RING, GRAV2D])
def test_step_host_equals_step(lrmd, torch, model):
    eps = _eps(model)
    N = 5000
    st = _state(model, N, 2)
    a = lrmd.Context(model, N, eps)
    a.set_state(*st)
    a.step(4, 0.01)
    b = lrmd.Context(model, N, eps)
    b.set_state(*[np.zeros(N) for _ in st])
    host = [torch.from_numpy(x.copy()).pin_memory() for x in st]
    b.step_host(host, 4, 0.01)
    for x, y in zip(a.state_numpy(), host):
        assert np.array_equal(x, y.numpy())
    a.close(); b.close()


def test_set_state_invalidates_cached_force(lrmd, ref, torch):
    N = 700
    st = _state(RING, N, 1)
    ctx = lrmd.Context(RING, N, 0.01)
    ctx.set_state(*st)
    f_a = ctx.forces().cpu().numpy()
    st2 = _state(RING, N, 2)
    ctx.set_state(*st2)
    f_b = ctx.forces().cpu().numpy()
    ctx.close()
    want = ref.forces(RING, 0.01, st2[0], form=0)
    assert np.max(np.abs(f_b - want)) < 1e-10 and np.max(np.abs(f_a - f_b)) > 1e-3


def test_negative_n_and_nonfinite_dt_rejected(lrmd, torch):
    ctx = lrmd.Context(HMF, 100)
    ctx.set_state(*_state(HMF, 100, 0))
    with pytest.raises(lrmd.LrmdError):
        ctx.step(-1, 0.1)
    with pytest.raises(lrmd.LrmdError):
        ctx.step(1, float("nan"))
    before = ctx.state_numpy()
    ctx.step(0, 0.1)
    assert all(np.array_equal(a, b) for a, b in zip(before, ctx.state_numpy()))
    ctx.close()


# ---- per-step observables and paper-shaped runs (Figs. 3-6) --------------

@pytest.mark.parametrize("model", [HMF, RING, GRAV2D])
def test_step_observe_records_match_oracle(lrmd, ref, torch, model):
    """lrmd_step_observe: K(t), V(t) records every 3 steps against the oracle stepped alongside."""
    eps = _eps(model)
    N = 1500
    st = _state(model, N, 61)
    ctx = lrmd.Context(model, N, eps)
    ctx.set_state(*st)
    rec = ctx.step_observe(10, 0.01, 3).cpu().numpy()          # records at steps 0, 3, 6, 9; 10 steps taken
    fin = ctx.state_numpy()
    ctx.close()
    assert rec.shape == (4, 4)
    r = [a.copy() for a in st]
    q0, q1 = _q(model, r)
    p0, p1 = _p(model, r)
    f0 = f1 = None
    for k in range(4):
        er, ea = ref.energy(model, eps, q0, q1, p0, p1)
        assert abs(rec[k, 0] - er[0]) <= 1e-9 * max(ea[0], 1e-300) and abs(rec[k, 1] - er[1]) <= 1e-9 * max(ea[1], 0.5 * N)
        f0, f1 = ref.step(model, eps, q0, q1, p0, p1, 3 if k < 3 else 1, 0.01, f0, f1, force_valid=(k > 0), form=(0 if model == HMF else 1))
    for g, w in zip(fin, r):
        assert np.max(np.abs(g - w)) <= XTOL


def test_paper_shaped_runs_conserve_energy(lrmd, torch):
    """homogeneous state at rest (HMF dt = 0.1; Ring eps = 1e-3, dt = 0.005) and the 2D annulus
    1.0 <= r <= 1.5 at rest: K starts at 0, grows as the system collapses / relaxes, the relative energy
    error stays at the 4th-order level."""
    from paper_1212_0262_b200 import paper_runs
    for name, n, tol in (("hmf", 20_000, 1e-5), ("ring", 4096, 1e-4), ("grav2d", 4096, 1e-6)):
        out = paper_runs.run(name, n, steps=60, every=10)
        assert out["K"][0] == 0.0 and len(out["K"]) == 7
        assert out["K"][-1] > 0.0
        assert max(out["energy_error"]) < tol, (name, max(out["energy_error"]))


@pytest.mark.parametrize("name,symmetric", [("hmf", -1), ("ring", 0), ("ring", 1), ("ring", 2), ("grav2d", 0), ("grav2d", 1),
                                            ("grav2d", 2)])
def test_paper_shaped_runs_match_oracle(lrmd, ref, torch, name, symmetric):
    """The set-ups of the paper's section 4 against the oracle, not just energy conservation:
    homogeneous state at rest on the full circle [-pi, pi) (HMF dt = 0.1; Ring eps = 1e-3, dt = 0.005 — where the
    cancellation of eq.(9)'s denominator is strongest) and the 2D annulus 1.0 <= r <= 1.5 at rest (eps = 1e-3,
    dt = 0.005): forces at t = 0 within 1e-12 A_i, state within 1e-9 after 10 steps, K and V records every 5 steps."""
    from paper_1212_0262_b200 import paper_runs
    su = paper_runs.SETUPS[name]
    model, eps, dt = su["model"], su["eps"], su["dt"]
    N = 4099 if model != HMF else 10_007
    st = [np.array(a, dtype=np.float64) for a in paper_runs.initial_state(name, N)]
    opts = {} if model == HMF else {lrmd.OPT_PAIR_SYMMETRIC: symmetric}
    ctx = lrmd.Context(model, N, eps, options=opts or None)
    ctx.set_state(*st)
    f = ctx.forces()
    got = tuple(t.cpu().numpy() for t in f) if model == GRAV2D else (f.cpu().numpy(), None)
    q0, q1 = _q(model, st)
    f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=(1 if model == HMF else 0))
    _check_forces(model, got, (f0, f1), (A0, A1))
    rec = ctx.step_observe(10, dt, 5).cpu().numpy()
    fin = ctx.state_numpy()
    ctx.close()
    r = [a.copy() for a in st]
    rq0, rq1 = _q(model, r)
    rp0, rp1 = _p(model, r)
    g0 = g1 = None
    for k in range(3):
        er, ea = ref.energy(model, eps, rq0, rq1, rp0, rp1)
        assert abs(rec[k, 0] - er[0]) <= 1e-9 * max(ea[0], 1e-12) and abs(rec[k, 1] - er[1]) <= 1e-9 * max(ea[1], 0.5 * N)
        if k < 2:
            g0, g1 = ref.step(model, eps, rq0, rq1, rp0, rp1, 5, dt, g0, g1, force_valid=(k > 0), form=(0 if model == HMF else 1))
    assert rec[0, 0] == 0.0 and rec[2, 0] > 0.0          # at rest, then collapsing / relaxing
    for g, w in zip(fin, r):
        assert np.max(np.abs(g - w)) <= XTOL


@pytest.mark.parametrize("model", [RING, GRAV2D])
def test_update_fused_into_fold_is_bit_identical(lrmd, torch, model):
    """LRMD_OPT_PAIR_FUSE_UPDATE: the kick / drift after a single-launch symmetric force evaluation runs inside the
    fold kernel; same arithmetic, so trajectories, cached forces and energies are bit-identical to the separate
    update kernel, for step(n) and for n x step(1)."""
    eps = _eps(model)
    N = 5003
    st = _state(model, N, 321)
    res = []
    for fuse, single in ((1, False), (0, False), (1, True)):
        ctx = lrmd.Context(model, N, eps, options={lrmd.OPT_PAIR_FUSE_UPDATE: fuse})
        assert ctx.get_option(lrmd.OPT_PAIR_FUSE_UPDATE) == fuse
        ctx.set_state(*st)
        if single:
            for _ in range(6):
                ctx.step(1, 0.01)
        else:
            ctx.step(6, 0.01)
        f = ctx.forces()
        f = [t.cpu().numpy() for t in f] if model == GRAV2D else [f.cpu().numpy()]
        res.append(list(ctx.state_numpy()) + f + [ctx.energy().cpu().numpy()])
        ctx.close()
    for other in res[1:]:
        for x, y in zip(res[0], other):
            assert np.array_equal(x, y)


# ---- option combinations ------------------------------------------------------------------------------------------

def test_random_option_combinations_match_oracle(lrmd, ref, torch):
    """60 seeded combinations of (model, N, kernel choice, launch shape, workers / CTAs, tiles per launch, pair
    precision): forces within tolerance of the oracle and a 2-step trajectory within 1e-9 (1e-6 with fp32 pairs)."""
    rng = np.random.default_rng(20121204)
    for case in range(60):
        model = int(rng.choice([RING, GRAV2D]))
        N = int(rng.choice([1, 2, 31, 33, 200, 257, 1000, 2047, 2048, 2500, 4097]))
        opts = {lrmd.OPT_PAIR_SYMMETRIC: int(rng.choice([-1, 0, 1])), lrmd.OPT_PAIR_VARIANT: int(rng.choice([-1, 0, 1, 2])),
                lrmd.OPT_PAIR_CTAS: int(rng.choice([0, 1, 3, 40, 700])), lrmd.OPT_PAIR_SYM_TILES: int(rng.choice([0, 1, 5]))}
        f32 = model == GRAV2D and rng.random() < 0.3
        if f32:
            opts[lrmd.OPT_PAIR_PRECISION] = 1
        eps = _eps(model)
        st = _state(model, N, 9000 + case)
        q0, q1 = _q(model, st)
        f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=0)
        ctx = lrmd.Context(model, N, eps, options=opts)
        ctx.set_state(*st)
        f = ctx.forces()
        got = tuple(t.cpu().numpy() for t in f) if model == GRAV2D else (f.cpu().numpy(), None)
        ftol = F32TOL if f32 else FTOL
        for g, w, a in zip(got, (f0, f1), (A0, A1)):
            if g is not None:
                assert np.all(np.abs(g - w) <= ftol * a + 1e-300), (case, model, N, opts)
        ctx.step(2, 0.01)
        out = ctx.state_numpy()
        ctx.close()
        r = [a.copy() for a in st]
        rq0, rq1 = _q(model, r)
        rp0, rp1 = _p(model, r)
        ref.step(model, eps, rq0, rq1, rp0, rp1, 2, 0.01, form=1)
        for g, w in zip(out, r):
            assert np.max(np.abs(g - w)) <= (1e-6 if f32 else XTOL), (case, model, N, opts)


def test_random_hmf_option_combinations_match_oracle(lrmd, ref, torch):
    """40 seeded combinations of (N, kernel variant, grid, graph replay): forces at the final angles, a 9-step
    trajectory (graph replay needs >= 8 steady-state steps) and the energies against the oracle."""
    rng = np.random.default_rng(20121205)
    for case in range(40):
        N = int(rng.choice([1, 3, 4, 1000, 2049, 20_480, 20_481, 65_537, 300_000]))
        opts = {lrmd.OPT_HMF_VARIANT: int(rng.choice([-1, 0, 1, 2, 3])), lrmd.OPT_GRAPH: int(rng.choice([-1, 0, 1])),
                lrmd.OPT_HMF_GRID: int(rng.choice([0, 0, 1, 7, 148]))}
        if opts[lrmd.OPT_HMF_VARIANT] == 3 and opts[lrmd.OPT_HMF_GRID] not in (0,):
            opts[lrmd.OPT_HMF_GRID] = 0          # the cluster-resident kernel takes 0 (8 CTAs) or 16 only
        st = _state(HMF, N, 7000 + case)
        ctx = lrmd.Context(HMF, N, 0.0, options=opts)
        ctx.set_state(*st)
        ctx.step(9, 0.05)
        out = ctx.state_numpy()
        f = ctx.forces().cpu().numpy()
        e = ctx.energy().cpu().numpy()
        ctx.close()
        th, p = st[0].copy(), st[1].copy()
        ref.step(HMF, 0.0, th, None, p, None, 9, 0.05, form=0)
        assert np.max(np.abs(out[0] - th)) <= XTOL and np.max(np.abs(out[1] - p)) <= XTOL, (case, N, opts)
        _check_hmf_forces(ref, out[0], f, (case, N, opts), nsample=256)
        er, ea = ref.energy(HMF, 0.0, out[0], None, out[1], None)
        assert abs(e[0] - er[0]) <= 1e-12 * ea[0] + 1e-300, (case, N, opts)
        assert abs(e[1] - er[1]) <= 1e-12 * max(ea[1], 0.5 * N) + 1e-300, (case, N, opts)
