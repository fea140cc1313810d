"""Parity of the band kernel (LRMD_OPT_PAIR_SYMMETRIC = 2, csrc/band_kernels.cuh: Newton's third law with both
sides' sums kept on chip, SURVEY.md 8(f) N4 / PAPER.md:108) with the oracle, through the C ABI, on the same seeded
inputs and at BASELINE.json's tolerances (forces 1e-12 A_i, trajectory 1e-9 after 10 steps)."""
import math

import numpy as np
import pytest

from test_gpu_parity import FTOL, GRAV2D, RING, XTOL, _check_forces, _eps, _p, _q, _state, torch  # noqa: F401

pytestmark = pytest.mark.gpu


def _forces(lrmd, model, N, eps, st, opts):
    ctx = lrmd.Context(model, N, eps, options=opts)
    assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 2
    ctx.set_state(*st)
    f = ctx.forces()
    got = tuple(t.cpu().numpy() for t in f) if model == GRAV2D else (f.cpu().numpy(), None)
    ctx.close()
    return got


@pytest.mark.parametrize("model", [RING, GRAV2D])
@pytest.mark.parametrize("N", [1, 2, 31, 33, 257, 1000, 1024, 1025, 2047, 2049, 4099, 10_007, 20_011])
@pytest.mark.parametrize("variant", [0, 1])
def test_band_force_kernel_matches_oracle(lrmd, ref, torch, model, N, variant):
    """I-blocks of 1024 (variant 0) or 2048 (variant 1) rows: one block, several blocks, ragged last tile, last chunk
    and last block; any number of workers (pieces shorter than 8 chunks, workers without work) and band heights."""
    eps = _eps(model)
    st = _state(model, N, 7000 + N)
    q0, q1 = _q(model, st)
    f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=0)
    for workers, height in ((0, 0), (1, 0), (5, 1), (37, 2), (1000, 3)):
        opts = {lrmd.OPT_PAIR_SYMMETRIC: 2, lrmd.OPT_PAIR_VARIANT: variant, lrmd.OPT_PAIR_CTAS: workers,
                lrmd.OPT_PAIR_BAND_HEIGHT: height}
        got = _forces(lrmd, model, N, eps, st, opts)
        _check_forces(model, got, (f0, f1), (A0, A1))


@pytest.mark.parametrize("model", [RING, GRAV2D])
def test_band_kernel_default_shape_several_bands(lrmd, ref, torch, model):
    """N = 70,001: beyond the default switch (49,152), 35 I-blocks of 2048 rows, default band height and workers;
    forces on sampled rows against the oracle (each against all N)."""
    eps = _eps(model)
    N = 70_001
    st = _state(model, N, 71)
    q0, q1 = _q(model, st)
    ctx = lrmd.Context(model, N, eps)
    assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 2
    ctx.set_state(*st)
    f = ctx.forces()
    got = tuple(t.cpu().numpy() for t in f) if model == GRAV2D else (f.cpu().numpy(), None)
    ctx.close()
    rows = np.unique(np.concatenate([np.arange(0, 300), np.arange(N - 300, N),
                                     np.random.default_rng(5).choice(N, 3000, replace=False)]))
    r0, r1, A0, A1 = ref.forces_rows(model, eps, q0, q1, rows, form=0, with_abs=True)
    _check_forces(model, tuple(None if g is None else g[rows] for g in got), (r0, r1), (A0, A1))


@pytest.mark.parametrize("model", [RING, GRAV2D])
def test_band_kernel_trajectory_momentum_and_reproducibility(lrmd, ref, torch, model):
    eps = _eps(model)
    N = 6007
    st = _state(model, N, 89)
    outs = []
    for _ in range(2):
        ctx = lrmd.Context(model, N, eps, options={lrmd.OPT_PAIR_SYMMETRIC: 2, lrmd.OPT_PAIR_BAND_HEIGHT: 2})
        ctx.set_state(*st)
        ctx.step(10, 0.01)
        outs.append(ctx.state_numpy())
        ctx.close()
    for x, y in zip(*outs):
        assert np.array_equal(x, y)          # fixed order of every sum: bitwise reproducible
    r = [a.copy() for a in st]
    q0, q1 = _q(model, r)
    p0, p1 = _p(model, r)
    ref.step(model, eps, q0, q1, p0, p1, 10, 0.01, form=1)
    for g, w in zip(outs[0], r):
        assert np.max(np.abs(g - w)) <= XTOL
    pk = (2, 3) if model == GRAV2D else (1,)
    for k in pk:     # antisymmetric pair forces: total momentum conserved to rounding
        assert abs(math.fsum(outs[0][k]) - math.fsum(st[k])) <= 1e-13 * math.fsum(np.abs(st[k]))


@pytest.mark.parametrize("model", [RING, GRAV2D])
def test_band_update_fused_into_fold_is_bit_identical(lrmd, torch, model):
    eps = _eps(model)
    N = 5003
    st = _state(model, N, 322)
    res = []
    for fuse, single in ((1, False), (0, False), (1, True)):
        ctx = lrmd.Context(model, N, eps, options={lrmd.OPT_PAIR_SYMMETRIC: 2, lrmd.OPT_PAIR_FUSE_UPDATE: fuse})
        assert ctx.get_option(lrmd.OPT_PAIR_FUSE_UPDATE) == fuse
        ctx.set_state(*st)
        if single:
            for _ in range(5):
                ctx.step(1, 0.01)
        else:
            ctx.step(5, 0.01)
        f = ctx.forces()
        f = [t.cpu().numpy() for t in f] if model == GRAV2D else [f.cpu().numpy()]
        res.append(list(ctx.state_numpy()) + f + [ctx.energy().cpu().numpy()])
        ctx.close()
    for other in res[1:]:
        for x, y in zip(res[0], other):
            assert np.array_equal(x, y)


def test_band_kernel_agrees_with_the_other_pair_kernels(lrmd, torch):
    """Same state, three kernels (ordered, warp-level symmetric, band): forces agree to rounding of the sums."""
    N = 9001
    st = _state(GRAV2D, N, 17)
    fs = []
    for sym in (0, 1, 2):
        ctx = lrmd.Context(GRAV2D, N, 1e-3, options={lrmd.OPT_PAIR_SYMMETRIC: sym})
        assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == sym
        ctx.set_state(*st)
        fs.append([t.cpu().numpy() for t in ctx.forces()])
        ctx.close()
    scale = max(np.abs(fs[0][0]).max(), np.abs(fs[0][1]).max())
    for other in fs[1:]:
        for a, b in zip(fs[0], other):
            assert np.max(np.abs(a - b)) <= 1e-11 * scale


@pytest.mark.parametrize("model", [RING, GRAV2D])
@pytest.mark.parametrize("N,height,fuse", [(1500, 0, 1), (4099, 2, 1), (2049, 1, 0), (6000, 0, 1)])
def test_band_step_observe_uses_the_fused_potential(lrmd, ref, torch, model, N, height, fuse):
    """lrmd_step_observe on a band-kernel context: the force evaluation that ends each recorded step delivers V
    (PAPER.md:61 step 12; rows a-E2 / a-E3 fused into the force kernel): one launch fewer per record than a separate
    O(N^2) sweep, records equal to the oracle's stepped alongside, state equal to plain stepping bit for bit."""
    eps = _eps(model)
    st = _state(model, N, 63 + N)
    opts = {lrmd.OPT_PAIR_SYMMETRIC: 2, lrmd.OPT_PAIR_BAND_HEIGHT: height, lrmd.OPT_PAIR_FUSE_UPDATE: fuse}
    ctx = lrmd.Context(model, N, eps, options=opts)
    ctx.set_state(*st)
    l0 = ctx.launch_count()
    rec = ctx.step_observe(7, 0.01, 2).cpu().numpy()          # records at steps 0, 2, 4, 6; 7 steps taken
    launches = ctx.launch_count() - l0
    fin = ctx.state_numpy()
    e_after = ctx.energy().cpu().numpy()                      # separate sweep at the final state
    ctx.close()
    assert rec.shape == (4, 4)
    r = [a.copy() for a in st]
    q0, q1 = _q(model, r)
    p0, p1 = _p(model, r)
    f0 = f1 = None
    for k in range(4):
        er, ea = ref.energy(model, eps, q0, q1, p0, p1)
        assert abs(rec[k, 0] - er[0]) <= 1e-9 * max(ea[0], 1e-300)
        assert abs(rec[k, 1] - er[1]) <= 1e-12 * max(ea[1], 0.5 * N), (k, rec[k, 1], er[1])
        f0, f1 = ref.step(model, eps, q0, q1, p0, p1, 2 if k < 3 else 1, 0.01, f0, f1, force_valid=(k > 0), form=1)
    for g, w in zip(fin, r):
        assert np.max(np.abs(g - w)) <= XTOL
    er, ea = ref.energy(model, eps, q0, q1, p0, p1)
    assert abs(e_after[1] - er[1]) <= 1e-12 * max(ea[1], 0.5 * N)
    # the same steps without records: identical state (the fused potential changes no force arithmetic)
    ctx = lrmd.Context(model, N, eps, options=opts)
    ctx.set_state(*st)
    l0 = ctx.launch_count()
    ctx.step(2, 0.01); ctx.step(2, 0.01); ctx.step(2, 0.01); ctx.step(1, 0.01)
    plain = ctx.launch_count() - l0
    fin2 = ctx.state_numpy()
    ctx.close()
    for x, y in zip(fin, fin2):
        assert np.array_equal(x, y)
    # per record after the first: the kinetic partial kernel and the finalize kernel only (no pair sweep); the first
    # record takes the separate sweep (pack? no: + kinetic, energy kernel, finalize)
    assert launches - plain <= 3 + 3 * 2 + 2


@pytest.mark.parametrize("N", [1, 2, 3, 255, 1023, 2049, 4099, 20_011])
@pytest.mark.parametrize("variant", [0, 1, 2])
def test_band_f32_pair_variant_forces(lrmd, ref, torch, N, variant):
    """GRAV2D, fp32 pair terms in the band kernel: 1e-5 A_i, odd N (the fp32 stream's bulk copies move an
    even number of elements), any number of workers and band heights; bitwise reproducible."""
    st = _state(GRAV2D, N, 950 + N % 13)
    f0, f1, A0, A1 = ref.forces_abs(GRAV2D, 1e-3, st[0], st[1], form=0)
    # exchange -1 / 0: the j-side fp32 packet travels by shuffles (default); 1: it joins the fp64 slot sum every step
    for workers, height, xch in ((0, 0, -1), (3, 1, 0), (37, 2, -1), (0, 0, 1), (37, 2, 1)):
        opts = {lrmd.OPT_PAIR_PRECISION: 1, lrmd.OPT_PAIR_SYMMETRIC: 2, lrmd.OPT_PAIR_VARIANT: variant,
                lrmd.OPT_PAIR_CTAS: workers, lrmd.OPT_PAIR_BAND_HEIGHT: height, lrmd.OPT_PAIR_SYM_EXCHANGE: xch}
        got = _forces(lrmd, GRAV2D, N, 1e-3, st, opts)
        again = _forces(lrmd, GRAV2D, N, 1e-3, st, opts)
        for g, h, w, a in ((got[0], again[0], f0, A0), (got[1], again[1], f1, A1)):
            assert np.array_equal(g, h)
            err = np.abs(g - w)
            assert np.all(err <= 1e-5 * a + 1e-300), float((err / np.maximum(a, 1e-300)).max())


def test_band_f32_pair_variant_trajectory(lrmd, ref, torch):
    N = 70_001          # default choice at this size with fp32 pairs: the band kernel
    st = _state(GRAV2D, N, 24)
    ctx = lrmd.Context(GRAV2D, N, 1e-3, options={lrmd.OPT_PAIR_PRECISION: 1})
    assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 2
    ctx.set_state(*st)
    ctx.step(3, 0.005)
    got = ctx.state_numpy()
    ctx.close()
    r = [a.copy() for a in st]
    ref.step(GRAV2D, 1e-3, r[0], r[1], r[2], r[3], 3, 0.005, form=1)
    for g, w in zip(got, r):
        assert np.max(np.abs(g - w)) <= 1e-6


def test_band_fused_potential_at_config3_size(lrmd, ref, torch, inputs):
    """Config 3 (N = 65,536) in the default configuration: the V that the step's last force evaluation delivers
    (lrmd_step_observe) against the oracle's pair sum at the GPU's own final state, and against the separate sweep."""
    w = inputs.WORKLOADS["grav2d_64k"]
    ctx = lrmd.Context(GRAV2D, w.N, w.eps)
    assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 2
    ctx.set_state(*w.state())
    rec = ctx.step_observe(2, w.dt, 1).cpu().numpy()
    x, y, px, py = ctx.state_numpy()
    sweep = ctx.energy().cpu().numpy()
    ctx.close()
    er, ea = ref.energy(GRAV2D, w.eps, x, y, px, py)
    assert abs(rec[2, 0] - er[0]) <= 1e-12 * ea[0] and abs(rec[2, 1] - er[1]) <= 1e-12 * ea[1]
    assert abs(sweep[1] - er[1]) <= 1e-12 * ea[1] and abs(sweep[1] - rec[2, 1]) <= 1e-12 * ea[1]


def test_ring_512k_paper_table2_size_sampled_rows(lrmd, ref, torch, inputs):
    """The largest Ring run of the paper's Table 2 (N = 512,000) in the default configuration (band
    kernel, I-blocks of 2048 rows): forces on 2,048 sampled rows, each against all N, against the oracle's direct
    eq.(8) form, at t = 0 and at the GPU's own angles after one step; total momentum conserved over the step.  (K and V
    at this size are not compared with the oracle: its O(N^2) V takes minutes here; config 2 at full size covers them.)"""
    w = inputs.TABLE23_WORKLOADS["ring_512k"]
    th, p = w.state()
    ctx = lrmd.Context(RING, w.N, w.eps)
    assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 2
    ctx.set_state(th, p)
    f = ctx.forces().cpu().numpy()
    ctx.step(1, w.dt)
    th1, p1 = ctx.state_numpy()
    f1 = ctx.forces().cpu().numpy()
    ctx.close()
    rows = np.random.default_rng(8).choice(w.N, 2048, replace=False)
    for state, got in ((th, f), (th1, f1)):
        r0, _, A0, _ = ref.forces_rows(RING, w.eps, state, None, rows, form=0, with_abs=True)
        _check_forces(RING, (got[rows], None), (r0, None), (A0, None))
    assert abs(math.fsum(p1) - math.fsum(p)) <= 1e-12 * math.fsum(np.abs(p))


def test_band_kernel_beyond_the_l2_capped_height(lrmd, ref, torch):
    """N = 3,000,001 (ragged; 2.9x config 5): the scratch rows of the L2-resident band height would pass 1 GiB, so the
    unconstrained height is used (about 1.4 GB of scratch); one launch per force evaluation; forces on sampled rows,
    each against all N, against the oracle."""
    N = 3_000_001
    st = _state(GRAV2D, N, 31)
    ctx = lrmd.Context(GRAV2D, N, 1e-3)
    assert ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) == 2 and ctx.get_option(lrmd.OPT_PAIR_BAND_HEIGHT) > 16
    assert ctx.workspace_bytes() < 2_000_000_000
    ctx.set_state(*st)
    l0 = ctx.launch_count()
    f = ctx.forces()
    assert ctx.launch_count() - l0 == 4          # pack, band kernel, fold, copy-out
    got = tuple(t.cpu().numpy() for t in f)
    ctx.close()
    rows = np.unique(np.concatenate([np.arange(0, 64), np.arange(N - 64, N), np.random.default_rng(9).choice(N, 512, replace=False)]))
    r0, r1, A0, A1 = ref.forces_rows(GRAV2D, 1e-3, st[0], st[1], rows, form=0, with_abs=True)
    _check_forces(GRAV2D, tuple(g[rows] for g in got), (r0, r1), (A0, A1))
