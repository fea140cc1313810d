"""tests/golden/oracle_small.json — values written by tests/golden/make_golden.py from the oracle only
(the paper prints no worked example to store, PAPER.md has timings and absent figures only).

CPU: the oracle still reproduces the stored values bit for bit, and the stored forces agree with a
brute-force numpy evaluation of -dH/dq written from the printed Hamiltonians.
GPU: the CUDA path matches the stored forces / energies / 10-step trajectory within north_star's
tolerances — values written by the oracle alone (tests/golden/make_golden.py calls only oracle/).
"""
import json
import os

import numpy as np
import pytest

HMF, RING, GRAV2D = 0, 1, 2
PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_small.json")


def _un(lst):
    return np.array([float.fromhex(v) for v in lst], dtype=np.float64)


def _cases():
    with open(PATH) as fh:
        return json.load(fh)["cases"]


CASE_NAMES = sorted(_cases())


def _split(model, st):
    if model == GRAV2D:
        return (st[0], st[1]), (st[2], st[3])
    return (st[0], None), (st[1], None)


@pytest.mark.parametrize("name", CASE_NAMES)
def test_oracle_reproduces_golden_bitwise(ref, name):
    c = _cases()[name]
    model, eps = c["model"], c["eps"]
    st = [_un(a) for a in c["state0"]]
    (q0, q1), (p0, p1) = _split(model, st)
    f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=0, nthreads=1)
    assert np.array_equal(f0, _un(c["forces"][0])) and np.array_equal(A0, _un(c["abs_force_sums"][0]))
    if model == GRAV2D:
        assert np.array_equal(f1, _un(c["forces"][1])) and np.array_equal(A1, _un(c["abs_force_sums"][1]))
    e, _ = ref.energy(model, eps, q0, q1, p0, p1, nthreads=1)
    assert np.array_equal(e, _un(c["energy0"]))
    fin = [a.copy() for a in st]
    (fq0, fq1), (fp0, fp1) = _split(model, fin)
    ref.step(model, eps, fq0, fq1, fp0, fp1, c["steps"], c["dt"], form=0, nthreads=1)
    for a, g in zip(fin, c["state10"]):
        assert np.array_equal(a, _un(g))


@pytest.mark.parametrize("name", CASE_NAMES)
def test_golden_forces_are_minus_grad_h_by_numpy_brute_force(name):
    """Independent of the oracle's code: the pair sums of -dH/dq from eqs.(1)-(3) in plain numpy."""
    c = _cases()[name]
    model, eps, N = c["model"], c["eps"], c["N"]
    st = [_un(a) for a in c["state0"]]
    if model == GRAV2D:
        dx = st[0][:, None] - st[0][None, :]
        dy = st[1][:, None] - st[1][None, :]
        w = 1.0 / (dx * dx + dy * dy + eps)
        np.fill_diagonal(w, 0.0)
        want = [-(2.0 / N) * (dx * w).sum(1), -(2.0 / N) * (dy * w).sum(1)]
    else:
        d = st[0][:, None] - st[0][None, :]
        if model == HMF:
            t = np.sin(d)
            pre = -1.0 / N
        else:
            t = np.sin(d) / (1.0 - np.cos(d) + eps) ** 1.5
            pre = -1.0 / (2.0 * np.sqrt(2.0) * N)
        np.fill_diagonal(t, 0.0)
        want = [pre * t.sum(1)]
    for w_, g, A in zip(want, c["forces"], c["abs_force_sums"]):
        assert np.all(np.abs(w_ - _un(g)) <= 1e-13 * _un(A) + 1e-16)


@pytest.mark.gpu
@pytest.mark.parametrize("name", CASE_NAMES)
def test_cuda_path_matches_golden(lrmd, name):
    c = _cases()[name]
    model, eps, N = c["model"], c["eps"], c["N"]
    st = [_un(a) for a in c["state0"]]
    ctx = lrmd.Context(model, N, eps)
    ctx.set_state(*st)
    f = ctx.forces()
    got = [t.cpu().numpy() for t in f] if model == GRAV2D else [f.cpu().numpy()]
    for g, w, A in zip(got, c["forces"], c["abs_force_sums"]):
        assert np.all(np.abs(g - _un(w)) <= 1e-12 * _un(A) + 4e-16)
    e = ctx.energy().cpu().numpy()
    ea = _un(c["energy0_abs"])
    e0 = _un(c["energy0"])
    assert abs(e[0] - e0[0]) <= 1e-12 * ea[0] and abs(e[1] - e0[1]) <= 1e-12 * max(ea[1], 0.5 * N if model == HMF else 0.0)
    ctx.step(c["steps"], c["dt"])
    for g, w in zip(ctx.state_numpy(), c["state10"]):
        assert np.max(np.abs(g - _un(w))) <= 1e-9
    e10 = ctx.energy().cpu().numpy()
    w10 = _un(c["energy10"])
    assert abs((e10[0] + e10[1]) - (w10[0] + w10[1])) <= 1e-9 * max(1.0, abs(w10[0]) + abs(w10[1]))
    ctx.close()
