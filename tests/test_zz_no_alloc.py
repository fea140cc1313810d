"""lrmd_hmf_forces_static: HMF forces for callers that cannot provide scratch memory.

Who needs it: code that runs where device memory cannot be allocated — a plug-in inside an application that took all
of HBM for its own pool and passes only input and output pointers, or a routine in a latency-critical loop where
cudaMalloc / cudaFree (which stall the whole device) are forbidden.  Such callers cannot create the workspace that
lrmd_set_workspace wants, so the library keeps this one call's scratch (per-CTA cos / sin sums) in a 64 KiB array
that is part of the library image.  The price is a size limit (N <= LRMD_STATIC_MAX_N) and one array shared by all
calls in the process.

What is checked here: the call gives the same forces as the existing path (a Context with a caller-allocated
workspace, lrmd_forces) within the force tolerance of the other GPU tests (1e-12 * A_i, A_i = sum_j |f_ij| from the
oracle, plus the same 4e-16 floor as test_gpu_parity.py), on two calls in a row that reuse the shared array — the
second with a SMALLER N, so that stale sums of the first call sit right behind the entries the second one reads.

This file is named to be collected last (pytest -x stops at the first failure; a failure here must not hide the other
tests) and does not depend on what ran before it: it passes alone in a fresh process and at the end of the full suite.
"""
import ctypes as C

import numpy as np
import pytest

HMF = 0
FTOL = 1e-12


@pytest.fixture(scope="module")
def torch():
    import torch as _torch
    assert _torch.cuda.is_available(), "GPU tests need a CUDA device"
    return _torch


def _theta(N, seed):
    return np.random.default_rng(seed).uniform(-1.5, 1.5, N)


def _static_forces(lrmd, torch, theta_dev, stream=None):
    """One call of the no-allocation entry point on `stream` (default: torch's current stream); no synchronisation."""
    f = torch.empty_like(theta_dev)
    s = stream if stream is not None else torch.cuda.current_stream()
    rc, cuda_err = lrmd.lrmd_hmf_forces_static(theta_dev.data_ptr(), f.data_ptr(), theta_dev.numel(), int(s.cuda_stream))
    assert rc == lrmd.OK, (lrmd.strerror(rc), cuda_err)
    return f


def _context_forces(lrmd, theta):
    """The existing path: context + workspace allocated by the caller (torch) + lrmd_forces."""
    ctx = lrmd.Context(HMF, theta.size, 0.0)
    ctx.set_state(theta, np.zeros_like(theta))
    f = ctx.forces().cpu().numpy()
    ctx.close()
    return f


def _check(got, want, rows, A_rows):
    err = np.abs(got - want)
    tol = FTOL * A_rows + 4e-16
    bad = np.nonzero(err[rows] > tol)[0]
    assert bad.size == 0, (rows[bad[:5]], err[rows][bad[:5]], tol[bad[:5]])
    # every element, not only the rows whose A_i was computed: forces are O(1) and A_i >= 0.1 for this input, so
    # 1e-14 absolute is well inside 1e-12 * A_i
    assert float(err.max()) <= 1e-14, float(err.max())


def test_rejects_sizes_beyond_the_built_in_array(lrmd):
    """Argument checks come before any CUDA call, so this part runs without a GPU."""
    buf = (C.c_double * 4)()
    p = C.addressof(buf)
    assert lrmd.lrmd_hmf_forces_static(p, p, lrmd.STATIC_MAX_N + 1, 0)[0] == lrmd.ETOOBIG
    assert lrmd.lrmd_hmf_forces_static(p, p, 1 << 40, 0)[0] == lrmd.ETOOBIG
    assert "LRMD_STATIC_MAX_N" in lrmd.strerror(lrmd.ETOOBIG)
    assert lrmd.lrmd_hmf_forces_static(p, p, 0, 0)[0] == lrmd.EINVAL
    assert lrmd.lrmd_hmf_forces_static(None, p, 4, 0)[0] == lrmd.EINVAL
    assert lrmd.lrmd_hmf_forces_static(p, None, 4, 0)[0] == lrmd.EINVAL
    assert lrmd.lrmd_hmf_forces_static(p + 4, p, 2, 0)[0] == lrmd.EINVAL        # misaligned


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_context_path(lrmd, ref, torch):
    # sizes: several CTAs of 1024 particles plus a ragged tail; the second call is smaller than the first
    N1, N2 = 20_011, 4_099
    th1, th2 = _theta(N1, 11), _theta(N2, 12)
    d1, d2 = torch.as_tensor(th1, device="cuda"), torch.as_tensor(th2, device="cuda")
    f1 = _static_forces(lrmd, torch, d1)          # no synchronisation in between: same stream, so ordered
    f2 = _static_forces(lrmd, torch, d2)
    torch.cuda.synchronize()
    for th, got in ((th1, f1.cpu().numpy()), (th2, f2.cpu().numpy())):
        _, _, A, _ = ref.forces_abs(HMF, 0.0, th, None, form=1)
        _check(got, _context_forces(lrmd, th), np.arange(th.size), A)
    # the same input again gives the same bits (fixed summation trees, nothing left over from the calls before)
    f1b = _static_forces(lrmd, torch, d1)
    torch.cuda.synchronize()
    assert torch.equal(f1, f1b)


@pytest.mark.gpu
def test_largest_size_then_smallest_on_a_side_stream(lrmd, ref, torch):
    """N = LRMD_STATIC_MAX_N fills the whole array (4096 CTA sums); N = 1 right after it reads one entry of it.  Both on a
    stream other than the default one."""
    N = lrmd.STATIC_MAX_N
    th = _theta(N, 13)
    one = np.array([0.7])
    s = torch.cuda.Stream()
    d, d_one = torch.as_tensor(th, device="cuda"), torch.as_tensor(one, device="cuda")
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        f = _static_forces(lrmd, torch, d, s)
        f_one = _static_forces(lrmd, torch, d_one, s)
    s.synchronize()
    rows = np.random.default_rng(14).choice(N, 1024, replace=False)
    rows.sort()
    _, _, A, _ = ref.forces_rows(HMF, 0.0, th, None, rows, form=1, with_abs=True)
    _check(f.cpu().numpy(), _context_forces(lrmd, th), rows, A)
    # one particle: M = (cos, sin)(theta), f = cos*sin - sin*cos = 0 up to rounding, as on the context path
    got = f_one.cpu().numpy()
    assert np.all(np.abs(got - _context_forces(lrmd, one)) <= 4e-16)
    # one more than the maximum is refused and nothing is launched
    big = torch.empty(N + 1, dtype=torch.float64, device="cuda")
    rc, _ = lrmd.lrmd_hmf_forces_static(big.data_ptr(), big.data_ptr(), N + 1, int(s.cuda_stream))
    assert rc == lrmd.ETOOBIG
