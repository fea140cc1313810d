"""Stream semantics of the C ABI (include/lrmd.h, "Conventions": every call enqueues on the given CUDA stream and returns
without synchronising unless stated).  The other GPU tests all run on torch's current (= default) stream; here

  * every call of the path runs on a side stream while the default stream is kept busy, and must give the same bits
    as on the default stream without waiting for it;
  * two contexts run interleaved on two streams;
  * lrmd_energy and lrmd_step are captured into a caller's CUDA graph and replayed.

The expected values are the library's own results on the default stream — those are what test_gpu_parity.py compares
with the oracle — plus one direct oracle comparison per model so that the file also stands alone.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

HMF, RING, GRAV2D = 0, 1, 2
BUSY_CYCLES = 1_000_000_000        # torch.cuda._sleep: about 0.5 s at 1.9 GHz


@pytest.fixture(scope="module")
def torch():
    import torch as _torch
    assert _torch.cuda.is_available(), "GPU tests need a CUDA device"
    return _torch


def _state(model, N, seed):
    rng = np.random.default_rng(seed)
    if model == GRAV2D:
        r, ph = np.sqrt(rng.random(N)), 2 * np.pi * rng.random(N)
        px, py = 0.1 * rng.standard_normal(N), 0.1 * rng.standard_normal(N)
        return [r * np.cos(ph), r * np.sin(ph), px - px.mean(), py - py.mean()]
    a = 1.5 if model == HMF else 1.0
    return [rng.uniform(-a, a, N), rng.uniform(-0.5, 0.5, N)]


# (model, N, eps, dt, options): one case per kernel family of the path
CASES = [
    pytest.param(HMF, 10_000, 0.0, 0.05, None, id="hmf-cluster"),
    pytest.param(HMF, 100_003, 0.0, 0.05, None, id="hmf-grid"),
    pytest.param(HMF, 1_200_001, 0.0, 0.05, None, id="hmf-tma-graph"),
    pytest.param(HMF, 50_001, 0.0, 0.05, {5: 0}, id="hmf-prefetch-graph"),
    pytest.param(RING, 1_500, 0.01, 0.01, None, id="ring-ordered"),
    pytest.param(RING, 6_001, 0.01, 0.01, None, id="ring-symmetric"),
    pytest.param(GRAV2D, 6_001, 1e-3, 0.005, None, id="grav2d-symmetric"),
    pytest.param(GRAV2D, 50_001, 1e-3, 0.005, None, id="grav2d-band"),
    pytest.param(GRAV2D, 6_001, 1e-3, 0.005, {0: 1}, id="grav2d-f32pairs"),
]


def _sequence(lrmd, torch, model, N, eps, dt, options, st, stream):
    """set_state / forces / step / energy / step_observe / step_host, all on `stream` (None = the default stream).
    Returns the results as numpy arrays; synchronises only `stream`, and only at the end."""
    ctx = lrmd.Context(model, N, eps, options=options)
    ctx.set_state(*st)
    torch.cuda.synchronize()                     # the state copies above ran on the default stream
    busy_checked = None
    if stream is not None:
        torch.cuda._sleep(BUSY_CYCLES)           # default stream busy from here on
    f = ctx.forces(stream=stream)
    ctx.step(11, dt, stream=stream)              # 1 + 8 (one graph replay where the variant has one) + 2 steady steps
    e = ctx.energy(stream=stream)
    if stream is not None:
        with torch.cuda.stream(stream):          # step_observe allocates its output: do that on the side stream too
            rec = ctx.step_observe(4, dt, every=2, stream=stream)
    else:
        rec = ctx.step_observe(4, dt, every=2)
    host = [torch.from_numpy(a.copy()).pin_memory() for a in st]
    ctx.step_host(host, 2, dt, stream=stream)    # synchronises `stream`
    if stream is not None:
        stream.synchronize()
        busy_checked = not torch.cuda.default_stream().query()     # True: the default stream was still busy
    torch.cuda.synchronize()
    f = tuple(t.cpu().numpy() for t in f) if model == GRAV2D else (f.cpu().numpy(),)
    out = {"f": f, "e": e.cpu().numpy(), "rec": rec.cpu().numpy(), "state": ctx.state_numpy(),
           "host": tuple(h.numpy().copy() for h in host), "busy": busy_checked}
    ctx.close()
    return out


def _same(a, b):
    for k in ("f", "state", "host"):
        for x, y in zip(a[k], b[k]):
            assert np.array_equal(x, y), k
    assert np.array_equal(a["e"], b["e"]) and np.array_equal(a["rec"], b["rec"])


@pytest.mark.parametrize("model,N,eps,dt,options", CASES)
def test_side_stream_gives_the_default_streams_bits_without_waiting_for_it(lrmd, ref, torch, model, N, eps, dt, options):
    st = _state(model, N, 31 + N % 13)
    base = _sequence(lrmd, torch, model, N, eps, dt, options, st, None)
    side = _sequence(lrmd, torch, model, N, eps, dt, options, st, torch.cuda.Stream())
    _same(base, side)
    # the whole sequence finished on the side stream while the default stream was still spinning: no call waited for it
    assert side["busy"] is True
    # stand-alone anchor: the 2-step host round trip against the oracle (1e-9, or 1e-6 with fp32 pair terms)
    r = [a.copy() for a in st]
    two = model == GRAV2D
    ref.step(model, eps, r[0], r[1] if two else None, r[2] if two else r[1], r[3] if two else None, 2, dt,
             form=(0 if model == HMF else 1))
    tol = 1e-6 if (options or {}).get(0) == 1 else 1e-9
    for g, w in zip(side["host"], r):
        assert np.max(np.abs(g - w)) <= tol


def test_two_contexts_interleaved_on_two_streams(lrmd, torch):
    specs = [(HMF, 300_007, 0.0, 0.05), (GRAV2D, 9_001, 1e-3, 0.005), (RING, 5_003, 0.01, 0.01), (HMF, 9_000, 0.0, 0.05)]
    states = [_state(m, N, 70 + k) for k, (m, N, _, _) in enumerate(specs)]

    def run(streams):
        ctxs = []
        for (m, N, eps, _), st in zip(specs, states):
            c = lrmd.Context(m, N, eps)
            c.set_state(*st)
            ctxs.append(c)
        torch.cuda.synchronize()
        es = [None] * len(ctxs)
        for rnd in range(3):                     # round-robin: every context's calls interleave with the others'
            for k, (c, (_, _, _, dt)) in enumerate(zip(ctxs, specs)):
                s = streams[k % len(streams)] if streams else None
                c.step(3 + rnd, dt, stream=s)
                es[k] = c.energy(stream=s)
        torch.cuda.synchronize()
        out = [(c.state_numpy(), e.cpu().numpy()) for c, e in zip(ctxs, es)]
        for c in ctxs:
            c.close()
        return out

    seq = run(None)
    par = run([torch.cuda.Stream(), torch.cuda.Stream()])
    for (sa, ea), (sb, eb) in zip(seq, par):
        for x, y in zip(sa, sb):
            assert np.array_equal(x, y)
        assert np.array_equal(ea, eb)


GRAPH_CASES = [
    pytest.param(HMF, 1_200_001, 0.0, 0.05, None, id="hmf-tma"),
    pytest.param(HMF, 50_001, 0.0, 0.05, {5: 0}, id="hmf-prefetch"),
    pytest.param(RING, 6_001, 0.01, 0.01, None, id="ring-symmetric"),
    pytest.param(GRAV2D, 50_001, 1e-3, 0.005, None, id="grav2d-band"),
    pytest.param(GRAV2D, 1_500, 1e-3, 0.005, None, id="grav2d-ordered"),
]


@pytest.mark.parametrize("model,N,eps,dt,options", GRAPH_CASES)
def test_energy_and_step_replay_from_a_callers_cuda_graph(lrmd, torch, model, N, eps, dt, options):
    """include/lrmd.h, "Capturing calls in a CUDA graph": after one eager lrmd_step (force cached, kernel attributes
    set) lrmd_step and lrmd_energy consist of plain kernel launches on the given stream, so a caller may capture them;
    every replay then advances the bound state by the captured number of steps and rewrites the energy record."""
    st = _state(model, N, 90 + N % 7)
    # eager: 1 + 2 + 2 steps, energy after each block of 2
    a = lrmd.Context(model, N, eps, options=options)
    a.set_state(*st)
    a.step(1, dt)
    a.energy()
    want = []
    for _ in range(2):
        a.step(2, dt)
        want.append(a.energy().cpu().numpy())
    want_state = a.state_numpy()
    a.close()
    # captured: the same, with the block of 2 steps + energy recorded once and replayed twice
    b = lrmd.Context(model, N, eps, options=options)
    b.set_state(*st)
    b.step(1, dt)
    b.energy()
    torch.cuda.synchronize()
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    before = [t.clone() for t in b.state]
    with torch.cuda.graph(g, stream=s):
        sp = int(torch.cuda.current_stream().cuda_stream)
        assert lrmd.lrmd_step(b._h, 2, dt, sp) == lrmd.OK
        assert lrmd.lrmd_energy(b._h, out.data_ptr(), sp) == lrmd.OK
    torch.cuda.synchronize()
    for x, y in zip(before, b.state):            # capturing enqueued nothing
        assert torch.equal(x, y)
    got = []
    for _ in range(2):
        g.replay()
        torch.cuda.synchronize()
        got.append(out.cpu().numpy().copy())
    for x, y in zip(want, got):
        assert np.array_equal(x, y)
    for x, y in zip(want_state, b.state_numpy()):
        assert np.array_equal(x, y)
    del g
    b.close()
