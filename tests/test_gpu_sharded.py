"""Sharded contexts (lrmd_set_shard) on ONE GPU: two ranks are emulated by
two host threads, each with its own ShardedContext over half of the particles; the exchange callbacks meet at a host
barrier and are carried out with plain torch ops on the shared device (no kernel ever waits on another kernel: the
waiting is on the host, and all work goes to the same stream in issue order).  The result must match the oracle —
and the unsharded context — within north_star's tolerances."""
import threading

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

HMF, RING, GRAV2D = 0, 1, 2


class ThreadColl:
    """Collectives among `world` threads of one process sharing one CUDA device."""

    def __init__(self, shared, rank, world):
        self.shared, self.rank, self.world = shared, rank, world

    def _meet(self):
        self.shared["barrier"].wait(timeout=120)

    def all_reduce_sum_(self, t):
        slots = self.shared["slots"]
        slots[self.rank] = t
        self._meet()
        if self.rank == 0:
            total = slots[0].clone()
            for r in range(1, self.world):
                total += slots[r]
            for r in range(self.world):
                slots[r].copy_(total)
        self._meet()

    def all_gather_inplace_(self, whole, byte_bounds):
        slots = self.shared["slots"]
        slots[self.rank] = whole
        self._meet()
        if self.rank == 0:
            for src, (b0, b1) in enumerate(byte_bounds):
                for dst in range(self.world):
                    if dst != src:
                        slots[dst][b0:b1].copy_(slots[src][b0:b1])
        self._meet()


def _run_ranks(world, fn):
    shared = {"barrier": threading.Barrier(world), "slots": [None] * world}
    out, err = [None] * world, []

    def body(r):
        try:
            out[r] = fn(ThreadColl(shared, r, world), r)
        except Exception as e:   # noqa: BLE001
            err.append(e)
            shared["barrier"].abort()

    ths = [threading.Thread(target=body, args=(r,)) for r in range(world)]
    for t in ths:
        t.start()
    for t in ths:
        t.join(300)
    assert not err, err
    return out


def _state(model, N, seed):
    rng = np.random.default_rng(seed)
    if model == GRAV2D:
        r, ph = np.sqrt(rng.random(N)), 2 * np.pi * rng.random(N)
        px, py = 0.1 * rng.standard_normal(N), 0.1 * rng.standard_normal(N)
        return [r * np.cos(ph), r * np.sin(ph), px - px.mean(), py - py.mean()]
    a = 1.5 if model == HMF else 1.0
    return [rng.uniform(-a, a, N), rng.uniform(-0.5, 0.5, N)]


@pytest.mark.parametrize("model,N,world", [(HMF, 30_001, 2), (HMF, 2_000_003, 2), (RING, 2001, 2), (GRAV2D, 2001, 2),
                                           (GRAV2D, 1500, 3)])
def test_two_emulated_ranks_match_oracle(lrmd, ref, model, N, world):
    import torch
    from paper_1212_0262_b200.sharded import ShardedContext
    eps = {HMF: 0.0, RING: 0.01, GRAV2D: 1e-3}[model]
    st = _state(model, N, 5 + N % 7)
    steps, dt = 5, 0.01

    def rank_fn(coll, r):
        ctx = ShardedContext(model, N, eps, coll)
        ctx.set_state_global(*st)
        f = ctx.forces()
        f = [t.cpu().numpy() for t in f] if model == GRAV2D else [f.cpu().numpy()]
        e0 = ctx.energy_global().cpu().numpy()
        ctx.step(steps, dt)
        fin = ctx.state_numpy()
        e1 = ctx.energy_global().cpu().numpy()
        i0, n = ctx.i0, ctx.N
        ctx.close()
        return i0, n, f, fin, e0, e1

    res = _run_ranks(world, rank_fn)
    torch.cuda.synchronize()
    two = model == GRAV2D
    q0, q1 = (st[0], st[1]) if two else (st[0], None)
    p0, p1 = (st[2], st[3]) if two else (st[1], None)
    f0, f1, A0, A1 = ref.forces_abs(model, eps, q0, q1, form=0)    # HMF: eqs.(6)-(7), A = the O(N) bound S_i
    er0, ea0 = ref.energy(model, eps, q0, q1, p0, p1)
    r = [a.copy() for a in st]
    rq0, rq1 = (r[0], r[1]) if two else (r[0], None)
    rp0, rp1 = (r[2], r[3]) if two else (r[1], None)
    ref.step(model, eps, rq0, rq1, rp0, rp1, steps, dt, form=(0 if model == HMF else 1))
    er1, ea1 = ref.energy(model, eps, rq0, rq1, rp0, rp1)
    covered = 0
    for i0, n, f, fin, e0, e1 in res:
        sl = slice(i0, i0 + n)
        covered += n
        assert np.all(np.abs(f[0] - f0[sl]) <= 1e-12 * A0[sl] + 4e-16)
        if two:
            assert np.all(np.abs(f[1] - f1[sl]) <= 1e-12 * A1[sl])
        for g, w in zip(fin, r):
            assert np.max(np.abs(g - w[sl])) <= 1e-9
        for e, er, ea in ((e0, er0, ea0), (e1, er1, ea1)):
            assert abs(e[0] - er[0]) <= 1e-11 * max(ea[0], 1e-300)
            assert abs(e[1] - er[1]) <= 1e-11 * max(ea[1], 0.5 * N if model == HMF else 0.0)
    assert covered == N


def test_single_shard_is_the_unsharded_path(lrmd):
    """N_total = N: no callbacks are needed and the bits equal those of a plain Context."""
    N = 3000
    st = _state(RING, N, 3)
    a = lrmd.Context(RING, N, 0.01)
    a.set_state(*st)
    a.step(3, 0.01)
    b = lrmd.Context(RING, N, 0.01)
    assert lrmd.load().lrmd_set_shard(b._h, N, 0, None, None, None) == lrmd.OK
    b._bind_workspace()
    b.set_state(*st)
    b.step(3, 0.01)
    for x, y in zip(a.state_numpy(), b.state_numpy()):
        assert np.array_equal(x, y)
    rc, h = lrmd.lrmd_create(HMF, 10, 0.0)
    assert lrmd.load().lrmd_set_shard(h, 20, 5, None, None, None) == lrmd.EINVAL     # a shard needs its all-reduce
    assert lrmd.load().lrmd_set_shard(h, 5, 0, None, None, None) == lrmd.EINVAL      # N_total < N
    lrmd.lrmd_destroy(h)
    a.close(); b.close()


class _FailingColl:
    """One rank that claims to be rank 0 of 2; its collectives raise."""
    rank, world = 0, 2

    def all_reduce_sum_(self, t):
        raise RuntimeError("link down (all_reduce)")

    def all_gather_inplace_(self, whole, byte_bounds):
        raise RuntimeError("link down (all_gather)")


@pytest.mark.parametrize("model,what", [(HMF, "all_reduce"), (GRAV2D, "all_gather")])
def test_a_failing_collective_surfaces_with_its_message(model, what):
    """A collective callback that raises cannot let the exception cross the C boundary: the library returns LRMD_ECOLL
    and the binding re-raises with the original exception attached, instead of a bare error code."""
    from paper_1212_0262_b200 import lrmd, sharded
    N = 4096
    ctx = sharded.ShardedContext(model, N, 0.0 if model == HMF else 1e-3, _FailingColl())
    rng = np.random.default_rng(3)
    ctx.set_state(*[rng.uniform(-1, 1, ctx.N) for _ in range(ctx.narrays)])
    with pytest.raises(lrmd.LrmdError) as ei:
        ctx.step(1, 0.01)
    assert ei.value.code == lrmd.ECOLL and "link down (%s)" % what in str(ei.value)
    assert isinstance(ei.value.__cause__, RuntimeError)
    ctx.close()
