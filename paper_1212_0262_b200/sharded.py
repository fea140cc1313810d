"""Multi-GPU sharding of the hot path: one process per
GPU, each owning a contiguous range of particles.  The arithmetic stays in the CUDA kernels behind the C ABI
(``lrmd_set_shard``); this module is plumbing only: shard bounds, and the two exchange steps handed to the library
as callbacks that run ``torch.distributed`` collectives (NCCL on GPUs) on views of the context's workspace:

  HMF          one all-reduce of 2 doubles per substage (each GPU's contribution to the magnetisation, summed);
  RING/GRAV2D  one all-gather of the packed positions per substage (every GPU needs all positions for its rows).

BASELINE.json's north_star fixes ONE GPU, so bench.py's default line never uses this module (replicas only);
``bench.py --sharded`` times it as an opt-in strong-scaling line.  It is covered by a two- and three-rank emulation on
one GPU (tests/test_gpu_sharded.py) and by gloo world-2 CPU tests of the collectives and of bench.py's host logic.
"""
from __future__ import annotations

import ctypes as C

from . import lrmd

ALLREDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p)
ALLGATHER_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int64, C.c_int64, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p)


def shard_bounds(n_total: int, world: int):
    """[(i0, n)] per rank: contiguous, sizes differ by at most one, every particle owned exactly once."""
    edges = [(n_total * r) // world for r in range(world + 1)]
    return [(edges[r], edges[r + 1] - edges[r]) for r in range(world)]


class TorchDistCollectives:
    """The two exchange steps on top of a ``torch.distributed``-like module (nccl on GPUs, gloo on CPU)."""

    def __init__(self, dist, rank: int, world: int, group=None):
        self.dist, self.rank, self.world, self.group = dist, rank, world, group

    def all_reduce_sum_(self, t):
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)

    def all_gather_inplace_(self, whole, byte_bounds):
        """``whole``: uint8 tensor of all ranks' elements; ``byte_bounds[r] = (b0, b1)`` is rank r's byte range, and
        this rank's range is already filled in."""
        sizes = {b1 - b0 for b0, b1 in byte_bounds}
        if len(sizes) == 1:
            b0, b1 = byte_bounds[self.rank]
            self.dist.all_gather_into_tensor(whole, whole[b0:b1].clone(), group=self.group)
        else:
            for r, (b0, b1) in enumerate(byte_bounds):
                if b1 > b0:
                    self.dist.broadcast(whole[b0:b1], src=r, group=self.group)


class SingleRankCollectives:
    """World of one rank: nothing to exchange (the library runs its unsharded path and never calls back)."""
    rank, world = 0, 1

    def all_reduce_sum_(self, t):
        pass

    def all_gather_inplace_(self, whole, byte_bounds):
        pass


class ShardedContext(lrmd.Context):
    """A ``Context`` that owns particles ``i0 .. i0 + n - 1`` of ``n_total``.  ``set_state`` takes the owned slices
    (or use ``set_state_global``); ``step`` / ``forces`` work on them; ``energy_global`` sums the parts over ranks."""

    def __init__(self, model: int, n_total: int, eps: float, coll, device="cuda:0", options: dict | None = None):
        self.coll = coll
        self.last_collective_error = None             # the exception behind the last LRMD_ECOLL, if any
        self.n_total = int(n_total)
        self.bounds = shard_bounds(self.n_total, coll.world)
        self.i0, n_local = self.bounds[coll.rank]
        if n_local < 1:
            raise ValueError("more ranks than particles")
        super().__init__(model, n_local, eps, device=device, options=options)
        self._ar = ALLREDUCE_FN(self._allreduce)      # keep the ctypes thunks alive as long as the context
        self._ag = ALLGATHER_FN(self._allgather)
        rc = lrmd.load().lrmd_set_shard(self._h, self.n_total, self.i0, self._ar, self._ag, None)
        self._chk(rc, "lrmd_set_shard")
        self._bind_workspace()

    def _chk(self, rc, what):
        """As Context._chk; an LRMD_ECOLL carries the exception the collective callback raised (it cannot cross the C
        boundary, so the callback stores it and returns 1)."""
        if rc == lrmd.ECOLL and self.last_collective_error is not None:
            exc, self.last_collective_error = self.last_collective_error, None
            raise lrmd.LrmdError(rc, "%s (collective callback raised %s: %s)" % (what, type(exc).__name__, exc)) from exc
        super()._chk(rc, what)

    # -- views of the workspace the library hands back as raw device pointers
    def _view(self, ptr: int, nbytes: int):
        off = ptr - self._ws.data_ptr()
        if off < 0 or off + nbytes > self._ws.numel():
            raise RuntimeError("collective buffer outside the workspace")
        return self._ws[off:off + nbytes]

    def _on_stream(self, stream):
        """Context manager that makes ``stream`` (the raw cudaStream_t the library launches its kernels on) torch's
        current stream, so that a ``torch.distributed`` collective issued inside is ordered after the kernels
        already enqueued on it and before the ones that follow (the process group orders its work against the
        current stream).  CPU tensors (gloo tests) have no stream: a null context."""
        import contextlib
        torch = self._torch
        if self._ws.device.type != "cuda":
            return contextlib.nullcontext()
        ext = torch.cuda.ExternalStream(int(stream or 0), device=self._ws.device)
        return torch.cuda.stream(ext)

    def _allreduce(self, ptr, count, stream, user):
        try:
            with self._on_stream(stream):
                self.coll.all_reduce_sum_(self._view(ptr, 8 * count).view(self._torch.float64))
            return 0
        except Exception as exc:   # never let an exception cross the C boundary; kept for the LRMD_ECOLL report
            self.last_collective_error = exc
            return 1

    def _allgather(self, ptr, elem_bytes, i0, n_local, n_total, stream, user):
        try:
            whole = self._view(ptr, elem_bytes * n_total)
            with self._on_stream(stream):
                self.coll.all_gather_inplace_(whole, [(b * elem_bytes, (b + n) * elem_bytes) for b, n in self.bounds])
            return 0
        except Exception as exc:
            self.last_collective_error = exc
            return 1

    def set_state_global(self, *arrays):
        """Slices this rank's particles out of arrays of length ``n_total``."""
        self.set_state(*[a[self.i0:self.i0 + self.N] for a in arrays])

    def energy_global(self, stream=None):
        """{K, V, a, b} of the whole system: the per-rank parts of ``lrmd_energy`` summed over ranks (HMF: only K
        is partial; V, Mx, My are already global)."""
        e = self.energy(stream).clone()
        if self.model == lrmd.HMF:
            self.coll.all_reduce_sum_(e[0:1])
        else:
            self.coll.all_reduce_sum_(e)
        return e
