"""Thin Python binding of the C ABI in ``include/lrmd.h`` (``liblrmd.so``).

Argument marshalling only: every step of the hot path (force evaluation, kick/drift updates,
energy sums, integrator sequencing — PAPER.md:46-110) runs in the CUDA kernels behind the C ABI.
PyTorch is used for device memory and streams, nothing else.  There is no CPU fallback: if the
library cannot be built/loaded, or a call is made without a CUDA device, this module raises.

Two layers:
  * module functions ``lrmd_create`` ... ``lrmd_coefficients`` — same names and argument order as
    the C calls, raw pointers as ints, return the C return code;
  * ``Context`` — owns the torch tensors (state, workspace) and raises ``LrmdError`` on a non-zero code.
"""
from __future__ import annotations

import ctypes as C
import os

HMF, RING, GRAV2D = 0, 1, 2
OK, EINVAL, ESTATE, ECUDA, EUNSUPPORTED, ECOLL, ETOOBIG = 0, -1, -2, -3, -4, -5, -6
STATIC_MAX_N = 4194304      # LRMD_STATIC_MAX_N of include/lrmd.h
OPT_PAIR_PRECISION, OPT_PAIR_CTAS, OPT_GRAPH, OPT_HMF_GRID, OPT_KERNEL_TIMING = 0, 1, 2, 3, 4
OPT_HMF_VARIANT, OPT_PAIR_VARIANT, OPT_PAIR_SLOTS, OPT_PAIR_SYMMETRIC, OPT_PAIR_SYM_TILES = 5, 6, 7, 8, 9
OPT_PAIR_FUSE_UPDATE = 10
OPT_PAIR_SYM_EXCHANGE = 11
OPT_PAIR_BAND_HEIGHT = 12

#: every symbol include/lrmd.h declares (tests check the library exports each of them)
SYMBOLS = (
    "lrmd_create", "lrmd_destroy", "lrmd_workspace_bytes", "lrmd_set_workspace", "lrmd_set_state",
    "lrmd_step", "lrmd_step_host", "lrmd_forces", "lrmd_energy", "lrmd_set_option", "lrmd_get_option",
    "lrmd_launch_count", "lrmd_kernel_time", "lrmd_last_cuda_error", "lrmd_strerror", "lrmd_coefficients", "lrmd_host_sincos",
    "lrmd_pair_partition", "lrmd_step_observe", "lrmd_set_shard", "lrmd_pair_sym_partition", "lrmd_fp64_peak",
    "lrmd_pair_band_partition", "lrmd_hmf_forces_static",
)

_lib = None
_vp, _i64, _dbl, _int = C.c_void_p, C.c_int64, C.c_double, C.c_int


class LrmdError(RuntimeError):
    def __init__(self, code: int, what: str, cuda_error: int = 0):
        self.code = code
        self.cuda_error = cuda_error
        msg = f"{what}: {strerror(code)} (code {code})"
        if cuda_error:
            msg += f", cudaError {cuda_error}"
        super().__init__(msg)


def library_path() -> str:
    from . import build as _build
    return _build.OUT


def load(build_if_missing: bool = True):
    """Load ``liblrmd.so`` (building it with nvcc first if missing or stale).  Raises on failure."""
    global _lib
    if _lib is not None:
        return _lib
    from . import build as _build
    path = _build.build() if build_if_missing else _build.OUT
    if not os.path.exists(path):
        raise RuntimeError(f"liblrmd.so not found at {path}: the CUDA library is required (no CPU fallback)")
    lib = C.CDLL(path)
    lib.lrmd_create.argtypes = [C.POINTER(_vp), _int, _i64, _dbl]
    lib.lrmd_destroy.argtypes = [_vp]
    lib.lrmd_workspace_bytes.argtypes = [_vp, C.POINTER(C.c_size_t)]
    lib.lrmd_set_workspace.argtypes = [_vp, _vp, C.c_size_t, _vp]
    lib.lrmd_set_state.argtypes = [_vp, _vp, _vp, _vp, _vp]
    lib.lrmd_step.argtypes = [_vp, _i64, _dbl, _vp]
    lib.lrmd_step_host.argtypes = [_vp, _vp, _vp, _vp, _vp, _i64, _dbl, _vp]
    lib.lrmd_forces.argtypes = [_vp, _vp, _vp, _vp]
    lib.lrmd_energy.argtypes = [_vp, _vp, _vp]
    lib.lrmd_set_option.argtypes = [_vp, _int, _i64]
    lib.lrmd_get_option.argtypes = [_vp, _int, C.POINTER(_i64)]
    lib.lrmd_launch_count.argtypes = [_vp, C.POINTER(_i64)]
    lib.lrmd_kernel_time.argtypes = [_vp, C.POINTER(_dbl), C.POINTER(_i64)]
    lib.lrmd_last_cuda_error.argtypes = [_vp]
    lib.lrmd_strerror.argtypes = [_int]
    lib.lrmd_strerror.restype = C.c_char_p
    lib.lrmd_coefficients.argtypes = [C.POINTER(_dbl)]
    lib.lrmd_host_sincos.argtypes = [_vp, _i64, _vp, _vp]
    lib.lrmd_pair_partition.argtypes = [_vp, _i64, _vp, _i64, C.POINTER(_i64)]
    lib.lrmd_step_observe.argtypes = [_vp, _i64, _dbl, _i64, _vp, _vp]
    lib.lrmd_set_shard.argtypes = [_vp, _i64, _i64, _vp, _vp, _vp]
    lib.lrmd_pair_sym_partition.argtypes = [_vp, _i64, _vp, C.POINTER(_i64)]
    lib.lrmd_pair_band_partition.argtypes = [_vp, _i64, _vp, C.POINTER(_i64)]
    lib.lrmd_fp64_peak.argtypes = [_int, _int, _int, _int, _int, _vp, C.c_size_t, C.POINTER(_dbl), _vp]
    lib.lrmd_hmf_forces_static.argtypes = [_vp, _vp, _i64, _vp, C.POINTER(_int)]
    for name in SYMBOLS:
        if name != "lrmd_strerror":
            getattr(lib, name).restype = _int
    _lib = lib
    return lib


# ---- raw calls: same names as the C ABI ---------------------------------------------------------------

def lrmd_create(model: int, N: int, eps: float):
    """Returns (rc, ctx_handle)."""
    h = _vp()
    rc = load().lrmd_create(C.byref(h), int(model), int(N), float(eps))
    return rc, h.value


def lrmd_destroy(ctx):
    return load().lrmd_destroy(ctx)


def lrmd_workspace_bytes(ctx):
    """Returns (rc, bytes)."""
    n = C.c_size_t(0)
    rc = load().lrmd_workspace_bytes(ctx, C.byref(n))
    return rc, int(n.value)


def lrmd_set_workspace(ctx, device_ptr: int, nbytes: int, stream: int = 0):
    return load().lrmd_set_workspace(ctx, device_ptr, nbytes, stream)


def lrmd_set_state(ctx, a0: int, a1: int, a2: int | None = None, a3: int | None = None):
    return load().lrmd_set_state(ctx, a0, a1, a2, a3)


def lrmd_step(ctx, n: int, dt: float, stream: int = 0):
    return load().lrmd_step(ctx, int(n), float(dt), stream)


def lrmd_step_observe(ctx, n: int, dt: float, every: int, out_device: int, stream: int = 0):
    return load().lrmd_step_observe(ctx, int(n), float(dt), int(every), out_device, stream)


def lrmd_step_host(ctx, h0: int, h1: int, h2: int | None, h3: int | None, n: int, dt: float, stream: int = 0):
    return load().lrmd_step_host(ctx, h0, h1, h2, h3, int(n), float(dt), stream)


def lrmd_forces(ctx, f0: int, f1: int | None = None, stream: int = 0):
    return load().lrmd_forces(ctx, f0, f1, stream)


def lrmd_energy(ctx, out4_device: int, stream: int = 0):
    return load().lrmd_energy(ctx, out4_device, stream)


def lrmd_hmf_forces_static(theta_device: int, f_device: int, N: int, stream: int = 0):
    """HMF forces without a context or a workspace, for callers that cannot allocate scratch (a plug-in inside an
    application that owns all device memory, a loop where cudaMalloc's device-wide stall is not acceptable): the
    library's built-in 64 KiB array holds the per-CTA sums, so N <= STATIC_MAX_N (else ETOOBIG).  Raw device pointers
    as ints.  Returns (rc, cudaError).  All calls share that one array: calls on one stream are safe, calls that may
    overlap on the GPU are not.  Make the first call on each device outside any stream capture.  See include/lrmd.h."""
    err = _int(0)
    rc = load().lrmd_hmf_forces_static(theta_device, f_device, int(N), stream, C.byref(err))
    return rc, int(err.value)


def lrmd_set_option(ctx, key: int, value: int):
    return load().lrmd_set_option(ctx, int(key), int(value))


def lrmd_get_option(ctx, key: int):
    """Returns (rc, value)."""
    v = _i64(0)
    rc = load().lrmd_get_option(ctx, int(key), C.byref(v))
    return rc, int(v.value)


def lrmd_launch_count(ctx):
    """Returns (rc, launches)."""
    v = _i64(0)
    rc = load().lrmd_launch_count(ctx, C.byref(v))
    return rc, int(v.value)


def lrmd_kernel_time(ctx):
    """Returns (rc, ms_total, launches)."""
    ms, n = _dbl(0.0), _i64(0)
    rc = load().lrmd_kernel_time(ctx, C.byref(ms), C.byref(n))
    return rc, float(ms.value), int(n.value)


def lrmd_last_cuda_error(ctx) -> int:
    return load().lrmd_last_cuda_error(ctx)


def strerror(code: int) -> str:
    return load().lrmd_strerror(int(code)).decode()


lrmd_strerror = strerror


def lrmd_coefficients():
    """(B0, B1, D0, D1) used by lrmd_step."""
    out = (_dbl * 4)()
    rc = load().lrmd_coefficients(out)
    if rc != OK:
        raise LrmdError(rc, "lrmd_coefficients")
    return tuple(float(v) for v in out)


def lrmd_host_sincos(x):
    """Diagnostic: the library's own sincos arithmetic evaluated on the host.  numpy in, (sin, cos) out."""
    import numpy as np
    x = np.ascontiguousarray(x, dtype=np.float64)
    s = np.empty_like(x)
    c = np.empty_like(x)
    rc = load().lrmd_host_sincos(x.ctypes.data, x.size, s.ctypes.data, c.ctypes.data)
    if rc != OK:
        raise LrmdError(rc, "lrmd_host_sincos")
    return s, c


def lrmd_pair_partition(ctx, cta: int, max_seg: int = 64):
    """Diagnostic: (rc, segments) of CTA ``cta`` of the pair kernels; segments is an (n, 4) int64 numpy
    array of rows {tile, jbeg, jend, slot}."""
    import numpy as np
    buf = np.zeros((max(max_seg, 1), 4), dtype=np.int64)
    n = _i64(0)
    rc = load().lrmd_pair_partition(ctx, int(cta), buf.ctypes.data, int(max_seg), C.byref(n))
    if rc == OK and n.value > max_seg:
        return lrmd_pair_partition(ctx, cta, int(n.value))
    return rc, buf[: n.value].copy()


def lrmd_pair_sym_partition(ctx):
    """Diagnostic: (rc, table) with one row {tile, chunk, units, launch, tile size} per worker of the symmetric
    pair kernel (an empty table if it is not in use)."""
    import numpy as np
    n = _i64(0)
    rc = load().lrmd_pair_sym_partition(ctx, 0, None, C.byref(n))
    tab = np.zeros((n.value, 5), dtype=np.int64)
    for w in range(n.value):
        if rc != OK:
            break
        rc = load().lrmd_pair_sym_partition(ctx, w, tab[w].ctypes.data, None)
    return rc, tab


def lrmd_pair_band_partition(ctx):
    """Diagnostic: (rc, table) with one row {band, c0, c1, worker, first I-block of the band, I-blocks in the band,
    IB, workers} per piece of the band kernel's partition (an empty table if it is not in use)."""
    import numpy as np
    n = _i64(0)
    rc = load().lrmd_pair_band_partition(ctx, 0, None, C.byref(n))
    tab = np.zeros((n.value, 8), dtype=np.int64)
    for k in range(n.value):
        if rc != OK:
            break
        rc = load().lrmd_pair_band_partition(ctx, k, tab[k].ctypes.data, None)
    return rc, tab


def lrmd_fp64_peak(op: int, mix: int, extra_per_16: int, warps_per_sm: int, iters: int, scratch_device: int,
                   scratch_bytes: int, stream: int = 0):
    """Diagnostic: (rc, (fp64 instr/s, SM MHz held, FP64 lanes per clock per SM, ms)) of the issue-rate microbenchmark."""
    out = (_dbl * 4)()
    rc = load().lrmd_fp64_peak(int(op), int(mix), int(extra_per_16), int(warps_per_sm), int(iters), scratch_device,
                               int(scratch_bytes), out, stream)
    return rc, tuple(float(v) for v in out)


# ---- convenience object ---------------------------------------------------------------------------------

class Context:
    """One simulation context on one CUDA device.  Owns the state tensors and the workspace.

    ``state`` is (theta, p) for HMF/RING or (x, y, px, py) for GRAV2D, as numpy arrays or torch
    tensors; they are copied to fp64 device tensors which ``step`` updates in place.
    """

    def __init__(self, model: int, N: int, eps: float = 0.0, device="cuda:0", options: dict | None = None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1212_0262_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self._torch = torch
        self.device = torch.device(device)
        self.model, self.N, self.eps = int(model), int(N), float(eps)
        load()
        with torch.cuda.device(self.device):
            rc, self._h = lrmd_create(model, N, eps)
        if rc != OK:
            self._h = None
            raise LrmdError(rc, "lrmd_create")
        self._ws = None
        self._state = None
        self._host = None
        for k, v in (options or {}).items():
            self._chk(lrmd_set_option(self._h, k, v), "lrmd_set_option")
        self._bind_workspace()

    # -- helpers
    def _chk(self, rc, what):
        if rc != OK:
            raise LrmdError(rc, what, lrmd_last_cuda_error(self._h) if self._h else 0)

    def _stream(self, stream=None) -> int:
        s = stream if stream is not None else self._torch.cuda.current_stream(self.device)
        return int(s.cuda_stream)

    def _bind_workspace(self):
        torch = self._torch
        rc, nbytes = lrmd_workspace_bytes(self._h)
        self._chk(rc, "lrmd_workspace_bytes")
        self._ws = torch.empty(max(nbytes, 256) + 256, dtype=torch.uint8, device=self.device)
        ptr = (self._ws.data_ptr() + 255) // 256 * 256
        self._chk(lrmd_set_workspace(self._h, ptr, nbytes, self._stream()), "lrmd_set_workspace")

    def workspace_bytes(self) -> int:
        """Scratch the library asked for with the current options (lrmd_workspace_bytes)."""
        rc, nbytes = lrmd_workspace_bytes(self._h)
        self._chk(rc, "lrmd_workspace_bytes")
        return nbytes

    @property
    def narrays(self) -> int:
        return 4 if self.model == GRAV2D else 2

    def set_option(self, key: int, value: int):
        self._chk(lrmd_set_option(self._h, key, value), "lrmd_set_option")
        if key not in (OPT_KERNEL_TIMING, OPT_PAIR_FUSE_UPDATE, OPT_PAIR_SYM_EXCHANGE):   # the others may change the workspace size
            self._bind_workspace()

    def get_option(self, key: int) -> int:
        rc, v = lrmd_get_option(self._h, key)
        self._chk(rc, "lrmd_get_option")
        return v

    def set_state(self, *arrays):
        torch = self._torch
        if len(arrays) != self.narrays:
            raise ValueError(f"model {self.model} takes {self.narrays} state arrays")
        st = []
        for a in arrays:
            t = torch.as_tensor(a, dtype=torch.float64)
            if t.numel() != self.N:
                raise ValueError("state arrays must have length N")
            st.append(t.to(self.device, copy=True).contiguous())
        self._state = st
        ptrs = [t.data_ptr() for t in st] + [None] * (4 - len(st))
        self._chk(lrmd_set_state(self._h, *ptrs), "lrmd_set_state")

    @property
    def state(self):
        """The device tensors, updated in place by ``step``."""
        return tuple(self._state)

    def state_numpy(self):
        return tuple(t.cpu().numpy() for t in self._state)

    def step(self, n: int, dt: float, stream=None):
        with self._torch.cuda.device(self.device):
            self._chk(lrmd_step(self._h, n, dt, self._stream(stream)), "lrmd_step")

    def step_observe(self, n: int, dt: float, every: int = 1, stream=None):
        """``n`` steps with an ``lrmd_energy`` record {K, V, a, b} of the initial state and after every
        ``every``-th step: returns a device tensor of shape (n // every + 1, 4)."""
        torch = self._torch
        out = torch.empty((n // every + 1, 4), dtype=torch.float64, device=self.device)
        with torch.cuda.device(self.device):
            self._chk(lrmd_step_observe(self._h, n, dt, every, out.data_ptr(), self._stream(stream)), "lrmd_step_observe")
        return out

    def step_host(self, host_arrays, n: int, dt: float, stream=None):
        """End to end through ``lrmd_step_host``: ``host_arrays`` are (pinned) CPU fp64 tensors,
        read as the initial state and overwritten with the final one."""
        ptrs = [t.data_ptr() for t in host_arrays] + [None] * (4 - len(host_arrays))
        with self._torch.cuda.device(self.device):
            self._chk(lrmd_step_host(self._h, *ptrs, n, dt, self._stream(stream)), "lrmd_step_host")

    def forces(self, stream=None):
        torch = self._torch
        f0 = torch.empty(self.N, dtype=torch.float64, device=self.device)
        f1 = torch.empty(self.N, dtype=torch.float64, device=self.device) if self.model == GRAV2D else None
        with torch.cuda.device(self.device):
            self._chk(lrmd_forces(self._h, f0.data_ptr(), None if f1 is None else f1.data_ptr(),
                                  self._stream(stream)), "lrmd_forces")
        return (f0, f1) if f1 is not None else f0

    def energy(self, stream=None):
        """Device tensor {K, V, a, b} (see lrmd_energy)."""
        torch = self._torch
        out = torch.empty(4, dtype=torch.float64, device=self.device)
        with torch.cuda.device(self.device):
            self._chk(lrmd_energy(self._h, out.data_ptr(), self._stream(stream)), "lrmd_energy")
        return out

    def launch_count(self) -> int:
        rc, v = lrmd_launch_count(self._h)
        self._chk(rc, "lrmd_launch_count")
        return v

    def kernel_time(self):
        """(ms_total, launches) of the dominant kernel since the last read (needs OPT_KERNEL_TIMING = 1)."""
        rc, ms, n = lrmd_kernel_time(self._h)
        self._chk(rc, "lrmd_kernel_time")
        return ms, n

    def close(self):
        if getattr(self, "_h", None):
            lrmd_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
