"""Host-side checks of the C-ABI library (no GPU needed): it loads, exports every symbol
include/lrmd.h declares, validates its arguments, resolves options, and its in-kernel sincos
arithmetic (csrc/trig.cuh, run on the host through lrmd_host_sincos) is accurate to ~1 ulp
against extended precision / mpmath (NOT against the oracle: the two share nothing)."""
import ctypes as C
import math
import os
import re

import mpmath as mp
import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HMF, RING, GRAV2D = 0, 1, 2


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "lrmd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lrmd_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lrmd):
    lib = C.CDLL(lrmd.library_path())
    declared = _declared_symbols()
    assert len(declared) >= 14
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/lrmd.h but not exported"
    assert set(declared) == set(lrmd.SYMBOLS)


def test_create_validates_arguments(lrmd):
    assert lrmd.lrmd_create(3, 10, 0.1)[0] == lrmd.EINVAL
    assert lrmd.lrmd_create(-1, 10, 0.1)[0] == lrmd.EINVAL
    assert lrmd.lrmd_create(HMF, 0, 0.0)[0] == lrmd.EINVAL
    for eps in (0.0, -1.0, float("nan"), float("inf")):
        assert lrmd.lrmd_create(RING, 10, eps)[0] == lrmd.EINVAL       # reading G6
        assert lrmd.lrmd_create(GRAV2D, 10, eps)[0] == lrmd.EINVAL
    rc, h = lrmd.lrmd_create(HMF, 10, float("nan"))                    # eps ignored for HMF
    assert rc == lrmd.OK and h
    assert lrmd.lrmd_destroy(h) == lrmd.OK
    assert lrmd.lrmd_destroy(None) == lrmd.EINVAL


def test_calls_before_state_and_workspace_are_estate(lrmd):
    rc, h = lrmd.lrmd_create(RING, 1000, 0.01)
    assert rc == lrmd.OK
    assert lrmd.lrmd_step(h, 1, 0.1) == lrmd.ESTATE
    assert lrmd.lrmd_forces(h, 256, None) == lrmd.ESTATE
    assert lrmd.lrmd_energy(h, 256) == lrmd.ESTATE
    assert lrmd.lrmd_step(None, 1, 0.1) == lrmd.EINVAL
    # NULL pattern of set_state (pointers are never dereferenced on the host)
    assert lrmd.lrmd_set_state(h, 4096, 8192, 4096, None) == lrmd.EINVAL
    assert lrmd.lrmd_set_state(h, 4096, None) == lrmd.EINVAL
    assert lrmd.lrmd_set_state(h, 4096 + 8, 8192) == lrmd.EINVAL      # misaligned
    assert lrmd.lrmd_set_state(h, 4096, 8192) == lrmd.OK
    assert lrmd.lrmd_step(h, 1, 0.1) == lrmd.ESTATE                    # workspace still missing
    rc, nbytes = lrmd.lrmd_workspace_bytes(h)
    assert rc == lrmd.OK and nbytes >= 1000 * 16 + 1000 * 8
    assert lrmd.lrmd_set_workspace(h, 4096 + 16, nbytes) == lrmd.EINVAL  # not 256-aligned
    assert lrmd.lrmd_set_workspace(h, 4096, nbytes - 1) == lrmd.EINVAL   # too small
    lrmd.lrmd_destroy(h)
    rc, h = lrmd.lrmd_create(GRAV2D, 1000, 1e-3)
    assert lrmd.lrmd_set_state(h, 4096, 8192, None, None) == lrmd.EINVAL
    assert lrmd.lrmd_set_state(h, 4096, 8192, 12288, 16384) == lrmd.OK
    lrmd.lrmd_destroy(h)


def test_options(lrmd):
    rc, h = lrmd.lrmd_create(RING, 16384, 0.01)
    assert lrmd.lrmd_get_option(h, lrmd.OPT_PAIR_SYMMETRIC) == (lrmd.OK, 1)     # chosen for this size (row N4)
    rc, W = lrmd.lrmd_get_option(h, lrmd.OPT_PAIR_CTAS)
    assert rc == lrmd.OK and W % 148 == 0                                        # workers (warps) of the symmetric kernel
    assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_SYMMETRIC, 3) == lrmd.EINVAL
    assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_SYMMETRIC, 2) == lrmd.OK        # band kernel
    assert lrmd.lrmd_get_option(h, lrmd.OPT_PAIR_SYMMETRIC) == (lrmd.OK, 2)
    assert lrmd.lrmd_get_option(h, lrmd.OPT_PAIR_CTAS) == (lrmd.OK, 296)           # CTAs, 2 per SM
    assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_SYMMETRIC, 0) == lrmd.OK        # the paper's every-ordered-pair scheme
    rc, G = lrmd.lrmd_get_option(h, lrmd.OPT_PAIR_CTAS)
    assert rc == lrmd.OK and G % 148 == 0 and G >= 148   # whole waves of the 148 SMs
    rc, slots = lrmd.lrmd_get_option(h, lrmd.OPT_PAIR_SLOTS)
    assert rc == lrmd.OK and 1 <= slots <= 64
    assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_CTAS, 3) == lrmd.OK
    assert lrmd.lrmd_get_option(h, lrmd.OPT_PAIR_CTAS) == (lrmd.OK, 3)
    assert lrmd.lrmd_get_option(h, lrmd.OPT_PAIR_SLOTS) == (lrmd.OK, 2)   # ranges longer than N: a tile meets <= 2 CTAs
    assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_CTAS, -2) == lrmd.EINVAL
    assert lrmd.lrmd_set_option(h, 99, 0) == lrmd.EINVAL
    assert lrmd.lrmd_set_option(h, lrmd.OPT_HMF_GRID, 8) == lrmd.EINVAL   # not an HMF context
    assert lrmd.lrmd_set_option(h, lrmd.OPT_HMF_VARIANT, 1) == lrmd.EINVAL
    assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_VARIANT, 9999) == lrmd.EINVAL
    assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_PRECISION, 2) == lrmd.EINVAL
    rc, b64 = lrmd.lrmd_workspace_bytes(h)
    assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_PRECISION, 1) == lrmd.OK             # Ring, fp32 pairs: half-angle stream
    assert lrmd.lrmd_workspace_bytes(h)[1] > b64
    assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_PRECISION, 0) == lrmd.OK
    rc, hh = lrmd.lrmd_create(HMF, 1000, 0.0)
    assert lrmd.lrmd_set_option(hh, lrmd.OPT_PAIR_PRECISION, 1) == lrmd.EUNSUPPORTED  # HMF has no pair arithmetic
    lrmd.lrmd_destroy(hh)
    rc, b3 = lrmd.lrmd_workspace_bytes(h)
    lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_CTAS, 32 * 6)
    rc, b6 = lrmd.lrmd_workspace_bytes(h)
    assert b6 > b3                                     # partial-force rows grow with the number of CTAs per tile
    assert lrmd.lrmd_get_option(h, lrmd.OPT_PAIR_SLOTS)[1] in (6, 7)   # 6 equal ranges per tile, boundaries not tile-aligned
    lrmd.lrmd_destroy(h)
    rc, h = lrmd.lrmd_create(GRAV2D, 5000, 1e-3)
    assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_SYMMETRIC, 0) == lrmd.OK
    rc, b0 = lrmd.lrmd_workspace_bytes(h)
    assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_PRECISION, 1) == lrmd.OK
    assert lrmd.lrmd_get_option(h, lrmd.OPT_PAIR_PRECISION) == (lrmd.OK, 1)
    rc, b1 = lrmd.lrmd_workspace_bytes(h)
    assert b1 >= b0 + 5000 * 8                         # the fp32 copy of the positions
    lrmd.lrmd_destroy(h)
    rc, h = lrmd.lrmd_create(HMF, 50_000_000, 0.0)
    rc, g = lrmd.lrmd_get_option(h, lrmd.OPT_HMF_GRID)
    assert rc == lrmd.OK and g % 148 == 0 and g >= 148   # whole waves of the 148 SMs
    lrmd.lrmd_destroy(h)
    rc, h = lrmd.lrmd_create(HMF, 5, 0.0)
    assert lrmd.lrmd_get_option(h, lrmd.OPT_HMF_GRID)[1] >= 1
    lrmd.lrmd_destroy(h)


@pytest.mark.parametrize("model", [RING, GRAV2D])
@pytest.mark.parametrize("N,G", [(1, 0), (2, 0), (700, 0), (3000, 0), (16384, 0), (65536, 0), (3000, 1), (3000, 7),
                                 (3000, 18000), (5000, 999), (1_048_576, 0), (200_003, 4321)])
def test_pair_partition_covers_every_pair_once(lrmd, model, N, G):
    """Host logic of the pair kernels' work partition (every ordered pair is computed):
    the CTAs' segments tile each i-tile's j-range [0, N) exactly once and in order, each CTA's share of
    pairs differs by at most one j-position, and slot numbers are 0..k-1 per tile with k <= PAIR_SLOTS."""
    rc, h = lrmd.lrmd_create(model, N, 1e-3)
    assert rc == lrmd.OK
    assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_SYMMETRIC, 0) == lrmd.OK    # the ordered kernels' partition
    if G:
        assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_CTAS, G) == lrmd.OK
    ctas = lrmd.lrmd_get_option(h, lrmd.OPT_PAIR_CTAS)[1]
    slots = lrmd.lrmd_get_option(h, lrmd.OPT_PAIR_SLOTS)[1]
    assert ctas >= 1 and (G == 0 or ctas == min(G, ctas))
    if ctas > 3000:     # sample the CTAs of a large grid: the first, the last and a stride in between
        pick = sorted(set([0, 1, ctas - 2, ctas - 1] + list(range(0, ctas, max(1, ctas // 997)))))
    else:
        pick = list(range(ctas))
    lengths, per_tile = [], {}
    prev_end = None
    for k in pick:
        rc, seg = lrmd.lrmd_pair_partition(h, k)
        assert rc == lrmd.OK and len(seg) >= 1
        lengths.append(int((seg[:, 2] - seg[:, 1]).sum()))
        for tile, jb, je, slot in seg:
            assert 0 <= jb < je <= N and 0 <= slot < slots
            per_tile.setdefault(int(tile), []).append((int(jb), int(je), int(slot)))
        # consecutive segments of one CTA continue into the next tile at j = 0
        for a, b in zip(seg[:-1], seg[1:]):
            assert a[2] == N and b[1] == 0 and b[0] == a[0] + 1
        if prev_end is not None and k == prev_end[0] + 1:      # consecutive CTAs continue where the last ended
            t, je = prev_end[1], prev_end[2]
            assert (seg[0][0], seg[0][1]) == ((t, je) if je < N else (t + 1, 0))
        prev_end = (k, int(seg[-1][0]), int(seg[-1][2]))
    assert max(lengths) - min(lengths) <= 1
    if len(pick) == ctas:
        itile = None
        ntiles = len(per_tile)
        assert sorted(per_tile) == list(range(ntiles))
        for t, segs in per_tile.items():
            assert segs[0][0] == 0 and segs[-1][1] == N
            assert [s[2] for s in segs] == list(range(len(segs)))
            for a, b in zip(segs[:-1], segs[1:]):
                assert a[1] == b[0]
        assert sum(lengths) == ntiles * N
    assert lrmd.lrmd_pair_partition(h, ctas)[0] == lrmd.EINVAL
    assert lrmd.lrmd_pair_partition(h, -1)[0] == lrmd.EINVAL
    lrmd.lrmd_destroy(h)
    rc, h = lrmd.lrmd_create(HMF, 100, 0.0)
    assert lrmd.lrmd_pair_partition(h, 0)[0] == lrmd.EINVAL
    lrmd.lrmd_destroy(h)


@pytest.mark.parametrize("model", [RING, GRAV2D])
@pytest.mark.parametrize("N,workers,tiles,variant", [(2048, 0, 0, -1), (5000, 7, 0, 0), (5000, 0, 3, 1), (16_384, 0, 0, -1),
                                                     (65_536, 0, 0, -1), (33, 5, 1, 0), (1000, 1, 0, 1), (300_001, 0, 0, -1)])
def test_symmetric_work_table_covers_every_unit_once(lrmd, model, N, workers, tiles, variant):
    """Host logic of the symmetric pair kernel: every (tile, chunk >= first chunk of the tile) unit
    belongs to exactly one worker, in tile-major order; launches take consecutive tiles; inside a launch the
    workers' unit counts differ by at most one."""
    rc, h = lrmd.lrmd_create(model, N, 1e-3)
    assert rc == lrmd.OK
    assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_SYMMETRIC, 1) == lrmd.OK
    if variant >= 0:
        assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_VARIANT, variant) == lrmd.OK
    if workers:
        assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_CTAS, workers) == lrmd.OK
    if tiles:
        assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_SYM_TILES, tiles) == lrmd.OK
    rc, tab = lrmd.lrmd_pair_sym_partition(h)
    assert rc == lrmd.OK and len(tab) >= 1
    T = int(tab[0, 4])
    R = T // 32
    assert T == (128 if (variant == 0 or (variant < 0 and model == RING)) else 256)   # Ring 4, 2D 8 i per lane by default
    ntiles, nchunks = -(-N // T), -(-N // 32)
    tile, chunk = 0, 0                     # the unit the next worker must start with
    launch, per_launch = 0, {}
    for t0, c0, units, b, _ in tab:
        assert (t0, c0) == (tile, chunk) and units >= 1
        assert b in (launch, launch + 1)
        if b == launch + 1:
            assert chunk == tile * R        # a launch starts at the beginning of a tile
            launch = b
        per_launch.setdefault(int(b), []).append(int(units))
        for _ in range(int(units)):
            assert tile < ntiles and tile * R <= chunk < nchunks
            chunk += 1
            if chunk == nchunks:
                tile += 1
                chunk = tile * R
    assert tile == ntiles                  # all units consumed, nothing left over
    for b, us in per_launch.items():
        assert max(us) - min(us) <= 1
        if workers:
            assert len(us) <= workers
    if tiles:
        assert len(per_launch) == -(-ntiles // tiles)
    lrmd.lrmd_destroy(h)
    rc, h = lrmd.lrmd_create(model, 100, 1e-3)          # below 2048 the ordered kernel is chosen: empty table
    rc, tab = lrmd.lrmd_pair_sym_partition(h)
    assert rc == lrmd.OK and len(tab) == 0
    lrmd.lrmd_destroy(h)


def test_strerror_and_coefficients(lrmd):
    assert lrmd.strerror(0) == "ok"
    for code in (-1, -2, -3, -4, -77):
        assert isinstance(lrmd.strerror(code), str) and lrmd.strerror(code)
    B0, B1, D0, D1 = lrmd.lrmd_coefficients()
    # Yoshida's order conditions (ref. [33] of the paper; reading G4), not the oracle's numbers
    assert abs(2 * D0 + D1 - 1) < 1e-15 and abs(2 * (B0 + B1) - 1) < 1e-15
    assert abs(2 * D0 ** 3 + D1 ** 3) < 1e-14
    assert abs(B0 - D0 / 2) < 1e-16 and abs(B1 - (D0 + D1) / 2) < 1e-16


def _ulp_err(got, exact_ld):
    """|got - exact| in units of ulp(exact) (fp64), exact given in extended precision."""
    e = np.asarray(exact_ld, dtype=np.longdouble)
    ulp = np.spacing(np.abs(e).astype(np.float64)).astype(np.longdouble)
    return np.abs(got.astype(np.longdouble) - e) / ulp


@pytest.mark.parametrize("lo,hi", [(-0.8, 0.8), (-4.0, 4.0), (-100.0, 100.0), (-1e6, 1e6)])
def test_kernel_sincos_accuracy_bulk(lrmd, lo, hi):
    """x87 long double sin/cos (64-bit mantissa) as the reference on 200k points per range."""
    if np.finfo(np.longdouble).nmant < 63:
        pytest.skip("no extended-precision long double on this host")
    rng = np.random.default_rng(17)
    x = rng.uniform(lo, hi, 200_000)
    s, c = lrmd.lrmd_host_sincos(x)
    xl = x.astype(np.longdouble)
    es, ec = _ulp_err(s, np.sin(xl)), _ulp_err(c, np.cos(xl))
    # near zeros of sin/cos the error is bounded absolutely (2^-53 scale), not in ulps of the result
    big_s, big_c = np.abs(s) > 1e-3, np.abs(c) > 1e-3
    assert es[big_s].max() < 1.5 and ec[big_c].max() < 1.5
    assert np.abs(s.astype(np.longdouble) - np.sin(xl)).max() < 2.5e-16
    assert np.abs(c.astype(np.longdouble) - np.cos(xl)).max() < 2.5e-16
    assert np.all(np.abs(s * s + c * c - 1) < 1e-15)


def test_kernel_sincos_special_points_mpmath(lrmd):
    mp.mp.dps = 40
    pts = [0.0, -0.0, 1e-300, 1e-9, math.pi / 4, -math.pi / 4, math.pi / 2, math.pi, 3 * math.pi / 2, 2 * math.pi,
           0.7853981633974484, 0.7853981633974482, 1.5, -1.5, 22.0, 355.0, 1e5 * math.pi, 2.0 ** 29, -(2.0 ** 29),
           2.0 ** 30 - 1.0, 2.0 ** 30, 1e12, -1e15]
    x = np.array(pts)
    s, c = lrmd.lrmd_host_sincos(x)
    for xi, si, ci in zip(pts, s, c):
        es, ec = mp.sin(mp.mpf(xi)), mp.cos(mp.mpf(xi))
        assert abs(mp.mpf(float(si)) - es) < mp.mpf(2) ** -52, (xi, si, es)
        assert abs(mp.mpf(float(ci)) - ec) < mp.mpf(2) ** -52, (xi, ci, ec)
    assert s[0] == 0.0 and c[0] == 1.0
    sn, cn = lrmd.lrmd_host_sincos(np.array([float("nan"), float("inf")]))
    assert np.all(np.isnan(sn)) and np.all(np.isnan(cn))


@pytest.mark.gpu
@pytest.mark.parametrize("how", ["set_option", "set_shard"])
def test_reresolving_a_symmetric_context_unbinds_the_workspace(lrmd, how):
    """Raw C ABI, no Context object: a RING context with N = 4096 uses the symmetric kernel, whose work tables live in
    the workspace.  lrmd_set_option / lrmd_set_shard after lrmd_set_workspace rebuild those tables on the host, so the
    context must return to 'workspace not set' (LRMD_ESTATE) instead of launching with stale table pointers; after a
    re-bind the step runs and matches a fresh context bit for bit."""
    import numpy as np
    import torch
    assert torch.cuda.is_available()
    N = 4096
    rng = np.random.default_rng(5)
    th0, p0 = rng.uniform(-1, 1, N), rng.uniform(-0.3, 0.3, N)

    def fresh():
        rc, h = lrmd.lrmd_create(RING, N, 0.01)
        assert rc == lrmd.OK
        rc, nbytes = lrmd.lrmd_workspace_bytes(h)
        ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
        ptr = (ws.data_ptr() + 255) // 256 * 256
        assert lrmd.lrmd_set_workspace(h, ptr, nbytes) == lrmd.OK
        th = torch.tensor(th0, device="cuda")
        p = torch.tensor(p0, device="cuda")
        assert lrmd.lrmd_set_state(h, th.data_ptr(), p.data_ptr()) == lrmd.OK
        return h, ws, ptr, nbytes, th, p

    h, ws, ptr, nbytes, th, p = fresh()
    assert lrmd.lrmd_get_option(h, lrmd.OPT_PAIR_SYMMETRIC) == (lrmd.OK, 1)
    if how == "set_option":
        assert lrmd.lrmd_set_option(h, lrmd.OPT_GRAPH, 0) == lrmd.OK
    else:
        assert lrmd.load().lrmd_set_shard(h, N, 0, None, None, None) == lrmd.OK
    assert lrmd.lrmd_step(h, 1, 0.01) == lrmd.ESTATE
    rc, nbytes2 = lrmd.lrmd_workspace_bytes(h)
    assert rc == lrmd.OK and nbytes2 <= nbytes
    assert lrmd.lrmd_set_workspace(h, ptr, nbytes) == lrmd.OK
    assert lrmd.lrmd_step(h, 2, 0.01) == lrmd.OK
    torch.cuda.synchronize()
    h2, ws2, _, _, th2, p2 = fresh()
    assert lrmd.lrmd_step(h2, 2, 0.01) == lrmd.OK
    torch.cuda.synchronize()
    assert torch.equal(th, th2) and torch.equal(p, p2)
    lrmd.lrmd_destroy(h)
    lrmd.lrmd_destroy(h2)


@pytest.mark.parametrize("model,N,workers,height,variant", [
    (GRAV2D, 65_536, 0, 0, -1), (GRAV2D, 1_048_576, 0, 0, -1), (RING, 100_003, 0, 0, -1), (GRAV2D, 50_000, 7, 3, 0),
    (RING, 2049, 0, 0, 1), (GRAV2D, 33, 0, 0, -1), (GRAV2D, 300_000, 1, 0, -1), (RING, 70_001, 1000, 2, 0),
    (GRAV2D, 4_000_000, 0, 0, -1),
])
def test_band_partition_covers_every_column_once_and_is_balanced(lrmd, model, N, workers, height, variant):
    """Host logic of the band kernel (LRMD_OPT_PAIR_SYMMETRIC = 2): the pieces of a band are consecutive column ranges
    that cover [first row of the band, N) exactly once; pieces are handed to the workers in order; the workers'
    weights (FP64 instructions: 11 / 12 per pair above the diagonal block, 9 / 11 inside it) differ by at most one
    chunk column of the tallest band."""
    rc, h = lrmd.lrmd_create(model, N, 1e-3)
    assert rc == lrmd.OK
    assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_SYMMETRIC, 2) == lrmd.OK
    if variant >= 0:
        assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_VARIANT, variant) == lrmd.OK
    if workers:
        assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_CTAS, workers) == lrmd.OK
    if height:
        assert lrmd.lrmd_set_option(h, lrmd.OPT_PAIR_BAND_HEIGHT, height) == lrmd.OK
    rc, v = lrmd.lrmd_get_option(h, lrmd.OPT_PAIR_SYMMETRIC)
    assert rc == lrmd.OK and v == 2
    rc, tab = lrmd.lrmd_pair_band_partition(h)
    assert rc == lrmd.OK and len(tab) >= 1
    IB, P = int(tab[0, 6]), int(tab[0, 7])
    R = 4 if variant == 0 else 8           # 8 rows per lane by default, for both models
    assert IB == 8 * 32 * R and P == (workers or 296)
    JB = IB // 32
    nIB, nchunks = -(-N // IB), -(-N // 32)
    wsym, wdiag = (12, 11) if model == RING else (11, 9)
    # bands in order, each covered once by consecutive pieces
    band, blk_next, col = -1, 0, None
    weights = [0] * P
    last_worker = 0
    for b, c0, c1, w, blk0, nblk, _, _ in (tuple(int(x) for x in row) for row in tab):
        assert 0 <= w < P and w >= last_worker
        last_worker = w
        if b != band:
            if band >= 0:
                assert col == nchunks                  # the previous band reached the last column
            assert b == band + 1 and blk0 == blk_next and nblk >= 1
            band, blk_next, col = b, blk0 + nblk, blk0 * JB
            if height:
                assert nblk == min(height, nIB - blk0)
        assert c0 == col and c1 > c0 and c1 <= nchunks
        col = c1
        for c in range(c0, c1):
            blk = c // JB
            weights[w] += wsym * min(max(blk - blk0, 0), nblk) + (wdiag if blk0 <= blk < blk0 + nblk else 0)
    assert col == nchunks and blk_next == nIB
    hb_max = max(int(r[5]) for r in tab)
    busy = [x for x in weights if x > 0]
    assert max(busy) - min(busy) <= 2 * (wsym * hb_max) or len(busy) < P
    expected = 0
    for blk0, nblk in sorted({(int(r[4]), int(r[5])) for r in tab}):
        for blk in range(blk0, nIB):
            nch = min((blk + 1) * JB, nchunks) - blk * JB
            expected += (wsym * min(blk - blk0, nblk) + (wdiag if blk < blk0 + nblk else 0)) * nch
    assert sum(weights) == expected
    rc, nbytes = lrmd.lrmd_workspace_bytes(h)
    assert rc == lrmd.OK
    if N == 1_048_576:
        assert nbytes < 1_000_000_000          # one launch per force evaluation on < 1 GB of scratch (was 3.56 GB, 128 launches)
    lrmd.lrmd_destroy(h)
    rc, h = lrmd.lrmd_create(model, 4096, 1e-3)          # below 49,152 the warp-level kernel is the default: empty table
    rc, tab = lrmd.lrmd_pair_band_partition(h)
    assert rc == lrmd.OK and len(tab) == 0
    lrmd.lrmd_destroy(h)
