// pair_kernels.cuh — Ring and 2D self-gravitating models (section 3.2):
// all-pairs force and potential-energy kernels, bound by the FP64 pipe issue rate.
//
// The paper's tile scheme (after GPU Gems 3): CTA l owns N_threads i-particles,
// loops over N/N_threads j-tiles staged in shared memory, one i per thread.  What is kept: the
// j-tile in shared memory, every ordered pair computed (no Newton's third law), an
// approximate reciprocal (square root).  What is new for sm_100a:
//   * R i-particles per thread in registers, so one broadcast LDS.128 of a packed (cos,sin) /
//     (x,y) j-element feeds R pair evaluations (the smem port is idle 95 % of the time);
//   * the j-stream is a packed double2 array written by the update kernel, and tiles are brought
//     in by 1-D TMA bulk copies (cp.async.bulk -> UBLKCP) into a 2-stage ring guarded by mbarriers,
//     issued by one thread while the CTA computes on the other stage;
//   * a balanced 1-D partition of the flattened (i-tile, j) space over 148 x MINB x waves CTAs
//     (PairPart below): N/ITILE alone does not fill 148 SMs for N = 16,384; each CTA writes one
//     partial force row per tile it touches and the update kernel adds a tile's partial rows in
//     slot order (deterministic, no atomics);
//   * MUFU.RCP64H / MUFU.RSQ64H seed (~2^-20) + one cubic fp64 correction instead of rsqrt():
//     2D 9 FP64 instructions per pair (7 DFMA + 2 DADD), Ring 11 (7 DFMA + 4 DMUL).
// The j = i pair is computed like any other (PAPER.md:105 loops over all k): for eps > 0 it
// contributes exactly 0 in 2D (dx = dy = 0) and a rounding-level term in the Ring rewrite eq.(9)
// (s_i c_i - c_i s_i evaluated with one FMA), which the epilogue removes again.
#pragma once

#include <type_traits>

#include "common.cuh"
#include "trig.cuh"

namespace lrmd {

// Launch shape of the pair kernels: THREADS threads per CTA, R i-particles per thread (i-tile =
// THREADS x R), TJ j-elements per shared-memory stage, MINB resident CTAs per SM (register cap),
// UNROLL j-iterations unrolled in the inner loop.
template <int THREADS_, int R_, int TJ_, int MINB_, int UNROLL_>
struct PairCfg {
    static constexpr int THREADS = THREADS_, R = R_, TJ = TJ_, MINB = MINB_, UNROLL = UNROLL_;
    static constexpr int ITILE = THREADS_ * R_;
};

// Work partition.  The N x N pair rectangle is cut into i-tiles of ITILE rows; the (i-tile, j)
// space is flattened to L = itiles x N positions (position = tile * N + j) and divided into G
// contiguous ranges of equal length (the first r ranges hold q + 1 positions, the others q), one
// per CTA.  With G = 148 x MINB x waves every CTA carries the same number of pairs whatever N is
// (N = 16,384 does not fill 148 SMs with whole tiles: SURVEY.md hard part 3).  A CTA's range
// crosses at most ceil(q / N) tile boundaries; for each tile it touches it writes one partial
// force row partial[slot][i], slot = cta - (first CTA touching the tile), and the update kernel
// adds a tile's slots in slot order: deterministic, no atomics.
struct PairPart {
    long long N;      // particles = j-elements of the packed stream (all of them, on every rank)
    long long Ni;     // rows (i-particles) this context owns: global indices i0 .. i0 + Ni - 1
    long long i0;     //   (Ni = N, i0 = 0 unless the context is one shard of a multi-GPU run)
    long long q, r;   // range lengths: q + 1 for CTAs < r, q for the others (q >= 1)
    int G;            // CTAs
    int itile;        // rows per i-tile
};
__host__ __device__ __forceinline__ long long part_bound(const PairPart& P, long long k) {
    return k * P.q + (k < P.r ? k : P.r);
}
__host__ __device__ __forceinline__ long long part_owner(const PairPart& P, long long pos) {
    const long long big = P.r * (P.q + 1);
    return pos < big ? pos / (P.q + 1) : P.r + (pos - big) / P.q;
}
// slots of tile t: CTAs first..last touch it
__host__ __device__ __forceinline__ void part_tile_ctas(const PairPart& P, long long t, long long& first,
                                                        long long& last) {
    first = part_owner(P, t * P.N);
    last = part_owner(P, (t + 1) * P.N - 1);
}

// ---- per-pair arithmetic ---------------------------------------------------------------------------

// 2D: F_i += (r_i - r_j) / (|r_i - r_j|^2 + eps)   [prefactor -2/N applied once per i]
__device__ __forceinline__ void grav_pair(double xi, double yi, double2 q, double eps, double& fx, double& fy) {
    const double dx = xi - q.x;
    const double dy = yi - q.y;
    double r2 = fma(dx, dx, eps);
    r2 = fma(dy, dy, r2);
    const double y0 = rcp_seed(r2);            // MUFU.RCP64H, rel. error d ~ 2^-20
    const double e = fma(-r2, y0, 1.0);        // e = -d (exact up to one rounding)
    const double t = fma(e, e, e);             // e + e^2
    const double y = fma(y0, t, y0);           // y0 (1 + e + e^2) = (1/r2)(1 - e^3)
    fx = fma(dx, y, fx);
    fy = fma(dy, y, fy);
}

// d^(-1/2) from the seed with one cubic correction: y0 (1 + e/2 + 3 e^2/8), e = 1 - d y0^2
__device__ __forceinline__ double rsqrt_refined(double d) {
    const double y0 = rsqrt_seed(d);           // MUFU.RSQ64H
    const double t = d * y0;
    const double e = fma(-t, y0, 1.0);
    const double g = fma(0.375, e, 0.5);
    const double ye = y0 * e;
    return fma(ye, g, y0);
}

// Ring eq.(9): the pair term num d^(-3/2) as a product c * p of
//   c = num y0^3                      (y0 = MUFU seed of d^(-1/2), relative error ~2^-20)
//   p = 1 + (3/2) e + (15/8) e^2      (e = 1 - d y0^2;  (1 - e)^(-3/2) = p + O(e^3), |e^3| < 2^-56)
// 11 FP64 instructions per pair with the accumulating FMA (7 DFMA + 4 DMUL) + 1 MUFU.RSQ64H:
// num 2, d 2, y0^2 1, e 1, num y0 1, (num y0) y0^2 1, p 2, accumulate 1.
__device__ __forceinline__ void ring_pair_parts(double ci, double si, double2 q, double onepe, double& c, double& p) {
    const double num = fma(si, q.x, -(ci * q.y));          // s_i c_j - c_i s_j
    const double d = fma(-si, q.y, fma(-ci, q.x, onepe));  // 1 + eps - c_i c_j - s_i s_j
    const double y0 = rsqrt_seed(d);
    const double b = y0 * y0;
    const double e = fma(-d, b, 1.0);
    const double a = num * y0;
    c = a * b;
    const double g = fma(1.875, e, 1.5);
    p = fma(g, e, 1.0);
}

// ---- j-tile pipeline ----------------------------------------------------------------------------------

template <typename T, int TJ>
struct PairSmem {
    alignas(128) T tile[2][TJ];
    alignas(8) uint64_t full[2];
};

// Two-stage ring of j-tiles filled by 1-D TMA bulk copies.  init() once per CTA; run() may be
// called for several j-ranges in turn (every copy it issues is consumed before it returns, so the
// barrier phases carry over).
template <typename T, int TJ>
struct JTilePipe {
    PairSmem<T, TJ>& sm;
    uint32_t phases = 0u;   // bit s = parity the next wait on stage s expects
    __device__ __forceinline__ explicit JTilePipe(PairSmem<T, TJ>& s) : sm(s) {}
    __device__ __forceinline__ void init() {
        if (threadIdx.x == 0) {
            mbar_init(&sm.full[0], 1);
            mbar_init(&sm.full[1], 1);
            mbar_fence_init();
        }
        __syncthreads();
    }
    // Calls body(tile_ptr, count, j0) for consecutive tiles of [jbeg, jend) of the packed j-stream.
    // Bulk copies move multiples of 16 bytes from 16-byte aligned addresses: for 8-byte elements
    // (the fp32 stream) the copies start at the even index at or below jbeg and end at the even
    // index at or above jend (the array is padded to an even length), and body() is handed the
    // valid part only.
    template <typename Body>
    __device__ __forceinline__ void run(const T* __restrict__ js, long long jbeg, long long jend, Body body) {
        constexpr long long A = 16 / sizeof(T);              // elements per 16 bytes: 1 (double2) or 2 (float2)
        static_assert(A >= 1 && TJ % A == 0, "tile length must keep the copies aligned");
        const long long ja = jbeg & ~(A - 1);
        const long long je = (jend + A - 1) & ~(A - 1);
        const int ntiles = (int)((je - ja + TJ - 1) / TJ);
        if (threadIdx.x == 0 && ntiles > 0) {
            const long long c0 = (je - ja < TJ) ? (je - ja) : TJ;
            mbar_expect_tx(&sm.full[0], (uint32_t)(c0 * sizeof(T)));
            bulk_g2s(sm.tile[0], js + ja, (uint32_t)(c0 * sizeof(T)), &sm.full[0]);
        }
        for (int t = 0; t < ntiles; ++t) {
            const int s = t & 1;
            const long long j0 = ja + (long long)t * TJ;
            if (threadIdx.x == 0 && t + 1 < ntiles) {
                // stage s^1 was consumed in iteration t-1; every thread passed the barrier that ended it
                const long long j1 = j0 + TJ;
                const long long c1 = (je - j1 < TJ) ? (je - j1) : TJ;
                mbar_expect_tx(&sm.full[s ^ 1], (uint32_t)(c1 * sizeof(T)));
                bulk_g2s(sm.tile[s ^ 1], js + j1, (uint32_t)(c1 * sizeof(T)), &sm.full[s ^ 1]);
            }
            mbar_wait(&sm.full[s], (phases >> s) & 1u);
            phases ^= 1u << s;
            const int skip = (A > 1 && t == 0) ? (int)(jbeg - ja) : 0;
            const int cnt = (int)((jend - j0 < TJ) ? (jend - j0) : TJ);
            body(sm.tile[s] + skip, cnt - skip, j0 + skip);
            __syncthreads();
        }
    }
};

// Iterates over the (i-tile, j-range) segments of CTA k's range: next() yields the pairs
// (i in tile) x (jbeg <= j < jend) and the partial force row `slot` they are added into.
struct PairSegments {
    long long pos, end, k;
    __host__ __device__ __forceinline__ PairSegments(const PairPart& P, long long cta)
        : pos(part_bound(P, cta)), end(part_bound(P, cta + 1)), k(cta) {}
    __host__ __device__ __forceinline__ bool next(const PairPart& P, long long& tile, long long& jbeg, long long& jend,
                                                  int& slot) {
        if (pos >= end) return false;
        tile = pos / P.N;
        jbeg = pos - tile * P.N;
        jend = (end - pos < P.N - jbeg) ? jbeg + (end - pos) : P.N;
        slot = (int)(k - part_owner(P, tile * P.N));
        pos += jend - jbeg;
        return true;
    }
};

// ---- force kernels (rows a-P1r, a-P1g) --------------------------------------------------------------

// grid = P.G CTAs.  partial0/1: [slots][N] partial forces (with the model's prefactor).
template <int MODEL, typename CFG>
__global__ void __launch_bounds__(CFG::THREADS, CFG::MINB)
pair_force_kernel(const double2* __restrict__ js, PairPart P, double eps, double pre,
                  double* __restrict__ partial0, double* __restrict__ partial1) {
    constexpr int R = CFG::R, THREADS = CFG::THREADS, TJ = CFG::TJ;
    __shared__ PairSmem<double2, TJ> sm;
    JTilePipe<double2, TJ> pipe(sm);
    pipe.init();
    const long long N = P.Ni;     // rows of this context; partial rows have this stride
    const double onepe = 1.0 + eps;

    PairSegments segs(P, blockIdx.x);
    long long tile, jbeg, jend;
    int slot;
    while (segs.next(P, tile, jbeg, jend, slot)) {
        const long long ibase = tile * CFG::ITILE + threadIdx.x;
        double a[R], b[R], f0[R], f1[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long i = ibase + (long long)r * THREADS;
            const double2 q = (i < N) ? js[P.i0 + i] : make_double2(0.0, 0.0);
            a[r] = q.x;
            b[r] = q.y;
            f0[r] = 0.0;
            f1[r] = 0.0;
        }
        auto pair = [&](const double2 q) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if (MODEL == 2) {
                    grav_pair(a[r], b[r], q, eps, f0[r], f1[r]);
                } else {
                    double c, p;
                    ring_pair_parts(a[r], b[r], q, onepe, c, p);
                    f0[r] = fma(c, p, f0[r]);
                }
            }
        };
        pipe.run(js, jbeg, jend, [&](const double2* tl, int cnt, long long) {
            if (cnt == TJ) {
                // the next group's j-elements are loaded (broadcast LDS.128) before this group's arithmetic
                constexpr int U = CFG::UNROLL;
                double2 qn[U];
#pragma unroll
                for (int u = 0; u < U; ++u) qn[u] = tl[u];
#pragma unroll 1
                for (int jj = 0; jj < TJ; jj += U) {
                    double2 q[U];
#pragma unroll
                    for (int u = 0; u < U; ++u) q[u] = qn[u];
                    const int nx = (jj + U < TJ) ? jj + U : 0;   // last group: harmless reload of group 0
#pragma unroll
                    for (int u = 0; u < U; ++u) qn[u] = tl[nx + u];
#pragma unroll
                    for (int u = 0; u < U; ++u) pair(q[u]);
                }
            } else {
#pragma unroll 2
                for (int jj = 0; jj < cnt; ++jj) pair(tl[jj]);
            }
        });
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long i = ibase + (long long)r * THREADS;
            if (i < N) {
                if (MODEL == 1) {
                    if (P.i0 + i >= jbeg && P.i0 + i < jend) {   // remove the rounding-level j = i term again
                        double c, p;
                        ring_pair_parts(a[r], b[r], make_double2(a[r], b[r]), onepe, c, p);
                        f0[r] -= __dmul_rn(c, p);   // the rounded product, so that N = 1 gives exactly 0
                    }
                    partial0[(long long)slot * N + i] = pre * f0[r];
                } else {
                    partial0[(long long)slot * N + i] = pre * f0[r];
                    partial1[(long long)slot * N + i] = pre * f1[r];
                }
            }
        }
    }
}

// ---- 2D force, fp32 pair arithmetic ----------------------------------
// The paper's mixed-precision variant (paraphrased): all data stay in double precision in global
// memory, each position component is stored in single precision in shared memory, the force between two particles
// "is then computed in single precision but added in a double precision variable".  Here: a second packed stream float2 xy32[] (positions rounded to fp32 by the update
// kernel), pair terms in fp32 (4 FADD/FFMA for dx, dy, r^2 + eps; MUFU.RCP; 2 FFMA), summed in fp32
// over at most kF32Chunk consecutive j and then added to the fp64 accumulators (reading G16: a
// pure fp32 accumulator over 1e6 terms would miss the 1e-5 tolerance).  Bound by the special-
// function unit: one MUFU.RCP per pair at 16 lanes per SM per clock.
constexpr int kF32Chunk = 32;

__device__ __forceinline__ float rcp_f32(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <typename CFG>
__global__ void __launch_bounds__(CFG::THREADS, CFG::MINB)
grav_force_f32_kernel(const float2* __restrict__ js32, PairPart P, float eps, double pre,
                      double* __restrict__ partial0, double* __restrict__ partial1) {
    constexpr int R = CFG::R, THREADS = CFG::THREADS, TJ = CFG::TJ;
    __shared__ PairSmem<float2, TJ> sm;
    JTilePipe<float2, TJ> pipe(sm);
    pipe.init();
    const long long N = P.Ni;

    PairSegments segs(P, blockIdx.x);
    long long tile, jbeg, jend;
    int slot;
    while (segs.next(P, tile, jbeg, jend, slot)) {
        const long long ibase = tile * CFG::ITILE + threadIdx.x;
        float a[R], b[R];
        double f0[R], f1[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long i = ibase + (long long)r * THREADS;
            const float2 q = (i < N) ? js32[P.i0 + i] : make_float2(0.f, 0.f);
            a[r] = q.x;
            b[r] = q.y;
            f0[r] = 0.0;
            f1[r] = 0.0;
        }
        pipe.run(js32, jbeg, jend, [&](const float2* tl, int cnt, long long) {
            for (int c0 = 0; c0 < cnt; c0 += kF32Chunk) {
                const int m = (cnt - c0 < kF32Chunk) ? (cnt - c0) : kF32Chunk;
                float sx[R], sy[R];
#pragma unroll
                for (int r = 0; r < R; ++r) sx[r] = sy[r] = 0.f;
                auto pair = [&](const float2 q) {
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const float dx = a[r] - q.x;
                        const float dy = b[r] - q.y;
                        const float r2 = fmaf(dy, dy, fmaf(dx, dx, eps));
                        const float w = rcp_f32(r2);
                        sx[r] = fmaf(dx, w, sx[r]);
                        sy[r] = fmaf(dy, w, sy[r]);
                    }
                };
                if (m == kF32Chunk) {
#pragma unroll 8
                    for (int jj = 0; jj < kF32Chunk; ++jj) pair(tl[c0 + jj]);   // broadcast LDS.64
                } else {
                    for (int jj = 0; jj < m; ++jj) pair(tl[c0 + jj]);
                }
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    f0[r] += (double)sx[r];
                    f1[r] += (double)sy[r];
                }
            }
        });
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long i = ibase + (long long)r * THREADS;
            if (i < N) {
                partial0[(long long)slot * N + i] = pre * f0[r];
                partial1[(long long)slot * N + i] = pre * f1[r];
            }
        }
    }
}

// ---- Ring force, fp32 pair arithmetic ---------------------------------------
// "computing the force between the two particles using single precision arithmetic do not compromise the overall
// accuracy".  Eq.(9)'s denominator 1 + eps - c_i c_j - s_i s_j cancels to ~eps for close
// pairs: rounded to fp32 its relative error is ~1.5e-7 / eps, i.e. ~2e-5 on the pair term at eps = 0.01 — above the
// 1e-5 A_i tolerance.  The half-angle form has no cancellation: with (ch, sh)_i = (cos, sin)(theta_i / 2) stored in fp32,
//     S = sin((ti - tj)/2) = sh_i ch_j - ch_i sh_j,   C = cos((ti - tj)/2) = ch_i ch_j + sh_i sh_j,
//     1 - cos(ti - tj) = 2 S^2,   sin(ti - tj) = 2 S C,   term = 2 S C (eps + 2 S^2)^(-3/2),
// every operation in fp32 (12 FADD/FMUL/FFMA + MUFU.RSQ per pair); the relative error of eps + 2 S^2 stays ~1e-7.
// S uses two rounded products, so j = i gives exactly 0.  Sums as in grav_force_f32_kernel (reading G16): fp32 over at
// most kF32Chunk consecutive j, then added to the fp64 accumulator.
__device__ __forceinline__ float rsqrt_f32(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <typename CFG>
__global__ void __launch_bounds__(CFG::THREADS, CFG::MINB)
ring_force_f32_kernel(const float2* __restrict__ hs32, PairPart P, float eps, double pre, double* __restrict__ partial0) {
    constexpr int R = CFG::R, THREADS = CFG::THREADS, TJ = CFG::TJ;
    __shared__ PairSmem<float2, TJ> sm;
    JTilePipe<float2, TJ> pipe(sm);
    pipe.init();
    const long long N = P.Ni;

    PairSegments segs(P, blockIdx.x);
    long long tile, jbeg, jend;
    int slot;
    while (segs.next(P, tile, jbeg, jend, slot)) {
        const long long ibase = tile * CFG::ITILE + threadIdx.x;
        float ch[R], sh[R];
        double f0[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long i = ibase + (long long)r * THREADS;
            const float2 q = (i < N) ? hs32[P.i0 + i] : make_float2(1.f, 0.f);
            ch[r] = q.x;
            sh[r] = q.y;
            f0[r] = 0.0;
        }
        pipe.run(hs32, jbeg, jend, [&](const float2* tl, int cnt, long long) {
            for (int c0 = 0; c0 < cnt; c0 += kF32Chunk) {
                const int m = (cnt - c0 < kF32Chunk) ? (cnt - c0) : kF32Chunk;
                float acc[R];
#pragma unroll
                for (int r = 0; r < R; ++r) acc[r] = 0.f;
                auto pair = [&](const float2 q) {
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const float S = __fsub_rn(__fmul_rn(sh[r], q.x), __fmul_rn(ch[r], q.y));
                        const float C = fmaf(ch[r], q.x, sh[r] * q.y);
                        const float S2 = S + S;
                        const float d = fmaf(S2, S, eps);
                        const float y = rsqrt_f32(d);
                        const float w = (S2 * C) * y;
                        acc[r] = fmaf(w, y * y, acc[r]);
                    }
                };
                if (m == kF32Chunk) {
#pragma unroll 8
                    for (int jj = 0; jj < kF32Chunk; ++jj) pair(tl[c0 + jj]);   // broadcast LDS.64
                } else {
                    for (int jj = 0; jj < m; ++jj) pair(tl[c0 + jj]);
                }
#pragma unroll
                for (int r = 0; r < R; ++r) f0[r] += (double)acc[r];
            }
        });
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long i = ibase + (long long)r * THREADS;
            if (i < N) partial0[(long long)slot * N + i] = pre * f0[r];
        }
    }
}

// ---- symmetric force kernels: Newton's third law ------------------------------------
// The paper computes every ordered pair ("the symmetry ... would introduce unnecessary complications with no
// significant speed gain").  On an FP64-issue-bound B200 kernel halving the pair evaluations is
// the one large factor left: per UNORDERED pair 2D 7 + 2 + 2 = 11 and Ring 11 + 2 = 13 FP64 instructions, i.e.
// 5.5 / 6.5 per ordered pair instead of 9 / 11.
// Scheme (one warp = one worker, no shared memory, no barriers): a warp owns an i-tile of 32 x R particles in
// registers (R per lane) and walks over chunks of 32 j-particles with index beyond its tile; lane l loads
// j = 32 c + l, and the j-packet (position + the force it collects) travels once around the warp by
// shuffles: in each of 32 steps every lane evaluates its R i-particles against the packet it holds, adds
// +f to its own i-accumulators and -f to the packet.  After 32 steps the packet is home again carrying the
// force of the whole i-tile on j: it is written to jpart[tile][j].  The chunks of the tile itself are walked
// the same way but only the i-side is kept (each ordered pair of the tile is met once that way).
// Work = (tile, chunk) units in tile-major order, divided evenly over the warps (table built on the host);
// a warp's i-side sums go to ipart[slot][i] like the ordered kernel's, and the consumer adds a
// particle's ipart rows and the jpart rows of all lower tiles in a fixed order: deterministic, no atomics.
struct SymPart {
    long long N;
    int T;            // particles per i-tile = 32 R
    int ntiles;       // ceil(N / T)
    int nchunks;      // ceil(N / 32)
    int G;            // workers (warps) of this launch
    int w0;           // index of this launch's first worker in wstart (launches = batches of tiles tile0 .. tile1 - 1,
    int tile0, tile1; //   so that the j-side rows of one launch fit their scratch: jpart[tile - tile0][j])
    const int4* wstart;    // first unit of every worker: (tile, chunk, number of units, 0)
    const int2* tile_rng;  // [ntiles] first and last (global) worker touching the tile
};

constexpr int kSymThreads = 128;   // 4 independent workers per CTA

template <int MODEL, int R, bool MASK, bool DIAG>
__device__ __forceinline__ void sym_chunk(const double (&a)[R], const double (&b)[R], const bool (&vi)[R],
                                          double (&f0)[R], double (&f1)[R], double2 q, bool vq, double eps,
                                          double onepe, double& g0, double& g1) {
    const unsigned lane = threadIdx.x & 31u, src = (lane + 31u) & 31u;   // the packet moves to lane + 1
#pragma unroll 8
    for (int s = 0; s < 32; ++s) {
        // the position part of the next packet is requested before this step's arithmetic; the force part
        // is summed per step (h0, h1) and joins the travelling sum only at the end, so that the shuffle
        // latency of g never sits on the pair arithmetic's dependency chain
        const double qnx = __shfl_sync(0xffffffffu, q.x, src);
        const double qny = __shfl_sync(0xffffffffu, q.y, src);
        const bool vqn = MASK ? (__shfl_sync(0xffffffffu, (int)vq, src) != 0) : true;
        double h0 = 0.0, h1 = 0.0;
        // The R pair evaluations of a step are written stage by stage over groups of 4, so that the four
        // dependency chains (difference -> r^2 -> MUFU seed -> correction -> accumulate) are interleaved in
        // the instruction stream: written pair by pair, the compiler reused one register set and ran the
        // chains back to back, every correction waiting for its own seed.
#pragma unroll
        for (int r0 = 0; r0 < R; r0 += 4) {
            if (MODEL == 2) {
                double dx[4], dy[4], r2[4], y0[4], y[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    dx[k] = a[r0 + k] - q.x;
                    dy[k] = b[r0 + k] - q.y;
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) r2[k] = fma(dy[k], dy[k], fma(dx[k], dx[k], eps));
#pragma unroll
                for (int k = 0; k < 4; ++k) y0[k] = rcp_seed(r2[k]);
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const double e = fma(-r2[k], y0[k], 1.0);
                    y[k] = fma(e, e, e);
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    y[k] = fma(y0[k], y[k], y0[k]);
                    if (MASK) y[k] = (vi[r0 + k] && vq) ? y[k] : 0.0;
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    f0[r0 + k] = fma(dx[k], y[k], f0[r0 + k]);
                    f1[r0 + k] = fma(dy[k], y[k], f1[r0 + k]);
                    if (!DIAG) {
                        h0 = fma(-dx[k], y[k], h0);
                        h1 = fma(-dy[k], y[k], h1);
                    }
                }
            } else {
                double num[4], d[4], y0[4], c[4], p[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    num[k] = fma(b[r0 + k], q.x, -(a[r0 + k] * q.y));                 // s_i c_j - c_i s_j
                    d[k] = fma(-b[r0 + k], q.y, fma(-a[r0 + k], q.x, onepe));      // 1 + eps - c_i c_j - s_i s_j
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) y0[k] = rsqrt_seed(d[k]);
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const double bb = y0[k] * y0[k];
                    const double e = fma(-d[k], bb, 1.0);
                    c[k] = (num[k] * y0[k]) * bb;
                    p[k] = fma(fma(1.875, e, 1.5), e, 1.0);
                    if (MASK) c[k] = (vi[r0 + k] && vq) ? c[k] : 0.0;
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    f0[r0 + k] = fma(c[k], p[k], f0[r0 + k]);
                    if (!DIAG) h0 = fma(-c[k], p[k], h0);
                }
            }
        }
        if (!DIAG) {
            g0 = __shfl_sync(0xffffffffu, g0 + h0, src);
            if (MODEL == 2) g1 = __shfl_sync(0xffffffffu, g1 + h1, src);
        }
        q.x = qnx;
        q.y = qny;
        if (MASK) vq = vqn;
    }
}

// The same walk with the packet held in shared memory instead of travelling by shuffles (one 1 KB buffer per
// warp): lane l owns slot l (position of j = 32 c + l and the force that j collects); in step s every lane works
// on slot (l + s) mod 32 — one conflict-free LDS.128 for the position, and the slot's force sum is read, extended
// by the lane's R pair terms and written back (LDS.128 / STS.128); __syncwarp() orders a step's write-back before
// the neighbour lane's read of the same slot in the next step.  Measured on B200 with lrmd_fp64_peak
// (bench.py --fp64-peak, profiles/r02_fp64_peak.md): next to DFMA traffic an LDS / STS / integer instruction costs no FP64 issue
// cycle, a SHFL costs about one (the shuffle walk spends 8 per step), and the position of the next step no longer
// depends on a shuffle chain.
struct SymWarpSmem {
    double2 pos[32];
    double2 g[32];
};

// WITHV: the walk also collects the potential of the pairs it meets (rows a-E2 / a-E3 fused into the force kernel, one
// extra DMUL (2D) or four extra instructions (Ring) per pair): 2D  vp *= r^2 + eps with the exponent moved to the integer
// counter ve once per step (needs 2^-127 <= r^2 + eps <= 2^127; sum log = log prod as in pair_energy_kernel);
// Ring  vp += d^(-1/2).  A DIAG walk meets every pair of the block twice and j = i once: the caller halves and corrects.
template <int MODEL, int R, bool MASK, bool DIAG, bool WITHV = false>
__device__ __forceinline__ void sym_chunk_smem(const double (&a)[R], const double (&b)[R], const bool (&vi)[R],
                                               double (&f0)[R], double (&f1)[R], const double2* __restrict__ spos,
                                               double2* __restrict__ sg, int nvalid, double eps, double onepe,
                                               double* vp_ = nullptr, int* ve_ = nullptr) {
    double vp = WITHV ? *vp_ : 0.0;
    int ve = WITHV ? *ve_ : 0;
    // spos / sg: the 32 slots of the packet in shared memory (positions; force sums, read and written when !DIAG)
    const int lane = threadIdx.x & 31;
    double2 qn = spos[lane];
#pragma unroll 8
    for (int s = 0; s < 32; ++s) {
        const int idx = (lane + s) & 31;
        const double2 q = qn;
        qn = spos[(idx + 1) & 31];                   // next step's position, loaded a step ahead
        double h0 = 0.0, h1 = 0.0;
        if (!DIAG) {                                 // the slot's force sum so far
            const double2 g = sg[idx];
            h0 = g.x;
            h1 = g.y;
        }
        const bool vq = MASK ? (idx < nvalid) : true;
#pragma unroll
        for (int r0 = 0; r0 < R; r0 += 4) {
            if (MODEL == 2) {
                double dx[4], dy[4], r2[4], y0[4], y[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    dx[k] = a[r0 + k] - q.x;
                    dy[k] = b[r0 + k] - q.y;
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) r2[k] = fma(dy[k], dy[k], fma(dx[k], dx[k], eps));
#pragma unroll
                for (int k = 0; k < 4; ++k) y0[k] = rcp_seed(r2[k]);
                if (WITHV) {
#pragma unroll
                    for (int k = 0; k < 4; ++k) vp *= MASK ? ((vi[r0 + k] && vq) ? r2[k] : 1.0) : r2[k];
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const double e = fma(-r2[k], y0[k], 1.0);
                    y[k] = fma(e, e, e);
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    y[k] = fma(y0[k], y[k], y0[k]);
                    if (MASK) y[k] = (vi[r0 + k] && vq) ? y[k] : 0.0;
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    f0[r0 + k] = fma(dx[k], y[k], f0[r0 + k]);
                    if (!DIAG) h0 = fma(-dx[k], y[k], h0);
                    f1[r0 + k] = fma(dy[k], y[k], f1[r0 + k]);
                    if (!DIAG) h1 = fma(-dy[k], y[k], h1);
                }
            } else {
                double num[4], d[4], y0[4], c[4], p[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    num[k] = fma(b[r0 + k], q.x, -(a[r0 + k] * q.y));                 // s_i c_j - c_i s_j
                    d[k] = fma(-b[r0 + k], q.y, fma(-a[r0 + k], q.x, onepe));      // 1 + eps - c_i c_j - s_i s_j
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) y0[k] = rsqrt_seed(d[k]);
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const double bb = y0[k] * y0[k];
                    const double e = fma(-d[k], bb, 1.0);
                    c[k] = (num[k] * y0[k]) * bb;
                    p[k] = fma(fma(1.875, e, 1.5), e, 1.0);
                    if (MASK) c[k] = (vi[r0 + k] && vq) ? c[k] : 0.0;
                    if (WITHV) {     // d^(-1/2) = y0 (1 + e/2 + 3 e^2/8), the arithmetic of rsqrt_refined
                        const double rs = fma(y0[k] * e, fma(0.375, e, 0.5), y0[k]);
                        vp += MASK ? ((vi[r0 + k] && vq) ? rs : 0.0) : rs;
                    }
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    f0[r0 + k] = fma(c[k], p[k], f0[r0 + k]);
                    if (!DIAG) h0 = fma(-c[k], p[k], h0);
                }
            }
        }
        if (WITHV && MODEL == 2) {      // move the product's exponent into the integer counter
            const int hi = __double2hiint(vp);
            ve += ((hi >> 20) & 0x7ff) - 1023;
            vp = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(vp));
        }
        if (!DIAG) {
            sg[idx] = make_double2(h0, h1);
            __syncwarp();
        }
    }
    if (WITHV) {
        *vp_ = vp;
        *ve_ = ve;
    }
}

// (launch bound of 2 CTAs per SM: with the full register budget ptxas interleaves the pair chains of a step —
//  184-255 registers instead of 140 — which is worth 5-6 % although only 8 warps per SM stay resident)
// XCH: 0 = the packet travels by shuffles, 1 = it lives in shared memory (sym_chunk_smem); MINB = resident CTAs per SM
// the register budget is set for.
template <int MODEL, int R, int XCH, int MINB>
__global__ void __launch_bounds__(kSymThreads, MINB)
pair_force_sym_kernel(const double2* __restrict__ js, SymPart S, double eps, double pre, double* __restrict__ ipart0,
                      double* __restrict__ ipart1, double* __restrict__ jpart0, double* __restrict__ jpart1) {
    __shared__ SymWarpSmem swarp[XCH ? kSymThreads / 32 : 1];
    SymWarpSmem& sw = swarp[XCH ? (threadIdx.x >> 5) : 0];
    const int w = blockIdx.x * (kSymThreads / 32) + (threadIdx.x >> 5);
    if (w >= S.G) return;
    const int lane = threadIdx.x & 31;
    const long long N = S.N;
    const double onepe = 1.0 + eps;
    const int4 st = S.wstart[S.w0 + w];
    int tile = st.x, chunk = st.y;
    const bool ragged = (N % S.T) != 0 || (N % 32) != 0;

    double a[R], b[R], f0[R], f1[R];
    bool vi[R];
    unsigned selfmask = 0u;   // rows whose own chunk this worker walked since load_tile (Ring: self term to remove)
    auto load_tile = [&](int t) {
        selfmask = 0u;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long i = (long long)t * S.T + r * 32 + lane;
            vi[r] = i < N;
            const double2 q = vi[r] ? js[i] : make_double2(0.0, 0.0);
            a[r] = q.x;
            b[r] = q.y;
            f0[r] = 0.0;
            f1[r] = 0.0;
        }
    };
    auto store_tile = [&](int t) {
        const int slot = S.w0 + w - S.tile_rng[t].x;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long i = (long long)t * S.T + r * 32 + lane;
            if (MODEL == 1 && ((selfmask >> r) & 1u)) {
                // remove the rounding-level j = i term of eq.(9) again (the rounded product: N = 1 gives exactly 0)
                double c, p;
                ring_pair_parts(a[r], b[r], make_double2(a[r], b[r]), onepe, c, p);
                f0[r] -= __dmul_rn(c, p);
            }
            if (vi[r]) {
                ipart0[(long long)slot * N + i] = pre * f0[r];
                if (MODEL == 2) ipart1[(long long)slot * N + i] = pre * f1[r];
            }
        }
    };
    load_tile(tile);
    long long jn = (long long)chunk * 32 + lane;
    double2 qn = (jn < N) ? js[jn] : make_double2(0.0, 0.0);
    for (int u = 0; u < st.z; ++u) {
        const int ctile = tile, cchunk = chunk;
        const long long j = jn;
        const double2 q = qn;
        const bool vq = j < N;
        // the next unit, and its packet loaded before this unit's arithmetic
        ++chunk;
        const bool tile_done = chunk == S.nchunks;
        if (tile_done) { ++tile; chunk = tile * R; }
        const bool more = u + 1 < st.z;
        if (more) {
            jn = (long long)chunk * 32 + lane;
            qn = (jn < N) ? js[jn] : make_double2(0.0, 0.0);
        }
        double g0 = 0.0, g1 = 0.0;
        const bool diag = cchunk < (ctile + 1) * R;
        const bool masked = ragged && (ctile == S.ntiles - 1 || cchunk == S.nchunks - 1);
        if (XCH) {
            const long long left = N - (long long)cchunk * 32;
            const int nvalid = left < 32 ? (int)left : 32;
            sw.pos[lane] = q;
            sw.g[lane] = make_double2(0.0, 0.0);
            __syncwarp();
            if (diag) {
                if (masked) sym_chunk_smem<MODEL, R, true, true>(a, b, vi, f0, f1, sw.pos, sw.g, nvalid, eps, onepe);
                else sym_chunk_smem<MODEL, R, false, true>(a, b, vi, f0, f1, sw.pos, sw.g, nvalid, eps, onepe);
            } else {
                if (masked) sym_chunk_smem<MODEL, R, true, false>(a, b, vi, f0, f1, sw.pos, sw.g, nvalid, eps, onepe);
                else sym_chunk_smem<MODEL, R, false, false>(a, b, vi, f0, f1, sw.pos, sw.g, nvalid, eps, onepe);
            }
            __syncwarp();
            const double2 g = sw.g[lane];
            g0 = g.x;
            g1 = g.y;
            __syncwarp();      // every lane has read its slot before the next unit overwrites the buffer
        }
        if (diag) {
            if (!XCH) {
                if (masked) sym_chunk<MODEL, R, true, true>(a, b, vi, f0, f1, q, vq, eps, onepe, g0, g1);
                else sym_chunk<MODEL, R, false, true>(a, b, vi, f0, f1, q, vq, eps, onepe, g0, g1);
            }
            selfmask |= 1u << (cchunk - ctile * R);   // this walk met j = i for that row of every lane (step 0)
        } else {
            if (!XCH) {
                if (masked) sym_chunk<MODEL, R, true, false>(a, b, vi, f0, f1, q, vq, eps, onepe, g0, g1);
                else sym_chunk<MODEL, R, false, false>(a, b, vi, f0, f1, q, vq, eps, onepe, g0, g1);
            }
            if (vq) {
                jpart0[(long long)(ctile - S.tile0) * N + j] = pre * g0;
                if (MODEL == 2) jpart1[(long long)(ctile - S.tile0) * N + j] = pre * g1;
            }
        }
        if (tile_done || !more) {
            store_tile(ctile);
            if (more) load_tile(tile);
        }
    }
}

// ---- potential-energy kernels (rows a-E2, a-E3) ---------------------------------------------------------
// Full N x N sweep with the same partition; the j = i term is masked out; CTA k writes
// vpart[k] = pre_half * sum over its ranges of sum_{i in tile} sum_{j in range, j != i} t_ij
// where pre_half already contains the 1/2 for double counting.
//   Ring  t_ij = d_ij^(-1/2),  V = -(1/(sqrt2 N)) sum_{i<j} t_ij             eq.(1)
//   2D    t_ij = log(r_ij^2 + eps), V = (1/N) sum_{i<j} t_ij                 eq.(3)
// 2D uses sum log d = log prod d: one DMUL per pair into a running product whose exponent is
// moved into an integer counter every 8 pairs (needs 2^-127 <= d <= 2^127), one log() per tile.
template <int MODEL, typename CFG>
__global__ void __launch_bounds__(CFG::THREADS, CFG::MINB)
pair_energy_kernel(const double2* __restrict__ js, PairPart P, double eps, double pre_half,
                   double* __restrict__ vpart) {
    constexpr int R = CFG::R, THREADS = CFG::THREADS, TJ = CFG::TJ;
    __shared__ PairSmem<double2, TJ> sm;
    __shared__ double scratch[THREADS / 32];
    JTilePipe<double2, TJ> pipe(sm);
    pipe.init();
    const long long N = P.Ni;
    const double onepe = 1.0 + eps;
    constexpr double kLn2 = 0x1.62e42fefa39efp-1;
    double vsum = 0.0;

    PairSegments segs(P, blockIdx.x);
    long long tile, jbeg, jend;
    int slot;
    while (segs.next(P, tile, jbeg, jend, slot)) {
        const long long ibase = tile * CFG::ITILE + threadIdx.x;
        double a[R], b[R], acc[R], prod[R];
        long long irow[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long i = ibase + (long long)r * THREADS;
            irow[r] = (i < N) ? P.i0 + i : -1;      // global index of the row, -1 for padding rows
            const double2 q = (i < N) ? js[P.i0 + i] : make_double2(0.0, 0.0);
            a[r] = q.x;
            b[r] = q.y;
            acc[r] = 0.0;
            prod[r] = 1.0;
        }
        pipe.run(js, jbeg, jend, [&](const double2* tl, int cnt, long long j0) {
            // only j-tiles that meet this i-tile's own rows can hold a j = i pair: they take the
            // masked sweep, all others the plain one (no compare / select per pair)
            const long long ilo = P.i0 + tile * CFG::ITILE;
            const bool diag = (j0 < ilo + CFG::ITILE) && (j0 + cnt > ilo);
            int jself[R];   // j - j0 of the row's own index (outside [0, cnt) if not in this tile)
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const long long dj = irow[r] - j0;
                jself[r] = (irow[r] >= 0 && dj >= 0 && dj < cnt) ? (int)dj : -1;
            }
            auto sweep = [&](auto masked) {
                constexpr bool MASK = decltype(masked)::value;
                if (MODEL == 1) {
#pragma unroll 4
                    for (int jj = 0; jj < cnt; ++jj) {
                        const double2 q = tl[jj];
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const double d = fma(-b[r], q.y, fma(-a[r], q.x, onepe));
                            const double y = rsqrt_refined(d);
                            acc[r] += (MASK && jself[r] == jj) ? 0.0 : y;
                        }
                    }
                } else {
                    int esum[R];
#pragma unroll
                    for (int r = 0; r < R; ++r) esum[r] = 0;
                    for (int jb = 0; jb < cnt; jb += 8) {
                        const int m = (cnt - jb < 8) ? (cnt - jb) : 8;
                        auto one = [&](int jj) {
                            const double2 q = tl[jj];
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                const double dx = a[r] - q.x, dy = b[r] - q.y;
                                double d = fma(dy, dy, fma(dx, dx, eps));
                                if (MASK) d = (jself[r] == jj) ? 1.0 : d;
                                prod[r] *= d;
                            }
                        };
                        if (m == 8) {
#pragma unroll
                            for (int u = 0; u < 8; ++u) one(jb + u);
                        } else {
                            for (int u = 0; u < m; ++u) one(jb + u);
                        }
#pragma unroll
                        for (int r = 0; r < R; ++r) {   // move the exponent into the integer counter
                            const int hi = __double2hiint(prod[r]);
                            esum[r] += ((hi >> 20) & 0x7ff) - 1023;
                            prod[r] = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(prod[r]));
                        }
                    }
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        acc[r] += fma((double)esum[r], kLn2, log(prod[r]));
                        prod[r] = 1.0;
                    }
                }
            };
            if (diag) sweep(std::true_type{});
            else sweep(std::false_type{});
        });
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (irow[r] >= 0) vsum += acc[r];
    }

    double v[1] = {vsum};
    block_sum<THREADS, 1>(v, scratch);
    if (threadIdx.x == 0) vpart[blockIdx.x] = pre_half * v[0];
}

// ---- symmetric force kernel, fp32 pair terms (rows N1 + N4) ---------------------------------------------------------
// The same walk on the float2 position stream.  Halving the evaluations halves the MUFU.RCP count, the
// unit that bounds grav_force_f32_kernel.  Precision follows reading G16: a lane's i-side sums run in fp32 over the 32
// steps of one pass (32 terms) and are then added to its fp64 accumulators; the travelling j-side sum is fp64, fed
// once per step with the fp32 sum of that step's R terms.
template <int R, bool MASK, bool DIAG>
__device__ __forceinline__ void sym_chunk_f32(const float (&a)[R], const float (&b)[R], const bool (&vi)[R],
                                              double (&f0)[R], double (&f1)[R], float2 q, bool vq, float eps,
                                              double& g0, double& g1) {
    const unsigned lane = threadIdx.x & 31u, src = (lane + 31u) & 31u;
    float sx[R], sy[R];
#pragma unroll
    for (int r = 0; r < R; ++r) sx[r] = sy[r] = 0.f;
#pragma unroll 4
    for (int s = 0; s < 32; ++s) {
        const float qnx = __shfl_sync(0xffffffffu, q.x, src);
        const float qny = __shfl_sync(0xffffffffu, q.y, src);
        const bool vqn = MASK ? (__shfl_sync(0xffffffffu, (int)vq, src) != 0) : true;
        float h0 = 0.f, h1 = 0.f;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float dx = a[r] - q.x, dy = b[r] - q.y;
            const float r2 = fmaf(dy, dy, fmaf(dx, dx, eps));
            float w = rcp_f32(r2);
            if (MASK) w = (vi[r] && vq) ? w : 0.f;
            sx[r] = fmaf(dx, w, sx[r]);
            sy[r] = fmaf(dy, w, sy[r]);
            if (!DIAG) {
                h0 = fmaf(-dx, w, h0);
                h1 = fmaf(-dy, w, h1);
            }
        }
        if (!DIAG) {
            g0 = __shfl_sync(0xffffffffu, g0 + (double)h0, src);
            g1 = __shfl_sync(0xffffffffu, g1 + (double)h1, src);
        }
        q.x = qnx;
        q.y = qny;
        if (MASK) vq = vqn;
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        f0[r] += (double)sx[r];
        f1[r] += (double)sy[r];
    }
}

template <int R>
__global__ void __launch_bounds__(kSymThreads, 2)
grav_force_sym_f32_kernel(const float2* __restrict__ js32, SymPart S, float eps, double pre, double* __restrict__ ipart0,
                          double* __restrict__ ipart1, double* __restrict__ jpart0, double* __restrict__ jpart1) {
    const int w = blockIdx.x * (kSymThreads / 32) + (threadIdx.x >> 5);
    if (w >= S.G) return;
    const int lane = threadIdx.x & 31;
    const long long N = S.N;
    const int4 st = S.wstart[S.w0 + w];
    int tile = st.x, chunk = st.y;
    const bool ragged = (N % S.T) != 0 || (N % 32) != 0;

    float a[R], b[R];
    double f0[R], f1[R];
    bool vi[R];
    auto load_tile = [&](int t) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long i = (long long)t * S.T + r * 32 + lane;
            vi[r] = i < N;
            const float2 q = vi[r] ? js32[i] : make_float2(0.f, 0.f);
            a[r] = q.x;
            b[r] = q.y;
            f0[r] = 0.0;
            f1[r] = 0.0;
        }
    };
    auto store_tile = [&](int t) {
        const int slot = S.w0 + w - S.tile_rng[t].x;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long i = (long long)t * S.T + r * 32 + lane;
            if (vi[r]) {
                ipart0[(long long)slot * N + i] = pre * f0[r];
                ipart1[(long long)slot * N + i] = pre * f1[r];
            }
        }
    };
    load_tile(tile);
    long long jn = (long long)chunk * 32 + lane;
    float2 qn = (jn < N) ? js32[jn] : make_float2(0.f, 0.f);
    for (int u = 0; u < st.z; ++u) {
        const int ctile = tile, cchunk = chunk;
        const long long j = jn;
        const float2 q = qn;
        const bool vq = j < N;
        ++chunk;
        const bool tile_done = chunk == S.nchunks;
        if (tile_done) { ++tile; chunk = tile * R; }
        const bool more = u + 1 < st.z;
        if (more) {
            jn = (long long)chunk * 32 + lane;
            qn = (jn < N) ? js32[jn] : make_float2(0.f, 0.f);
        }
        double g0 = 0.0, g1 = 0.0;
        const bool diag = cchunk < (ctile + 1) * R;
        const bool masked = ragged && (ctile == S.ntiles - 1 || cchunk == S.nchunks - 1);
        if (diag) {
            if (masked) sym_chunk_f32<R, true, true>(a, b, vi, f0, f1, q, vq, eps, g0, g1);
            else sym_chunk_f32<R, false, true>(a, b, vi, f0, f1, q, vq, eps, g0, g1);
        } else {
            if (masked) sym_chunk_f32<R, true, false>(a, b, vi, f0, f1, q, vq, eps, g0, g1);
            else sym_chunk_f32<R, false, false>(a, b, vi, f0, f1, q, vq, eps, g0, g1);
            if (vq) {
                jpart0[(long long)(ctile - S.tile0) * N + j] = pre * g0;
                jpart1[(long long)(ctile - S.tile0) * N + j] = pre * g1;
            }
        }
        if (tile_done || !more) {
            store_tile(ctile);
            if (more) load_tile(tile);
        }
    }
}

// ---- symmetric potential-energy kernel -------------------------------------------------------------------------
// V is a sum over unordered pairs to begin with (eqs.(1),(3): sum_{i<j}), so the walk of the symmetric force kernel
// gives it with every pair evaluated once and nothing to send back: only the packet's position travels.  The chunks
// of a tile itself count a pair only if j > i (masked walk, a small fraction of the units).  Worker w writes
// vpart[w0 + w] = pre * (its sum over its units), lanes combined by the fixed shuffle tree; energy_finalize_kernel
// adds the workers in index order.
template <int MODEL, int R, bool MASK>
__device__ __forceinline__ void sym_energy_chunk(const double (&a)[R], const double (&b)[R], const long long (&irow)[R],
                                                 const double2* __restrict__ spos, long long jbase, long long N, bool diag,
                                                 double eps, double onepe, double (&acc)[R], double (&prod)[R],
                                                 int (&esum)[R]) {
    // spos: the chunk's 32 positions in shared memory (the packet no longer travels by shuffles: a SHFL costs an FP64
    // issue slot, an LDS none, profiles/r02_fp64_peak.md); lane l meets slot (l + s) mod 32 in step s.
    const int lane = threadIdx.x & 31;
    double2 qn = spos[lane];
#pragma unroll 4
    for (int s = 0; s < 32; ++s) {
        const int idx = (lane + s) & 31;
        const double2 q = qn;
        qn = spos[(idx + 1) & 31];
        const long long jq = MASK ? ((jbase + idx < N) ? jbase + idx : -1) : 0;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            // counted: both particles exist, and inside the tile's own chunks only j > i
            const bool on = !MASK || (irow[r] >= 0 && jq >= 0 && (!diag || jq > irow[r]));
            if (MODEL == 1) {
                const double d = fma(-b[r], q.y, fma(-a[r], q.x, onepe));
                const double y = rsqrt_refined(d);
                acc[r] += on ? y : 0.0;
            } else {
                const double dx = a[r] - q.x, dy = b[r] - q.y;
                const double d = fma(dy, dy, fma(dx, dx, eps));
                prod[r] *= on ? d : 1.0;
            }
        }
        if (MODEL == 2 && (s & 7) == 7) {
#pragma unroll
            for (int r = 0; r < R; ++r) {   // move the exponent into the integer counter (2^-127 <= d <= 2^127)
                const int hi = __double2hiint(prod[r]);
                esum[r] += ((hi >> 20) & 0x7ff) - 1023;
                prod[r] = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(prod[r]));
            }
        }
    }
}

template <int MODEL, int R>
__global__ void __launch_bounds__(kSymThreads, 2)
pair_energy_sym_kernel(const double2* __restrict__ js, SymPart S, double eps, double pre, double* __restrict__ vpart) {
    __shared__ double2 wpos_all[kSymThreads / 32][32];
    double2* wpos = wpos_all[threadIdx.x >> 5];
    const int w = blockIdx.x * (kSymThreads / 32) + (threadIdx.x >> 5);
    if (w >= S.G) return;
    const int lane = threadIdx.x & 31;
    const long long N = S.N;
    const double onepe = 1.0 + eps;
    constexpr double kLn2 = 0x1.62e42fefa39efp-1;
    const int4 st = S.wstart[S.w0 + w];
    int tile = st.x, chunk = st.y;
    const bool ragged = (N % S.T) != 0 || (N % 32) != 0;

    double a[R], b[R], acc[R], prod[R];
    int esum[R];
    long long irow[R];
    double vsum = 0.0;
    auto load_tile = [&](int t) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long i = (long long)t * S.T + r * 32 + lane;
            irow[r] = i < N ? i : -1;
            const double2 q = i < N ? js[i] : make_double2(0.0, 0.0);
            a[r] = q.x;
            b[r] = q.y;
            acc[r] = 0.0;
            prod[r] = 1.0;
            esum[r] = 0;
        }
    };
    auto close_tile = [&]() {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (MODEL == 2) acc[r] = fma((double)esum[r], kLn2, log(prod[r]));
            vsum += acc[r];     // rows that do not exist never counted a pair: acc = 0 (Ring), log 1 = 0 (2D)
        }
    };
    load_tile(tile);
    long long jn = (long long)chunk * 32 + lane;
    double2 qn = (jn < N) ? js[jn] : make_double2(0.0, 0.0);
    for (int u = 0; u < st.z; ++u) {
        const int ctile = tile, cchunk = chunk;
        const long long j = jn;
        const double2 q = qn;
        ++chunk;
        const bool tile_done = chunk == S.nchunks;
        if (tile_done) { ++tile; chunk = tile * R; }
        const bool more = u + 1 < st.z;
        if (more) {
            jn = (long long)chunk * 32 + lane;
            qn = (jn < N) ? js[jn] : make_double2(0.0, 0.0);
        }
        const bool diag = cchunk < (ctile + 1) * R;
        const bool masked = diag || (ragged && (ctile == S.ntiles - 1 || cchunk == S.nchunks - 1));
        wpos[lane] = q;
        __syncwarp();
        if (masked) sym_energy_chunk<MODEL, R, true>(a, b, irow, wpos, (long long)cchunk * 32, N, diag, eps, onepe, acc, prod, esum);
        else sym_energy_chunk<MODEL, R, false>(a, b, irow, wpos, 0, N, false, eps, onepe, acc, prod, esum);
        __syncwarp();      // every lane has read the buffer before the next unit overwrites it
        if (tile_done || !more) {
            close_tile();
            if (more) load_tile(tile);
        }
    }
    vsum = warp_sum(vsum);
    if (lane == 0) vpart[S.w0 + w] = pre * vsum;
}

// ---- update kernels (row a-U1) --------------------------------------------------------------------------

constexpr int kUpdThreads = 256;

// js[i] = (cos th_i, sin th_i) (Ring; "computed and stored in global memory") or (x_i, y_i) (2D)
template <int MODEL>
__global__ void __launch_bounds__(kUpdThreads)
pair_pack_kernel(const double* __restrict__ q0, const double* __restrict__ q1, long long N, long long i0,
                 double2* __restrict__ js, float2* __restrict__ js32) {
    const long long i = (long long)blockIdx.x * kUpdThreads + threadIdx.x;
    if (i >= N) return;
    if (MODEL == 1) {
        double s, c;
        sincos_any(q0[i], s, c);
        js[i0 + i] = make_double2(c, s);
        if (js32) {     // fp32 pair arithmetic: (cos, sin)(theta / 2), see ring_force_f32_kernel
            sincos_any(0.5 * q0[i], s, c);
            js32[i0 + i] = make_float2((float)c, (float)s);
        }
    } else {
        js[i0 + i] = make_double2(q0[i], q1[i]);
        if (js32) js32[i0 + i] = make_float2((float)q0[i], (float)q1[i]);
    }
}

// Folds one launch (batch of tiles tile0 .. tile1 - 1) of the symmetric kernel into the force row out0 / out1:
// for particle i (from the batch's first particle on) the i-side rows of the workers that touched i's tile, if the
// tile is in the batch, + the j-side rows of the batch's tiles below i's tile.  The first batch writes, later ones
// add (batches run in tile order on one stream).  Block = 32 particles x 16 row groups: group k adds the rows
// k, k + 16, ... of each list in order, the group sums are combined in a fixed pairwise tree: deterministic, and
// sixteen times shorter than one dependent chain of ~100 loads per particle.
constexpr int kFoldGroups = 16;   // row groups per particle in pair_sym_fold_kernel (block = 32 x kFoldGroups threads)

// The update that follows a force evaluation (pair_update_kernel's arithmetic), fused into the fold of a
// single-launch evaluation: UPD = 0 none, 1 kick, 2 kick + drift, 3 two kicks + drift.
struct FusedUpdate {
    double *q0, *q1, *p0, *p1;
    double kickA, kickB, drift;
    double2* js;
    float2* js32;
};

// Tail of the fold kernels, run by the thread of group 0: combines the kFoldGroups partial sums of particle i in a
// fixed pairwise tree, writes (or adds to) the force row and applies the update UPD.
template <int MODEL, int UPD>
__device__ __forceinline__ void fold_finish(const double (&sf)[kFoldGroups][32], const double (&sg)[kFoldGroups][32],
                                            long long i, bool write, double* __restrict__ out0, double* __restrict__ out1,
                                            const FusedUpdate& U) {
    constexpr int GR = kFoldGroups;
    const int x = threadIdx.x;
    double ff[GR], gg[GR];
#pragma unroll
    for (int m = 0; m < GR; ++m) { ff[m] = sf[m][x]; gg[m] = sg[m][x]; }
#pragma unroll
    for (int w = 1; w < GR; w *= 2) {      // fixed pairwise tree: (0+1), (2+3), ... then (01+23), ...
#pragma unroll
        for (int m = 0; m < GR; m += 2 * w) { ff[m] += ff[m + w]; gg[m] += gg[m + w]; }
    }
    if (write) {
        out0[i] = ff[0];
        if (out1) out1[i] = gg[0];
    } else {
        out0[i] += ff[0];
        if (out1) out1[i] += gg[0];
    }
    if (UPD != 0) {     // only on single-launch evaluations: ff, gg are the whole force
        double p = fma(U.kickA, ff[0], U.p0[i]);
        if (UPD == 3) p = fma(U.kickB, ff[0], p);
        U.p0[i] = p;
        double pb = 0.0;
        if (MODEL == 2) {
            pb = fma(U.kickA, gg[0], U.p1[i]);
            if (UPD == 3) pb = fma(U.kickB, gg[0], pb);
            U.p1[i] = pb;
        }
        if (UPD >= 2) {
            const double xq = fma(U.drift, p, U.q0[i]);
            U.q0[i] = xq;
            if (MODEL == 2) {
                const double yq = fma(U.drift, pb, U.q1[i]);
                U.q1[i] = yq;
                U.js[i] = make_double2(xq, yq);
                if (U.js32) U.js32[i] = make_float2((float)xq, (float)yq);
            } else {
                double sn, cs;
                sincos_any(xq, sn, cs);
                U.js[i] = make_double2(cs, sn);
            }
        }
    }
}

template <int MODEL, int UPD>
__global__ void __launch_bounds__(32 * kFoldGroups)
pair_sym_fold_kernel(SymPart S, const double* __restrict__ ipart0, const double* __restrict__ ipart1,
                     const double* __restrict__ jpart0, const double* __restrict__ jpart1, double* __restrict__ out0,
                     double* __restrict__ out1, FusedUpdate U) {
    constexpr int GR = kFoldGroups;
    __shared__ double sf[GR][32], sg[GR][32];
    const long long N = S.N;
    const long long i = (long long)S.tile0 * S.T + (long long)blockIdx.x * 32 + threadIdx.x;
    const int k = threadIdx.y;
    double f = 0.0, g = 0.0;
    if (i < N) {
        const int t = (int)(i / S.T);
        if (t < S.tile1) {
            const int2 rng = S.tile_rng[t];
            for (int s = k; s <= rng.y - rng.x; s += GR) {
                f += ipart0[(long long)s * N + i];
                if (ipart1) g += ipart1[(long long)s * N + i];
            }
        }
        const int nrows = (t < S.tile1 ? t : S.tile1) - S.tile0;     // batch tiles below i's tile
        for (int a = k; a < nrows; a += GR) {
            f += jpart0[(long long)a * N + i];
            if (jpart1) g += jpart1[(long long)a * N + i];
        }
    }
    sf[k][threadIdx.x] = f;
    sg[k][threadIdx.x] = g;
    __syncthreads();
    if (k == 0 && i < N) fold_finish<MODEL, UPD>(sf, sg, i, S.tile0 == 0, out0, out1, U);
}

// The partial rows of a force evaluation: [slots][N] from the ordered kernels, or the single folded row of the
// symmetric kernel (single_row = 1).
struct ForceRows {
    const double* partial0;
    const double* partial1;
    int single_row;
};

// Number of partial rows of particle i's tile (the CTAs first..last of the partition touch it).
__device__ __forceinline__ int tile_slots(const PairPart& P, long long i) {
    long long first, last;
    part_tile_ctas(P, i / P.itile, first, last);
    return (int)(last - first + 1);
}

// f = sum_s partial[s][i] (slot order); p += kickA f [; p += kickB f]; if DRIFT: q += drift p and
// the packed j-stream is refreshed (listing steps 2-3, 5-6, 8-9, 11; "update kernel").
template <int MODEL, bool KICK2, bool DRIFT>
__global__ void __launch_bounds__(kUpdThreads)
pair_update_kernel(double* __restrict__ q0, double* __restrict__ q1, double* __restrict__ p0, double* __restrict__ p1,
                   PairPart P, ForceRows FR, double kickA, double kickB, double drift, double2* __restrict__ js,
                   float2* __restrict__ js32) {
    const long long N = P.Ni;
    const long long i = (long long)blockIdx.x * kUpdThreads + threadIdx.x;
    if (i >= N) return;
    double f, g = 0.0;
    {
        const int S = FR.single_row ? 1 : tile_slots(P, i);
        f = FR.partial0[i];
        for (int s = 1; s < S; ++s) f += FR.partial0[(long long)s * N + i];
        if (MODEL == 2) {
            g = FR.partial1[i];
            for (int s = 1; s < S; ++s) g += FR.partial1[(long long)s * N + i];
        }
    }
    double p = fma(kickA, f, p0[i]);
    if (KICK2) p = fma(kickB, f, p);
    p0[i] = p;
    double pb = 0.0;
    if (MODEL == 2) {
        pb = fma(kickA, g, p1[i]);
        if (KICK2) pb = fma(kickB, g, pb);
        p1[i] = pb;
    }
    if (DRIFT) {
        const double x = fma(drift, p, q0[i]);
        q0[i] = x;
        if (MODEL == 2) {
            const double y = fma(drift, pb, q1[i]);
            q1[i] = y;
            js[P.i0 + i] = make_double2(x, y);
            if (js32) js32[P.i0 + i] = make_float2((float)x, (float)y);
        } else {
            double sn, cs;
            sincos_any(x, sn, cs);
            js[P.i0 + i] = make_double2(cs, sn);
            if (js32) {
                sincos_any(0.5 * x, sn, cs);
                js32[P.i0 + i] = make_float2((float)cs, (float)sn);
            }
        }
    }
}

// lrmd_forces for the pair models: f = sum_s partial[s][i]
__global__ void __launch_bounds__(kUpdThreads)
pair_force_out_kernel(PairPart P, ForceRows FR, double* __restrict__ f0, double* __restrict__ f1) {
    const long long N = P.Ni;
    const long long i = (long long)blockIdx.x * kUpdThreads + threadIdx.x;
    if (i >= N) return;
    double f, g = 0.0;
    {
        const int S = FR.single_row ? 1 : tile_slots(P, i);
        f = FR.partial0[i];
        for (int s = 1; s < S; ++s) f += FR.partial0[(long long)s * N + i];
        if (f1) {
            g = FR.partial1[i];
            for (int s = 1; s < S; ++s) g += FR.partial1[(long long)s * N + i];
        }
    }
    f0[i] = f;
    if (f1) f1[i] = g;
}

}  // namespace lrmd
