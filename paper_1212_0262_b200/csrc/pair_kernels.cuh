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
//   * a 2-D grid (i-tile, j-chunk): N/ITILE alone does not fill 148 SMs for N = 16,384, so the j
//     range is split into S chunks; each CTA writes a partial force row partial[s][i] and the
//     update kernel adds the S partials in index order (deterministic, no atomics);
//   * MUFU.RCP64H / MUFU.RSQ64H seed (~2^-20) + one cubic fp64 correction instead of rsqrt():
//     2D 9 FP64 instructions per pair (7 DFMA + 2 DADD), Ring 12 (7 DFMA + 5 DMUL).
// The j = i pair is computed like any other (PAPER.md:105 loops over all k): for eps > 0 it
// contributes exactly 0 in 2D (dx = dy = 0) and a rounding-level term in the Ring rewrite eq.(9)
// (s_i c_i - c_i s_i evaluated with one FMA), which the epilogue removes again.
#pragma once

#include "common.cuh"
#include "trig.cuh"

namespace lrmd {

constexpr int kPairThreads = 128;   // threads per CTA
constexpr int kPairR = 4;           // i-particles per thread
constexpr int kPairITile = kPairThreads * kPairR;
constexpr int kPairTJ = 256;        // j-elements per smem stage (4 KB)
constexpr int kPairCtasPerSm = 4;   // enforced by __launch_bounds__ (<= 128 registers)

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

// Ring eq.(9): returns (num * y, y^2) with y = d^(-1/2); term = num y^3
__device__ __forceinline__ void ring_pair_parts(double ci, double si, double2 q, double onepe, double& ny, double& y2) {
    const double num = fma(si, q.x, -(ci * q.y));          // s_i c_j - c_i s_j
    const double d = fma(-si, q.y, fma(-ci, q.x, onepe));  // 1 + eps - c_i c_j - s_i s_j
    const double y = rsqrt_refined(d);
    ny = num * y;
    y2 = y * y;
}

// ---- j-tile pipeline ----------------------------------------------------------------------------------

struct PairSmem {
    alignas(128) double2 tile[2][kPairTJ];
    alignas(8) uint64_t full[2];
};

// Calls body(tile_ptr, count, j0) for consecutive tiles of [jbeg, jend) of the packed j-stream.
template <typename Body>
__device__ __forceinline__ void for_each_jtile(PairSmem& sm, const double2* __restrict__ js, long long jbeg,
                                               long long jend, Body body) {
    const int ntiles = (int)((jend - jbeg + kPairTJ - 1) / kPairTJ);
    if (threadIdx.x == 0) {
        mbar_init(&sm.full[0], 1);
        mbar_init(&sm.full[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (threadIdx.x == 0 && ntiles > 0) {
        const long long c0 = (jend - jbeg < kPairTJ) ? (jend - jbeg) : kPairTJ;
        mbar_expect_tx(&sm.full[0], (uint32_t)(c0 * sizeof(double2)));
        bulk_g2s(sm.tile[0], js + jbeg, (uint32_t)(c0 * sizeof(double2)), &sm.full[0]);
    }
    uint32_t phase[2] = {0u, 0u};
    for (int t = 0; t < ntiles; ++t) {
        const int s = t & 1;
        const long long j0 = jbeg + (long long)t * kPairTJ;
        if (threadIdx.x == 0 && t + 1 < ntiles) {
            // stage s^1 was consumed in iteration t-1; every thread passed the barrier that ended it
            const long long j1 = j0 + kPairTJ;
            const long long c1 = (jend - j1 < kPairTJ) ? (jend - j1) : kPairTJ;
            mbar_expect_tx(&sm.full[s ^ 1], (uint32_t)(c1 * sizeof(double2)));
            bulk_g2s(sm.tile[s ^ 1], js + j1, (uint32_t)(c1 * sizeof(double2)), &sm.full[s ^ 1]);
        }
        mbar_wait(&sm.full[s], phase[s]);
        phase[s] ^= 1u;
        const int cnt = (int)((jend - j0 < kPairTJ) ? (jend - j0) : kPairTJ);
        body(sm.tile[s], cnt, j0);
        __syncthreads();
    }
}

__device__ __forceinline__ void jchunk_bounds(long long N, int S, int s, long long& jbeg, long long& jend) {
    jbeg = (N * (long long)s) / S;
    jend = (N * (long long)(s + 1)) / S;
}

// ---- force kernels (rows a-P1r, a-P1g) --------------------------------------------------------------

// grid = (ceil(N/ITILE), S).  partial0/1: [S][N] partial forces (with the model's prefactor).
template <int MODEL>
__global__ void __launch_bounds__(kPairThreads, kPairCtasPerSm)
pair_force_kernel(const double2* __restrict__ js, long long N, double eps, double pre,
                  double* __restrict__ partial0, double* __restrict__ partial1) {
    __shared__ PairSmem sm;
    const long long ibase = (long long)blockIdx.x * kPairITile + threadIdx.x;
    const int S = gridDim.y, s = blockIdx.y;
    long long jbeg, jend;
    jchunk_bounds(N, S, s, jbeg, jend);

    double a[kPairR], b[kPairR], f0[kPairR], f1[kPairR];
#pragma unroll
    for (int r = 0; r < kPairR; ++r) {
        const long long i = ibase + (long long)r * kPairThreads;
        const double2 q = (i < N) ? js[i] : make_double2(0.0, 0.0);
        a[r] = q.x;
        b[r] = q.y;
        f0[r] = 0.0;
        f1[r] = 0.0;
    }
    const double onepe = 1.0 + eps;

    for_each_jtile(sm, js, jbeg, jend, [&](const double2* tile, int cnt, long long) {
#pragma unroll 4
        for (int jj = 0; jj < cnt; ++jj) {
            const double2 q = tile[jj];   // broadcast LDS.128
#pragma unroll
            for (int r = 0; r < kPairR; ++r) {
                if (MODEL == 2) {
                    grav_pair(a[r], b[r], q, eps, f0[r], f1[r]);
                } else {
                    double ny, y2;
                    ring_pair_parts(a[r], b[r], q, onepe, ny, y2);
                    f0[r] = fma(ny, y2, f0[r]);
                }
            }
        }
    });

#pragma unroll
    for (int r = 0; r < kPairR; ++r) {
        const long long i = ibase + (long long)r * kPairThreads;
        if (i < N) {
            if (MODEL == 1) {
                if (i >= jbeg && i < jend) {   // remove the rounding-level j = i term again
                    double ny, y2;
                    ring_pair_parts(a[r], b[r], make_double2(a[r], b[r]), onepe, ny, y2);
                    f0[r] -= __dmul_rn(ny, y2);   // the rounded product, so that N = 1 gives exactly 0
                }
                partial0[(long long)s * N + i] = pre * f0[r];
            } else {
                partial0[(long long)s * N + i] = pre * f0[r];
                partial1[(long long)s * N + i] = pre * f1[r];
            }
        }
    }
}

// ---- potential-energy kernels (rows a-E2, a-E3) ---------------------------------------------------------
// Full N x N sweep with the same tiling; the j = i term is masked out; the CTA writes
// vpart[blockIdx.y * gridDim.x + blockIdx.x] = pre_half * sum_{i in tile} sum_{j in chunk, j != i} t_ij
// where pre_half already contains the 1/2 for double counting.
//   Ring  t_ij = d_ij^(-1/2),  V = -(1/(sqrt2 N)) sum_{i<j} t_ij             eq.(1)
//   2D    t_ij = log(r_ij^2 + eps), V = (1/N) sum_{i<j} t_ij                 eq.(3)
// 2D uses sum log d = log prod d: one DMUL per pair into a running product whose exponent is
// moved into an integer counter every 8 pairs (needs 2^-127 <= d <= 2^127), one log() per tile.
template <int MODEL>
__global__ void __launch_bounds__(kPairThreads, kPairCtasPerSm)
pair_energy_kernel(const double2* __restrict__ js, long long N, double eps, double pre_half,
                   double* __restrict__ vpart) {
    __shared__ PairSmem sm;
    __shared__ double scratch[kPairThreads / 32];
    const long long ibase = (long long)blockIdx.x * kPairITile + threadIdx.x;
    const int S = gridDim.y, s = blockIdx.y;
    long long jbeg, jend;
    jchunk_bounds(N, S, s, jbeg, jend);

    double a[kPairR], b[kPairR], acc[kPairR], prod[kPairR];
    long long irow[kPairR];
#pragma unroll
    for (int r = 0; r < kPairR; ++r) {
        const long long i = ibase + (long long)r * kPairThreads;
        irow[r] = i;
        const double2 q = (i < N) ? js[i] : make_double2(0.0, 0.0);
        a[r] = q.x;
        b[r] = q.y;
        acc[r] = 0.0;
        prod[r] = 1.0;
    }
    const double onepe = 1.0 + eps;
    constexpr double kLn2 = 0x1.62e42fefa39efp-1;

    for_each_jtile(sm, js, jbeg, jend, [&](const double2* tile, int cnt, long long j0) {
        if (MODEL == 1) {
#pragma unroll 4
            for (int jj = 0; jj < cnt; ++jj) {
                const double2 q = tile[jj];
#pragma unroll
                for (int r = 0; r < kPairR; ++r) {
                    const double d = fma(-b[r], q.y, fma(-a[r], q.x, onepe));
                    const double y = rsqrt_refined(d);
                    acc[r] += (irow[r] == j0 + jj) ? 0.0 : y;
                }
            }
        } else {
            int esum[kPairR];
#pragma unroll
            for (int r = 0; r < kPairR; ++r) esum[r] = 0;
            for (int jb = 0; jb < cnt; jb += 8) {
                const int m = (cnt - jb < 8) ? (cnt - jb) : 8;
                if (m == 8) {
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const double2 q = tile[jb + u];
#pragma unroll
                        for (int r = 0; r < kPairR; ++r) {
                            const double dx = a[r] - q.x, dy = b[r] - q.y;
                            double d = fma(dy, dy, fma(dx, dx, eps));
                            d = (irow[r] == j0 + jb + u) ? 1.0 : d;
                            prod[r] *= d;
                        }
                    }
                } else {
                    for (int u = 0; u < m; ++u) {
                        const double2 q = tile[jb + u];
#pragma unroll
                        for (int r = 0; r < kPairR; ++r) {
                            const double dx = a[r] - q.x, dy = b[r] - q.y;
                            double d = fma(dy, dy, fma(dx, dx, eps));
                            d = (irow[r] == j0 + jb + u) ? 1.0 : d;
                            prod[r] *= d;
                        }
                    }
                }
#pragma unroll
                for (int r = 0; r < kPairR; ++r) {   // move the exponent into the integer counter
                    const int hi = __double2hiint(prod[r]);
                    esum[r] += ((hi >> 20) & 0x7ff) - 1023;
                    prod[r] = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(prod[r]));
                }
            }
#pragma unroll
            for (int r = 0; r < kPairR; ++r) {
                acc[r] += fma((double)esum[r], kLn2, log(prod[r]));
                prod[r] = 1.0;
            }
        }
    });

    double v[1] = {0.0};
#pragma unroll
    for (int r = 0; r < kPairR; ++r)
        if (irow[r] < N) v[0] += acc[r];
    block_sum<kPairThreads, 1>(v, scratch);
    if (threadIdx.x == 0) vpart[(long long)blockIdx.y * gridDim.x + blockIdx.x] = pre_half * v[0];
}

// ---- update kernels (row a-U1) --------------------------------------------------------------------------

constexpr int kUpdThreads = 256;

// js[i] = (cos th_i, sin th_i) (Ring; "computed and stored in global memory") or (x_i, y_i) (2D)
template <int MODEL>
__global__ void __launch_bounds__(kUpdThreads)
pair_pack_kernel(const double* __restrict__ q0, const double* __restrict__ q1, long long N, double2* __restrict__ js) {
    const long long i = (long long)blockIdx.x * kUpdThreads + threadIdx.x;
    if (i >= N) return;
    if (MODEL == 1) {
        double s, c;
        sincos_pi4(q0[i], s, c);
        js[i] = make_double2(c, s);
    } else {
        js[i] = make_double2(q0[i], q1[i]);
    }
}

// f = sum_s partial[s][i] (index order); p += kickA f [; p += kickB f]; if DRIFT: q += drift p and
// the packed j-stream is refreshed (listing steps 2-3, 5-6, 8-9, 11; "update kernel").
template <int MODEL, bool KICK2, bool DRIFT>
__global__ void __launch_bounds__(kUpdThreads)
pair_update_kernel(double* __restrict__ q0, double* __restrict__ q1, double* __restrict__ p0, double* __restrict__ p1,
                   long long N, const double* __restrict__ partial0, const double* __restrict__ partial1, int S,
                   double kickA, double kickB, double drift, double2* __restrict__ js) {
    const long long i = (long long)blockIdx.x * kUpdThreads + threadIdx.x;
    if (i >= N) return;
    double f = partial0[i];
    for (int s = 1; s < S; ++s) f += partial0[(long long)s * N + i];
    double p = fma(kickA, f, p0[i]);
    if (KICK2) p = fma(kickB, f, p);
    p0[i] = p;
    double pb = 0.0;
    if (MODEL == 2) {
        double g = partial1[i];
        for (int s = 1; s < S; ++s) g += partial1[(long long)s * N + i];
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
            js[i] = make_double2(x, y);
        } else {
            double sn, cs;
            sincos_pi4(x, sn, cs);
            js[i] = make_double2(cs, sn);
        }
    }
}

// lrmd_forces for the pair models: f = sum_s partial[s][i]
__global__ void __launch_bounds__(kUpdThreads)
pair_force_out_kernel(long long N, const double* __restrict__ partial0, const double* __restrict__ partial1, int S,
                      double* __restrict__ f0, double* __restrict__ f1) {
    const long long i = (long long)blockIdx.x * kUpdThreads + threadIdx.x;
    if (i >= N) return;
    double f = partial0[i];
    for (int s = 1; s < S; ++s) f += partial0[(long long)s * N + i];
    f0[i] = f;
    if (f1) {
        double g = partial1[i];
        for (int s = 1; s < S; ++s) g += partial1[(long long)s * N + i];
        f1[i] = g;
    }
}

}  // namespace lrmd
