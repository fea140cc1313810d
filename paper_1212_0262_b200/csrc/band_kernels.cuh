// band_kernels.cuh — Newton's-third-law force kernel for large N (PAPER.md:108 is the passage it
// overturns): the warp-systolic walk of pair_kernels.cuh (sym_chunk_smem) inside a two-level blocking that keeps BOTH
// sides' partial sums on chip, so that one launch serves any N and the scratch rows shrink from N^2 / 256 doubles per
// component (one j-side row per 256-particle tile) to about 25 N.
//
//   * A CTA of 8 warps holds an I-block of IB = 8 x 32 R particles in registers (R per lane, as before) and a J-block
//     of IB particles in shared memory: positions (TMA bulk copy) and the force sums they collect.  The 8 warps walk
//     the J-block's 32-particle chunks at staggered offsets; a chunk's force sums stay in shared memory from one warp's
//     visit to the next, so the j-side sum of the whole I-block is formed on chip.  CTA barriers every n / 8 chunk
//     walks keep the visits to a chunk in a fixed order: deterministic, no atomics.
//   * I-blocks are grouped into bands of hb consecutive blocks.  The work of band A — all columns from the band's first
//     row to N — is cut into contiguous column ranges ("pieces") of equal weight, one or two per CTA.  For every
//     J-block of its piece a CTA loops over the band's I-blocks: the J-block's sums meet hb x IB rows before they are
//     written to the band's j-side row jbuf[band][column] (written once per band and column); the i-side sums of an
//     I-block are added to the piece's private row ibuf[piece][row] (one read-modify-write per J-block, private to the
//     CTA, in J-block order).
//   * The J-block that holds the I-block's own rows is walked in DIAG mode by every warp (i-side only, each ordered
//     pair of the block once): all warps carry the same load; J-blocks below it are skipped (their pairs are met from
//     the other side).
//   * pair_band_fold_kernel adds, for particle i, the i-side rows of its band's pieces and the j-side rows of the bands
//     up to its own, in a fixed order, and applies the kick / drift that follows (as pair_sym_fold_kernel does).
#pragma once

#include "pair_kernels.cuh"

namespace lrmd {

constexpr int kBandWarps = 8;
constexpr int kBandThreads = 32 * kBandWarps;

struct BandPiece {
    int band;       // band the piece belongs to
    int c0, c1;     // its columns, in chunks of 32 particles: [c0, c1)
    int pad;
};
struct BandInfo {
    int blk0, nblk;     // I-blocks blk0 .. blk0 + nblk - 1
    int pf0, pf1;       // pieces pf0 .. pf1 - 1, in column order
    long long joff;     // offset (elements) of the band's j-side row: column col is at joff + col - 32 cstart
    int cstart;         // first column chunk of the band = blk0 * IB / 32
    int pad;
};
struct BandPart {
    long long N;
    long long istride;  // rows of a full band = hb * IB: stride between the pieces' i-side rows
    int IB;             // rows per I-block = columns per J-block = kBandWarps * 32 * R
    int nIB, nchunks, nbands, hb;
    int P;              // workers (CTAs)
    const int* wpiece;          // [P + 1] first piece of every worker
    const BandPiece* pieces;
    const BandInfo* bands;
};

// dynamic shared memory: positions and force sums of one J-block + one mbarrier
constexpr size_t band_smem_bytes(int R) { return (size_t)2 * kBandWarps * 32 * R * sizeof(double2) + 16; }

// WITHV: the launch also delivers the potential energy (rows a-E2 / a-E3 fused into the force kernel: "compute any
// properties of interest" every step, listing step 12): vband[CTA] = pre_v * (the CTA's pairs' terms,
// log(r^2 + eps) or d^(-1/2)); a block's own pairs are met twice and j = i once by the DIAG walk: halved, and the
// self terms (exactly log eps; for Ring the value the same arithmetic gives) removed again.
template <int MODEL, int R, bool WITHV>
__global__ void __launch_bounds__(kBandThreads, 2)
pair_force_band_kernel(const double2* __restrict__ js, BandPart B, double eps, double pre, double* __restrict__ ibuf0,
                       double* __restrict__ ibuf1, double* __restrict__ jbuf0, double* __restrict__ jbuf1, double pre_v,
                       double* __restrict__ vband) {
    extern __shared__ __align__(128) unsigned char band_smem[];
    constexpr int T = 32 * R;                 // rows per warp tile
    constexpr int IB = kBandWarps * T;        // rows per I-block, columns per J-block
    constexpr int JB = IB / 32;               // chunks per J-block
    double2* Jpos = reinterpret_cast<double2*>(band_smem);
    double2* Jg = Jpos + IB;
    uint64_t* bar = reinterpret_cast<uint64_t*>(Jg + IB);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long N = B.N;
    const double onepe = 1.0 + eps;
    const bool ragged = (N % T) != 0;
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    uint32_t phase = 0u;
    double vsym = 0.0, vdiag = 0.0;          // potential terms of this thread's pairs (WITHV)
    constexpr double kLn2 = 0x1.62e42fefa39efp-1;

    const int pfirst = B.wpiece[blockIdx.x], plast = B.wpiece[blockIdx.x + 1];
    for (int pc = pfirst; pc < plast; ++pc) {
        const BandPiece piece = B.pieces[pc];
        const BandInfo band = B.bands[piece.band];
        const int jbfirst = piece.c0 / JB;
        for (int jb = jbfirst; jb * JB < piece.c1; ++jb) {
            const int jc0 = piece.c0 > jb * JB ? piece.c0 : jb * JB;
            const int jc1 = piece.c1 < (jb + 1) * JB ? piece.c1 : (jb + 1) * JB;
            const int n = jc1 - jc0;                               // chunks of this J-block segment
            const long long col0 = (long long)jc0 * 32;
            const int ncol = (int)((N - col0 < (long long)n * 32) ? (N - col0) : (long long)n * 32);   // columns that exist
            __syncthreads();    // the previous segment's shared-memory reads are done
            if (threadIdx.x == 0) {
                // the previous segment's generic-proxy reads and zero-fill writes of Jpos, ordered before this thread by
                // the barrier, must also be ordered before the bulk copy's async-proxy writes to the same addresses
                fence_proxy_async_smem();
                mbar_expect_tx(bar, (uint32_t)ncol * (uint32_t)sizeof(double2));
                bulk_g2s(Jpos, js + col0, (uint32_t)ncol * (uint32_t)sizeof(double2), bar);
            }
            for (int x = threadIdx.x; x < n * 32; x += kBandThreads) {
                Jg[x] = make_double2(0.0, 0.0);
                if (x >= ncol) Jpos[x] = make_double2(0.0, 0.0);
            }
            mbar_wait(bar, phase);
            phase ^= 1u;
            __syncthreads();

            // virtual chunk count: with fewer than 8 chunks the warps take turns (one warp per chunk at a time)
            const int nv = n >= kBandWarps ? n : kBandWarps;
            const int off = (warp * nv) / kBandWarps;
            const int m = nv / kBandWarps;                          // barrier period: visits to a chunk are >= m walks apart
            const int blk_end = band.blk0 + band.nblk < jb + 1 ? band.blk0 + band.nblk : jb + 1;
            for (int b = band.blk0; b < blk_end; ++b) {
                const bool diag = b == jb;
                const int tile = b * kBandWarps + warp;
                const bool tile_any = (long long)tile * T < N;
                const bool masked_tile = ragged && (long long)(tile + 1) * T > N;
                double a[R], bb[R], f0[R], f1[R];
                bool vi[R];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const long long i = (long long)tile * T + r * 32 + lane;
                    vi[r] = i < N;
                    const double2 q = vi[r] ? js[i] : make_double2(0.0, 0.0);
                    a[r] = q.x;
                    bb[r] = q.y;
                    f0[r] = 0.0;
                    f1[r] = 0.0;
                }
                unsigned selfmask = 0u;
                double vp = MODEL == 2 ? 1.0 : 0.0;
                int ve = 0;
                for (int k = 0; k < nv; ++k) {
                    int x = k + off;
                    if (x >= nv) x -= nv;
                    if (tile_any && x < n) {
                        const int gc = jc0 + x;                       // global chunk index
                        const long long left = N - (long long)gc * 32;
                        const int nvalid = left < 32 ? (int)left : 32;
                        const bool masked = masked_tile || nvalid < 32;
                        const double2* sp = Jpos + x * 32;
                        double2* sg = Jg + x * 32;
                        if (diag) {
                            if (masked) sym_chunk_smem<MODEL, R, true, true, WITHV>(a, bb, vi, f0, f1, sp, sg, nvalid, eps, onepe, &vp, &ve);
                            else sym_chunk_smem<MODEL, R, false, true, WITHV>(a, bb, vi, f0, f1, sp, sg, nvalid, eps, onepe, &vp, &ve);
                            const int rr = gc - tile * R;             // the walk met j = i for row rr of every lane
                            if ((MODEL == 1 || WITHV) && rr >= 0 && rr < R) selfmask |= 1u << rr;
                        } else {
                            if (masked) sym_chunk_smem<MODEL, R, true, false, WITHV>(a, bb, vi, f0, f1, sp, sg, nvalid, eps, onepe, &vp, &ve);
                            else sym_chunk_smem<MODEL, R, false, false, WITHV>(a, bb, vi, f0, f1, sp, sg, nvalid, eps, onepe, &vp, &ve);
                        }
                    }
                    if (!diag && (k + 1) % m == 0 && k + 1 < nv) __syncthreads();
                }
                if (WITHV) {
                    double vt = MODEL == 2 ? fma((double)ve, kLn2, log(vp)) : vp;
                    if (diag) {
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            if (((selfmask >> r) & 1u) && vi[r]) {        // the j = i term this walk met
                                if (MODEL == 2) {
                                    vt -= log(eps);
                                } else {
                                    const double d = fma(-bb[r], bb[r], fma(-a[r], a[r], onepe));
                                    const double y0 = rsqrt_seed(d);
                                    const double e = fma(-d, y0 * y0, 1.0);
                                    vt -= fma(y0 * e, fma(0.375, e, 0.5), y0);
                                }
                            }
                        }
                        vdiag += vt;
                    } else {
                        vsym += vt;
                    }
                }
                // i-side sums of this (J-block, I-block) visit -> the piece's private row (first visit stores)
                const bool first = jb == (b > jbfirst ? b : jbfirst);
                const long long rbase = (long long)pc * B.istride - (long long)band.blk0 * IB;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const long long i = (long long)tile * T + r * 32 + lane;
                    if (MODEL == 1 && ((selfmask >> r) & 1u)) {
                        // remove the rounding-level j = i term of eq.(9) again (the rounded product: N = 1 gives exactly 0)
                        double c, p;
                        ring_pair_parts(a[r], bb[r], make_double2(a[r], bb[r]), onepe, c, p);
                        f0[r] -= __dmul_rn(c, p);
                    }
                    if (vi[r]) {
                        double v0 = pre * f0[r];
                        if (!first) v0 += ibuf0[rbase + i];
                        ibuf0[rbase + i] = v0;
                        if (MODEL == 2) {
                            double v1 = pre * f1[r];
                            if (!first) v1 += ibuf1[rbase + i];
                            ibuf1[rbase + i] = v1;
                        }
                    }
                }
                __syncthreads();    // this I-block's walks are done before the next one's (fixed order of the j-side sums)
            }
            // the J-block segment's force sums -> the band's j-side row
            const long long jbase = band.joff + col0 - (long long)band.cstart * 32;
            for (int x = threadIdx.x; x < ncol; x += kBandThreads) {
                const double2 g = Jg[x];
                jbuf0[jbase + x] = pre * g.x;
                if (MODEL == 2) jbuf1[jbase + x] = pre * g.y;
            }
        }
    }
    if (WITHV) {
        __syncthreads();                                  // the J-block buffers are free: reuse them as scratch
        double v[1] = {vsym + 0.5 * vdiag};
        block_sum<kBandThreads, 1>(v, reinterpret_cast<double*>(band_smem));
        if (threadIdx.x == 0) vband[blockIdx.x] = pre_v * v[0];
    }
}

// ---- band kernel, fp32 pair terms (rows N1 + N4, GRAV2D) ------------------------------------------------
// The same blocking on the float2 position stream: the J-block's positions are fp32 (8 bytes per column), the force sums
// it collects fp64.  A walk's arithmetic is sym_chunk_f32's (2 FADD + 6 FFMA + MUFU.RCP per unordered pair), with the
// packet in shared memory: per step the lane adds the fp32 sum of its R terms to the slot's fp64 sum (reading G16: fp32
// sums never run over more than R terms on the j side, 32 on the i side).  64 registers of state per thread instead of
// the warp-level kernel's 191: 16 resident warps per SM instead of 8.
template <int R, bool MASK, bool DIAG, bool JSHFL = false>
__device__ __forceinline__ void sym_chunk_f32_smem(const float (&a)[R], const float (&b)[R], const bool (&vi)[R],
                                                   double (&f0)[R], double (&f1)[R], const float2* __restrict__ spos,
                                                   double2* __restrict__ sg, int nvalid, float eps) {
    // JSHFL (LRMD_OPT_PAIR_SYM_EXCHANGE = 0): the j-side sum of the slot a lane faces is an fp32 packet that travels with
    // the slot from lane to lane (at step s lane l faces slot l + s, which lane l + 1 faced the step before) and is added
    // to the slot's fp64 sum ONCE per visit: 2 SHFL per step instead of LDS.128 + 2 F2F + 2 DADD + STS.128 + a warp
    // barrier — the two conversions share the 16-lane XU pipe with the R MUFU.RCP of the step.  The fp32 packet then runs
    // over 32 R terms (256 for R = 8) instead of R; the sums across visits stay fp64 (reading G16).
    const int lane = threadIdx.x & 31;
    float sx[R], sy[R];
#pragma unroll
    for (int r = 0; r < R; ++r) sx[r] = sy[r] = 0.f;
    float2 qn = spos[lane];
    float h0 = 0.f, h1 = 0.f;
#pragma unroll 4
    for (int s = 0; s < 32; ++s) {
        const int idx = (lane + s) & 31;
        const float2 q = qn;
        qn = spos[(idx + 1) & 31];
        double2 g = make_double2(0.0, 0.0);
        if (!DIAG && !JSHFL) g = sg[idx];
        const bool vq = MASK ? (idx < nvalid) : true;
        if (!JSHFL) { h0 = 0.f; h1 = 0.f; }
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
            if (JSHFL) {
                if (s < 31) {       // hand the packet to the lane that faces this slot next
                    h0 = __shfl_sync(0xffffffffu, h0, (lane + 1) & 31);
                    h1 = __shfl_sync(0xffffffffu, h1, (lane + 1) & 31);
                }
            } else {
                sg[idx] = make_double2(g.x + (double)h0, g.y + (double)h1);
                __syncwarp();
            }
        }
    }
    if (!DIAG && JSHFL) {
        const int idx = (lane + 31) & 31;       // the slot faced at the last step: its packet is complete
        const double2 g = sg[idx];
        sg[idx] = make_double2(g.x + (double)h0, g.y + (double)h1);
        __syncwarp();
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        f0[r] += (double)sx[r];
        f1[r] += (double)sy[r];
    }
}

constexpr size_t band_f32_smem_bytes(int R) { return (size_t)kBandWarps * 32 * R * (sizeof(float2) + sizeof(double2)) + 16; }

// (R = 16, launch shape 2: 255 registers, one CTA per SM; 3.5 % faster than R = 8 at N = 102,400, not the default.
//  Packed fp32x2 arithmetic (FADD2 / FFMA2) was tried for the walk and measured 5 % slower: the packed instructions
//  issue at half rate and the pair packing costs register moves.)
template <int R, bool JSHFL = false>
__global__ void __launch_bounds__(kBandThreads, (R <= 8 ? 2 : 1))
grav_force_band_f32_kernel(const float2* __restrict__ js32, BandPart B, float eps, double pre, double* __restrict__ ibuf0,
                           double* __restrict__ ibuf1, double* __restrict__ jbuf0, double* __restrict__ jbuf1) {
    extern __shared__ __align__(128) unsigned char band_smem[];
    constexpr int T = 32 * R, IB = kBandWarps * T, JB = IB / 32;
    double2* Jg = reinterpret_cast<double2*>(band_smem);
    float2* Jpos = reinterpret_cast<float2*>(Jg + IB);
    uint64_t* bar = reinterpret_cast<uint64_t*>(Jpos + IB);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long N = B.N;
    const bool ragged = (N % T) != 0;
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    uint32_t phase = 0u;

    const int pfirst = B.wpiece[blockIdx.x], plast = B.wpiece[blockIdx.x + 1];
    for (int pc = pfirst; pc < plast; ++pc) {
        const BandPiece piece = B.pieces[pc];
        const BandInfo band = B.bands[piece.band];
        const int jbfirst = piece.c0 / JB;
        for (int jb = jbfirst; jb * JB < piece.c1; ++jb) {
            const int jc0 = piece.c0 > jb * JB ? piece.c0 : jb * JB;
            const int jc1 = piece.c1 < (jb + 1) * JB ? piece.c1 : (jb + 1) * JB;
            const int n = jc1 - jc0;
            const long long col0 = (long long)jc0 * 32;
            const int ncol = (int)((N - col0 < (long long)n * 32) ? (N - col0) : (long long)n * 32);
            const int ncopy = (ncol + 1) & ~1;        // bulk copies move multiples of 16 bytes (the stream is padded by 2)
            __syncthreads();
            if (threadIdx.x == 0) {
                fence_proxy_async_smem();      // as in the fp64 kernel: generic accesses to Jpos before the async-proxy writes
                mbar_expect_tx(bar, (uint32_t)ncopy * (uint32_t)sizeof(float2));
                bulk_g2s(Jpos, js32 + col0, (uint32_t)ncopy * (uint32_t)sizeof(float2), bar);
            }
            for (int x = threadIdx.x; x < n * 32; x += kBandThreads) Jg[x] = make_double2(0.0, 0.0);
            mbar_wait(bar, phase);
            phase ^= 1u;
            for (int x = ncol + threadIdx.x; x < n * 32; x += kBandThreads) Jpos[x] = make_float2(0.f, 0.f);
            __syncthreads();

            const int nv = n >= kBandWarps ? n : kBandWarps;
            const int off = (warp * nv) / kBandWarps;
            const int m = nv / kBandWarps;
            const int blk_end = band.blk0 + band.nblk < jb + 1 ? band.blk0 + band.nblk : jb + 1;
            for (int b = band.blk0; b < blk_end; ++b) {
                const bool diag = b == jb;
                const int tile = b * kBandWarps + warp;
                const bool tile_any = (long long)tile * T < N;
                const bool masked_tile = ragged && (long long)(tile + 1) * T > N;
                float a[R], bb[R];
                double f0[R], f1[R];
                bool vi[R];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const long long i = (long long)tile * T + r * 32 + lane;
                    vi[r] = i < N;
                    const float2 q = vi[r] ? js32[i] : make_float2(0.f, 0.f);
                    a[r] = q.x;
                    bb[r] = q.y;
                    f0[r] = 0.0;
                    f1[r] = 0.0;
                }
                for (int k = 0; k < nv; ++k) {
                    int x = k + off;
                    if (x >= nv) x -= nv;
                    if (tile_any && x < n) {
                        const long long left = N - (long long)(jc0 + x) * 32;
                        const int nvalid = left < 32 ? (int)left : 32;
                        const bool masked = masked_tile || nvalid < 32;
                        const float2* sp = Jpos + x * 32;
                        double2* sg = Jg + x * 32;
                        if (diag) {
                            if (masked) sym_chunk_f32_smem<R, true, true, JSHFL>(a, bb, vi, f0, f1, sp, sg, nvalid, eps);
                            else sym_chunk_f32_smem<R, false, true, JSHFL>(a, bb, vi, f0, f1, sp, sg, nvalid, eps);
                        } else {
                            if (masked) sym_chunk_f32_smem<R, true, false, JSHFL>(a, bb, vi, f0, f1, sp, sg, nvalid, eps);
                            else sym_chunk_f32_smem<R, false, false, JSHFL>(a, bb, vi, f0, f1, sp, sg, nvalid, eps);
                        }
                    }
                    if (!diag && (k + 1) % m == 0 && k + 1 < nv) __syncthreads();
                }
                const bool first = jb == (b > jbfirst ? b : jbfirst);
                const long long rbase = (long long)pc * B.istride - (long long)band.blk0 * IB;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const long long i = (long long)tile * T + r * 32 + lane;
                    if (vi[r]) {
                        double v0 = pre * f0[r], v1 = pre * f1[r];
                        if (!first) { v0 += ibuf0[rbase + i]; v1 += ibuf1[rbase + i]; }
                        ibuf0[rbase + i] = v0;
                        ibuf1[rbase + i] = v1;
                    }
                }
                __syncthreads();
            }
            const long long jbase = band.joff + col0 - (long long)band.cstart * 32;
            for (int x = threadIdx.x; x < ncol; x += kBandThreads) {
                const double2 g = Jg[x];
                jbuf0[jbase + x] = pre * g.x;
                jbuf1[jbase + x] = pre * g.y;
            }
        }
    }
}

// out0 / out1[i] = the force on particle i from one launch of pair_force_band_kernel; then the update (UPD as in
// pair_sym_fold_kernel).  Block = 32 particles x kFoldGroups term groups; terms of particle i, in this order:
// the i-side rows of its band's pieces that reached its I-block, then the j-side rows of bands 0 .. its own.
template <int MODEL, int UPD>
__global__ void __launch_bounds__(32 * kFoldGroups)
pair_band_fold_kernel(BandPart B, const double* __restrict__ ibuf0, const double* __restrict__ ibuf1,
                      const double* __restrict__ jbuf0, const double* __restrict__ jbuf1, double* __restrict__ out0,
                      double* __restrict__ out1, FusedUpdate U) {
    constexpr int GR = kFoldGroups;
    __shared__ double sf[GR][32], sg[GR][32];
    const long long N = B.N;
    const long long i = (long long)blockIdx.x * 32 + threadIdx.x;
    const int k = threadIdx.y;
    double f = 0.0, g = 0.0;
    if (i < N) {
        const int b = (int)(i / B.IB);
        const int A = b / B.hb;
        const BandInfo band = B.bands[A];
        const int ni = band.pf1 - band.pf0;
        const int nt = ni + A + 1;
        for (int t = k; t < nt; t += GR) {
            if (t < ni) {
                const int pc = band.pf0 + t;
                if ((long long)B.pieces[pc].c1 * 32 > (long long)b * B.IB) {       // the piece has columns at or beyond block b
                    const long long idx = (long long)pc * B.istride + i - (long long)band.blk0 * B.IB;
                    f += ibuf0[idx];
                    if (MODEL == 2) g += ibuf1[idx];
                }
            } else {
                const BandInfo bj = B.bands[t - ni];
                const long long idx = bj.joff + i - (long long)bj.cstart * 32;
                f += jbuf0[idx];
                if (MODEL == 2) g += jbuf1[idx];
            }
        }
    }
    sf[k][threadIdx.x] = f;
    sg[k][threadIdx.x] = g;
    __syncthreads();
    if (k == 0 && i < N) fold_finish<MODEL, UPD>(sf, sg, i, true, out0, out1, U);
}

}  // namespace lrmd
