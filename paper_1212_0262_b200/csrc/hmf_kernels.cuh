// hmf_kernels.cuh — HMF model (section 3.1), HBM-bandwidth-bound path.
//
// One fused kernel per integrator substage (SURVEY.md 8(a) rows a-H1..a-H3):
//     (Mx,My) <- (1/N) * sum of the previous kernel's per-CTA partial sums        eq.(7)
//     s,c = sincos(theta_i);  f_i = c*My - s*Mx                                    eq.(6)
//     p_i += kickA*f_i [; p_i += kickB*f_i]                                        listing steps 2,5,8,11
//     theta_i += drift*p_i                                                         listing steps 3,6,9
//     s',c' = sincos(theta_i);  per-CTA partial (sum c', sum s') -> partial_out    eq.(7) at the new angles
// so every substage streams theta and p through HBM exactly once (32 B per particle: 16 read,
// 16 written in place).  The paper stores cos/sin in global memory to avoid recomputing them
// (PAPER.md:80); on B200 recomputing (20 FP64 instructions) is cheaper than +32 B per particle.
//
// Determinism: the grid size G is fixed per context; every thread visits a fixed set of
// particles in a fixed order, block sums use fixed trees, and the G partials are summed in a
// fixed order by EVERY CTA of the consuming kernel (no atomics, no "last block" ticket, no
// fences) — all CTAs therefore get bit-identical (Mx, My).
#pragma once

#include <cooperative_groups.h>

#include "common.cuh"
#include "trig.cuh"

namespace lrmd {

constexpr int kHmfThreads = 256;
constexpr int kHmfMaxGrid = 148 * 8;

struct alignas(32) dbl4 { double a, b, c, d; };

__device__ __forceinline__ dbl4 ld256(const double* p) {
    dbl4 v;
    asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v.a), "=d"(v.b), "=d"(v.c), "=d"(v.d) : "l"(p));
    return v;
}
__device__ __forceinline__ void st256(double* p, const dbl4& v) {
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(v.a), "d"(v.b), "d"(v.c), "d"(v.d) : "memory");
}

// (Mx, My) from the producer's partial sums; identical in every thread of every CTA.
template <int THREADS>
__device__ __forceinline__ void hmf_magnetisation(const double2* __restrict__ partial_in, int g_in, double inv_n,
                                                  double* scratch, double& Mx, double& My) {
    double v[2] = {0.0, 0.0};
    for (int i = threadIdx.x; i < g_in; i += THREADS) {
        const double2 q = partial_in[i];
        v[0] += q.x;
        v[1] += q.y;
    }
    block_sum<THREADS, 2>(v, scratch);
    Mx = v[0] * inv_n;
    My = v[1] * inv_n;
}

// sin / cos of four angles.  One range check for the group keeps the common path free of branches
// (the kernel is limited by instruction issue as much as by HBM); a group with an angle beyond
// 2^30 takes the checked per-particle form, which gives every particle the same bits either way.
__device__ __forceinline__ void sincos4(const double (&x)[4], double (&s)[4], double (&c)[4]) {
    if (sincos_is_small(x[0]) && sincos_is_small(x[1]) && sincos_is_small(x[2]) && sincos_is_small(x[3])) {
#pragma unroll
        for (int k = 0; k < 4; ++k) sincos_fast(x[k], s[k], c[k]);
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const double2 r = sincos_any_call(x[k]);
            s[k] = r.x;
            c[k] = r.y;
        }
    }
}

// One substage for four particles: kick with the force at the current angles, drift, and the
// cos / sin terms of the new angles added to the thread's partial sums (particles 0,1 count if
// v01, particles 2,3 if v23: invalid slots carry zeros and are computed but not summed).
template <bool KICK, bool KICK2, bool DRIFT, bool REDUCE>
__device__ __forceinline__ void hmf_group4(double (&th)[4], double (&p)[4], bool v01, bool v23, double Mx, double My,
                                           double kickA, double kickB, double drift, double& accC, double& accS) {
    double s[4], c[4];
    if (KICK) {
        sincos4(th, s, c);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const double f = fma(c[k], My, -(s[k] * Mx));
            p[k] = fma(kickA, f, p[k]);
            if (KICK2) p[k] = fma(kickB, f, p[k]);
        }
    }
    if (DRIFT) {
#pragma unroll
        for (int k = 0; k < 4; ++k) th[k] = fma(drift, p[k], th[k]);
    }
    if (REDUCE) {
        sincos4(th, s, c);
        if (v01) { accC += c[0]; accS += s[0]; accC += c[1]; accS += s[1]; }
        if (v23) { accC += c[2]; accS += s[2]; accC += c[3]; accS += s[3]; }
    }
}

// One particle (ragged tails).
template <bool KICK, bool KICK2, bool DRIFT, bool REDUCE>
__device__ __forceinline__ void hmf_particle(double& th, double& p, double Mx, double My, double kickA, double kickB,
                                             double drift, double& accC, double& accS) {
    if (KICK) {
        double s, c;
        sincos_any(th, s, c);
        const double f = fma(c, My, -(s * Mx));
        p = fma(kickA, f, p);
        if (KICK2) p = fma(kickB, f, p);
    }
    if (DRIFT) th = fma(drift, p, th);
    if (REDUCE) {
        double s, c;
        sincos_any(th, s, c);
        accC += c;
        accS += s;
    }
}

// KICK: apply p += kickA f (and kickB f if KICK2) with M from partial_in.
// DRIFT: theta += drift p.   REDUCE: write per-CTA (sum cos, sum sin) of the final angles.
template <bool KICK, bool KICK2, bool DRIFT, bool REDUCE>
__global__ void __launch_bounds__(kHmfThreads)
hmf_substage_kernel(double* __restrict__ theta, double* __restrict__ p, long long N, double inv_n, double kickA,
                    double kickB, double drift, const double2* __restrict__ partial_in, int g_in,
                    double2* __restrict__ partial_out) {
    __shared__ double scratch[2 * (kHmfThreads / 32)];
    const long long nvec = N >> 2;
    const long long stride = (long long)gridDim.x * kHmfThreads;
    long long v = (long long)blockIdx.x * kHmfThreads + threadIdx.x;

    // issue the first loads before the (latency-bound) magnetisation prologue
    dbl4 t4 = {0, 0, 0, 0}, p4 = {0, 0, 0, 0};
    const bool have = v < nvec;
    if (have) {
        t4 = ld256(theta + 4 * v);
        if (KICK || DRIFT) p4 = ld256(p + 4 * v);
    }
    double Mx = 0.0, My = 0.0;
    if (KICK) hmf_magnetisation<kHmfThreads>(partial_in, g_in, inv_n, scratch, Mx, My);

    double accC = 0.0, accS = 0.0;
    while (v < nvec) {
        const long long vn = v + stride;
        dbl4 tn = {0, 0, 0, 0}, pn = {0, 0, 0, 0};
        if (vn < nvec) {   // software prefetch of the next chunk
            tn = ld256(theta + 4 * vn);
            if (KICK || DRIFT) pn = ld256(p + 4 * vn);
        }
        {
            double tt[4] = {t4.a, t4.b, t4.c, t4.d}, pp[4] = {p4.a, p4.b, p4.c, p4.d};
            hmf_group4<KICK, KICK2, DRIFT, REDUCE>(tt, pp, true, true, Mx, My, kickA, kickB, drift, accC, accS);
            if (DRIFT) st256(theta + 4 * v, dbl4{tt[0], tt[1], tt[2], tt[3]});
            if (KICK) st256(p + 4 * v, dbl4{pp[0], pp[1], pp[2], pp[3]});
        }
        t4 = tn;
        p4 = pn;
        v = vn;
    }
    // ragged tail: N % 4 particles, one per thread of the lowest global thread ids
    {
        const long long g = (long long)blockIdx.x * kHmfThreads + threadIdx.x;
        const long long i = (nvec << 2) + g;
        if (g < 4 && i < N) {
            double th = theta[i], pp = (KICK || DRIFT) ? p[i] : 0.0;
            hmf_particle<KICK, KICK2, DRIFT, REDUCE>(th, pp, Mx, My, kickA, kickB, drift, accC, accS);
            if (DRIFT) theta[i] = th;
            if (KICK) p[i] = pp;
        }
    }
    if (REDUCE) {
        double r[2] = {accC, accS};
        block_sum<kHmfThreads, 2>(r, scratch);
        if (threadIdx.x == 0) partial_out[blockIdx.x] = make_double2(r[0], r[1]);
    }
}

// ---- TMA-staged variant of the fused substage (large N) ------------------------------------------------
// Same arithmetic per particle as hmf_substage_kernel, different data movement: a persistent CTA
// per SM slot streams its chunks of theta and p through an NS-stage shared-memory ring.
//   producer warp (one elected lane): 1-D TMA bulk loads global -> smem (mbarrier complete_tx),
//       and, once the consumers are done with a stage, bulk stores smem -> global of the updated
//       theta / p, then refills the stage as soon as the store has read it (wait_group.read);
//   consumer warps: wait full[s], update their 4 particles of the chunk in place in shared memory,
//       fence.proxy.async, one arrival per warp on done[s]; no CTA-wide barrier in the loop.
// Bytes in flight per SM are set by NS x chunk (up to ~190 KB) instead of by registers per thread,
// and both directions move as full-line bursts.  Chunk c goes to CTA c mod G (fixed), every
// consumer thread adds its cos/sin terms in chunk order, block sums use fixed trees: deterministic.
template <int CONSUMERS, int NS>
struct HmfTma {
    static constexpr int kChunk = 4 * CONSUMERS;            // particles per stage
    static constexpr int kThreads = CONSUMERS + 32;         // + the producer warp
    static constexpr size_t kSmemBytes = (size_t)NS * kChunk * 16 + 2 * NS * sizeof(uint64_t);
};

template <bool KICK, bool KICK2, bool DRIFT, bool REDUCE, int CONSUMERS, int NS, int MINB>
__global__ void __launch_bounds__(CONSUMERS + 32, MINB)
hmf_substage_tma_kernel(double* __restrict__ theta, double* __restrict__ p, long long N, double inv_n, double kickA,
                        double kickB, double drift, const double2* __restrict__ partial_in, int g_in,
                        double2* __restrict__ partial_out) {
    using Cfg = HmfTma<CONSUMERS, NS>;
    constexpr int C = Cfg::kChunk;
    constexpr int T = Cfg::kThreads;
    constexpr bool LOADP = KICK || DRIFT, STORE_TH = DRIFT, STORE_P = KICK, STORE = STORE_TH || STORE_P;
    extern __shared__ __align__(128) unsigned char hmf_smem[];
    double* sth = reinterpret_cast<double*>(hmf_smem);       // [NS][C]
    double* sp = sth + (size_t)NS * C;                       // [NS][C]
    uint64_t* full = reinterpret_cast<uint64_t*>(sp + (size_t)NS * C);
    uint64_t* done = full + NS;
    __shared__ double scratch[2 * (T / 32)];

    const int tid = threadIdx.x;
    const long long Nev = N & ~1LL;                          // bulk copies move multiples of 16 bytes
    const long long nchunks = (Nev + C - 1) / C;
    const long long first = blockIdx.x;
    const int nmine = first < nchunks ? (int)((nchunks - 1 - first) / gridDim.x) + 1 : 0;

    if (tid == CONSUMERS) {
        for (int s = 0; s < NS; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&done[s], CONSUMERS / 32);
        }
        mbar_fence_init();
    }
    __syncthreads();

    auto chunk_base = [&](int k) { return (first + (long long)k * gridDim.x) * C; };
    auto chunk_count = [&](long long i0) { return (int)((Nev - i0 < C) ? (Nev - i0) : C); };
    auto issue_load = [&](int k) {
        const int s = k % NS;
        const long long i0 = chunk_base(k);
        const uint32_t bytes = (uint32_t)chunk_count(i0) * 8u;
        mbar_expect_tx(&full[s], LOADP ? 2u * bytes : bytes);
        bulk_g2s(sth + (size_t)s * C, theta + i0, bytes, &full[s]);
        if (LOADP) bulk_g2s(sp + (size_t)s * C, p + i0, bytes, &full[s]);
    };
    // the first NS chunks are in flight before the (latency-bound) magnetisation prologue
    if (tid == CONSUMERS)
        for (int k = 0; k < NS && k < nmine; ++k) issue_load(k);

    double Mx = 0.0, My = 0.0;
    if (KICK) hmf_magnetisation<T>(partial_in, g_in, inv_n, scratch, Mx, My);

    double accC = 0.0, accS = 0.0;
    if (tid >= CONSUMERS) {
        if (tid == CONSUMERS) {
            for (int k = 0; k < nmine; ++k) {
                const int s = k % NS;
                mbar_wait(&done[s], (uint32_t)((k / NS) & 1));
                if (STORE) {
                    const long long i0 = chunk_base(k);
                    const uint32_t bytes = (uint32_t)chunk_count(i0) * 8u;
                    if (STORE_TH) bulk_s2g(theta + i0, sth + (size_t)s * C, bytes);
                    if (STORE_P) bulk_s2g(p + i0, sp + (size_t)s * C, bytes);
                    bulk_commit();
                }
                if (k + NS < nmine) {
                    if (STORE) bulk_wait_read<0>();   // the store has read stage s: it may be overwritten
                    issue_load(k + NS);
                }
            }
            if (STORE) bulk_wait<0>();
        }
        __syncwarp();
    } else {
        for (int k = 0; k < nmine; ++k) {
            const int s = k % NS;
            const int cnt = chunk_count(chunk_base(k));
            double2* t2 = reinterpret_cast<double2*>(sth + (size_t)s * C);
            double2* p2 = reinterpret_cast<double2*>(sp + (size_t)s * C);
            mbar_wait(&full[s], (uint32_t)((k / NS) & 1));
            // 16-byte units tid and tid + CONSUMERS of the chunk (conflict-free LDS.128 / STS.128)
            const int u0 = tid, u1 = tid + CONSUMERS;
            const bool h0 = 2 * u0 < cnt, h1 = 2 * u1 < cnt;
            double2 ta = make_double2(0.0, 0.0), tb = ta, pa = ta, pb = ta;
            if (h0) { ta = t2[u0]; if (LOADP) pa = p2[u0]; }
            if (h1) { tb = t2[u1]; if (LOADP) pb = p2[u1]; }
            {
                double tt[4] = {ta.x, ta.y, tb.x, tb.y}, pp[4] = {pa.x, pa.y, pb.x, pb.y};
                hmf_group4<KICK, KICK2, DRIFT, REDUCE>(tt, pp, h0, h1, Mx, My, kickA, kickB, drift, accC, accS);
                ta = make_double2(tt[0], tt[1]);
                tb = make_double2(tt[2], tt[3]);
                pa = make_double2(pp[0], pp[1]);
                pb = make_double2(pp[2], pp[3]);
            }
            if (STORE) {
                if (h0) { if (STORE_TH) t2[u0] = ta; if (STORE_P) p2[u0] = pa; }
                if (h1) { if (STORE_TH) t2[u1] = tb; if (STORE_P) p2[u1] = pb; }
                fence_proxy_async_smem();
            }
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(&done[s]);
        }
        // odd N: the last particle does not fit a 16-byte unit
        if (blockIdx.x == 0 && tid == 0 && (N & 1)) {
            const long long i = N - 1;
            double th = theta[i], pp = LOADP ? p[i] : 0.0;
            hmf_particle<KICK, KICK2, DRIFT, REDUCE>(th, pp, Mx, My, kickA, kickB, drift, accC, accS);
            if (STORE_TH) theta[i] = th;
            if (STORE_P) p[i] = pp;
        }
    }
    if (REDUCE) {
        double r[2] = {accC, accS};
        block_sum<T, 2>(r, scratch);
        if (tid == 0) partial_out[blockIdx.x] = make_double2(r[0], r[1]);
    }
}

// ---- cluster-resident variant (small N: the step is latency-bound, SURVEY.md hard part 4) ---------------
// One thread-block cluster of kHmfClusterCtas CTAs holds the whole state in registers (P particles
// per thread) and runs ALL n steps of an lrmd_step call in one launch: 3n + 1 reductions, each
//   per-thread sum -> warp shuffle tree -> shared memory -> warp 0 -> the CTA's (sum cos, sum sin)
//   written into every CTA's shared memory (distributed shared memory, st.shared::cluster)
//   -> barrier.cluster arrive.release / wait.acquire -> every thread adds the C partials in rank order,
// so a substage costs one CTA barrier and one cluster barrier instead of a kernel boundary.  sin / cos
// of the current angles stay in registers from the reduction to the next kick (one sincos per
// particle-substage instead of two).  Deterministic: fixed particle -> thread map, fixed trees.
constexpr int kHmfClusterCtas = 8;      // portable cluster size
constexpr int kHmfClusterCtasMax = 16;  // non-portable size, used when the device grants it
constexpr int kHmfClusterThreads = 320;

__device__ __forceinline__ unsigned cluster_ctarank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned cluster_nctarank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// store (a, b) at the address of `local` in CTA `rank` of the cluster
__device__ __forceinline__ void dsmem_store2(double2* local, unsigned rank, double a, double b) {
    unsigned remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(smem_u32(local)), "r"(rank));
    asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(remote), "d"(a), "d"(b) : "memory");
}

template <int P>
__global__ void __launch_bounds__(kHmfClusterThreads, 1)
hmf_cluster_kernel(double* __restrict__ theta, double* __restrict__ p, long long N, long long nsteps, double kB0,
                   double kB1, double dD0, double dD1, double2* __restrict__ partial_out) {
    constexpr int T = kHmfClusterThreads, NW = T / 32;
    __shared__ double2 warp_part[NW];
    __shared__ double2 cta_part[2][kHmfClusterCtasMax];      // [parity][rank of the writer]
    const int C = (int)cluster_nctarank();  // 8 or 16 CTAs
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const unsigned rank = cluster_ctarank();
    const double inv_n = 1.0 / (double)N;

    double th[P], pp[P], sn[P], cs[P];
    bool valid[P];
#pragma unroll
    for (int k = 0; k < P; ++k) {
        const long long i = (long long)k * (C * T) + (long long)rank * T + tid;
        valid[k] = i < N;
        th[k] = valid[k] ? theta[i] : 0.0;
        pp[k] = valid[k] ? p[i] : 0.0;
    }
    cluster_sync_all();     // every CTA of the cluster is running before the first remote store

    int parity = 0;
    double Mx = 0.0, My = 0.0;
    auto reduce = [&]() {
        bool small = true;
#pragma unroll
        for (int k = 0; k < P; ++k) small = small && sincos_is_small(th[k]);
        if (small) {
#pragma unroll
            for (int k = 0; k < P; ++k) sincos_fast(th[k], sn[k], cs[k]);
        } else {
#pragma unroll
            for (int k = 0; k < P; ++k) {
                const double2 r = sincos_any_call(th[k]);
                sn[k] = r.x;
                cs[k] = r.y;
            }
        }
        double aC = 0.0, aS = 0.0;
#pragma unroll
        for (int k = 0; k < P; ++k)
            if (valid[k]) { aC += cs[k]; aS += sn[k]; }
        aC = warp_sum(aC);
        aS = warp_sum(aS);
        if (lane == 0) warp_part[w] = make_double2(aC, aS);
        __syncthreads();
        if (w == 0) {
            const double2 q = (lane < NW) ? warp_part[lane] : make_double2(0.0, 0.0);
            const double tC = warp_sum(q.x), tS = warp_sum(q.y);
            if (lane < C) dsmem_store2(&cta_part[parity][rank], (unsigned)lane, tC, tS);
        }
        cluster_sync_all();
        double sC = 0.0, sS = 0.0;
        for (int r = 0; r < C; ++r) {
            const double2 q = cta_part[parity][r];
            sC += q.x;
            sS += q.y;
        }
        Mx = sC * inv_n;
        My = sS * inv_n;
        parity ^= 1;
    };
    auto kick = [&](double kc) {
#pragma unroll
        for (int k = 0; k < P; ++k) pp[k] = fma(kc, fma(cs[k], My, -(sn[k] * Mx)), pp[k]);
    };
    auto drift = [&](double dc) {
#pragma unroll
        for (int k = 0; k < P; ++k) th[k] = fma(dc, pp[k], th[k]);
    };

    reduce();                                   // f(q(t)): listing step 1
    for (long long s = 0; s < nsteps; ++s) {    // listing steps 2-11, readings G2-G4
        kick(kB0); drift(dD0); reduce();
        kick(kB1); drift(dD1); reduce();
        kick(kB1); drift(dD0); reduce();
        kick(kB0);
    }
#pragma unroll
    for (int k = 0; k < P; ++k) {
        const long long i = (long long)k * (C * T) + (long long)rank * T + tid;
        if (valid[k]) { theta[i] = th[k]; p[i] = pp[k]; }
    }
    // the sums at the final angles, for lrmd_forces / lrmd_energy / the next call (reading G3)
    if (rank == 0 && tid < C) partial_out[tid] = cta_part[parity ^ 1][tid];
}

// ---- grid-resident variant (20,480 < N < 1e6: the paper's Table 1 sizes 1e5 .. 1e6) ----------------
// Between the cluster-resident kernel and the HBM regime the state (16 N bytes) fits the GPU's shared memory, and a
// substage's arithmetic takes 0.2 - 2 us: what a step costs is the kernel boundary between substages (7.7 us each with
// a replayed CUDA graph).  One cooperative launch of one CTA per SM keeps the whole state — angles, momenta and the
// sin / cos of the current angles — in shared memory and runs ALL n steps of an lrmd_step call; a substage is one
// pass over the CTA's particles (kick, drift, sincos, partial sums), a block reduction, the CTA's (sum cos, sum sin)
// written to a double-buffered array in global memory, a grid barrier (cooperative groups grid.sync(); a hand-written
// all-gather on per-CTA flag words measured 7.5 us per substage against 3.1 us and was dropped), and a fixed tree over
// the G partials that every CTA evaluates identically.  Deterministic: fixed particle -> CTA -> thread map, fixed trees.
constexpr int kHmfGridThreads = 512;
constexpr int kHmfGridBytesPerParticle = 32;                        // theta, p, sin, cos
constexpr int kHmfGridMaxLocal = (227 * 1024 - 1024) / kHmfGridBytesPerParticle;   // particles per CTA that fit

__global__ void __launch_bounds__(kHmfGridThreads, 1)
hmf_grid_kernel(double* __restrict__ theta, double* __restrict__ p, long long N, int nlocal, long long nsteps, double kB0,
                double kB1, double dD0, double dD1, double2* __restrict__ part2, double2* __restrict__ partial_out) {
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    extern __shared__ __align__(16) unsigned char hmf_grid_smem[];
    constexpr int T = kHmfGridThreads, NW = T / 32;
    __shared__ double scratch[2 * NW];
    __shared__ double2 wtot[8];
    double* th = reinterpret_cast<double*>(hmf_grid_smem);
    double* pp = th + nlocal;
    double* sn = pp + nlocal;
    double* cs = sn + nlocal;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int G = (int)gridDim.x;
    const long long i0 = (long long)blockIdx.x * nlocal;
    const int n = (int)((N - i0 < nlocal) ? (N - i0 > 0 ? N - i0 : 0) : nlocal);
    const double inv_n = 1.0 / (double)N;
    for (int k = tid; k < n; k += T) {
        th[k] = theta[i0 + k];
        pp[k] = p[i0 + k];
    }
    __syncthreads();

    int parity = 0;
    double Mx = 0.0, My = 0.0;
    // One substage: [kick kA (+ kB)] -> [drift] -> sincos -> (Mx, My).  KICK = 0: the first reduction of the call.
    auto pass = [&](int kicks, double kA, double kB, double dc) {
        double aC = 0.0, aS = 0.0;
        for (int k = tid; k < n; k += T) {
            double x = th[k];
            if (kicks > 0) {
                const double f = fma(cs[k], My, -(sn[k] * Mx));
                double q = fma(kA, f, pp[k]);
                if (kicks > 1) q = fma(kB, f, q);
                pp[k] = q;
                x = fma(dc, q, x);
                th[k] = x;
            }
            double s, c;
            sincos_any(x, s, c);
            sn[k] = s;
            cs[k] = c;
            aC += c;
            aS += s;
        }
        double r[2] = {aC, aS};
        block_sum<T, 2>(r, scratch);
        if (tid == 0) {
            __stcg(reinterpret_cast<double*>(&part2[(size_t)parity * G + blockIdx.x]), r[0]);
            __stcg(reinterpret_cast<double*>(&part2[(size_t)parity * G + blockIdx.x]) + 1, r[1]);
        }
        grid.sync();
        // the same tree in every CTA: thread t < G takes partial t; xor-shuffle trees in warps 0 .. 7, then in order
        double qx = 0.0, qy = 0.0;
        if (tid < G) {
            qx = __ldcg(reinterpret_cast<const double*>(&part2[(size_t)parity * G + tid]));
            qy = __ldcg(reinterpret_cast<const double*>(&part2[(size_t)parity * G + tid]) + 1);
        }
        if (w < 8) {
            qx = warp_sum(qx);
            qy = warp_sum(qy);
            if (lane == 0) wtot[w] = make_double2(qx, qy);
        }
        __syncthreads();
        double sC = 0.0, sS = 0.0;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            sC += wtot[k].x;
            sS += wtot[k].y;
        }
        Mx = sC * inv_n;
        My = sS * inv_n;
        parity ^= 1;
        __syncthreads();      // wtot is rewritten by the next pass
    };

    pass(0, 0.0, 0.0, 0.0);                          // f(q(t)): listing step 1
    for (long long s = 0; s < nsteps; ++s) {         // listing steps 2-11, readings G2-G4
        // the closing kick B0 of the previous step and this step's opening kick: two FMAs with the same force
        if (s == 0) pass(1, kB0, 0.0, dD0);
        else pass(2, kB0, kB0, dD0);
        pass(1, kB1, 0.0, dD1);
        pass(1, kB1, 0.0, dD0);
    }
    for (int k = tid; k < n; k += T) {
        double q = pp[k];
        if (nsteps > 0) q = fma(kB0, fma(cs[k], My, -(sn[k] * Mx)), q);      // closing kick of the last step
        theta[i0 + k] = th[k];
        p[i0 + k] = q;
    }
    // the per-CTA sums at the final angles, for lrmd_forces / lrmd_energy / the next call (reading G3)
    if (blockIdx.x == 0 && tid < G) {
        const double2 v = make_double2(__ldcg(reinterpret_cast<const double*>(&part2[(size_t)(parity ^ 1) * G + tid])),
                                       __ldcg(reinterpret_cast<const double*>(&part2[(size_t)(parity ^ 1) * G + tid]) + 1));
        partial_out[tid] = v;
    }
}

// Sharded runs ("each GPU computes its contribution to the magnetisation, which are then summed"):
// the per-CTA partials of this rank, added in index order, as ONE (sum cos, sum sin) pair that the caller's
// all-reduce sums over ranks in place; the next kernel then reads it with g_in = 1.
__global__ void __launch_bounds__(kHmfThreads)
hmf_collapse_kernel(const double2* __restrict__ partial_in, int g_in, double2* __restrict__ out1) {
    __shared__ double scratch[2 * (kHmfThreads / 32)];
    double v[2] = {0.0, 0.0};
    for (int i = threadIdx.x; i < g_in; i += kHmfThreads) {
        const double2 q = partial_in[i];
        v[0] += q.x;
        v[1] += q.y;
    }
    block_sum<kHmfThreads, 2>(v, scratch);
    if (threadIdx.x == 0) *out1 = make_double2(v[0], v[1]);
}

// f_i = cos(theta_i) My - sin(theta_i) Mx  -> f   (lrmd_forces; eq.(6))
__global__ void __launch_bounds__(kHmfThreads)
hmf_force_kernel(const double* __restrict__ theta, double* __restrict__ f, long long N, double inv_n,
                 const double2* __restrict__ partial_in, int g_in) {
    __shared__ double scratch[2 * (kHmfThreads / 32)];
    double Mx, My;
    hmf_magnetisation<kHmfThreads>(partial_in, g_in, inv_n, scratch, Mx, My);
    const long long stride = (long long)gridDim.x * kHmfThreads;
    for (long long i = (long long)blockIdx.x * kHmfThreads + threadIdx.x; i < N; i += stride) {
        double s, c;
        sincos_any(theta[i], s, c);
        f[i] = fma(c, My, -(s * Mx));
    }
}

// Per-CTA partial sums of up to two arrays: (sum a^2 [+ b^2], sum a, sum b) -> part[3*blockIdx..]
// Used for K = 1/2 sum p^2 and the total momentum of all three models.
__global__ void __launch_bounds__(kHmfThreads)
kinetic_partial_kernel(const double* __restrict__ a, const double* __restrict__ b, long long N,
                       double* __restrict__ part) {
    __shared__ double scratch[3 * (kHmfThreads / 32)];
    double r[3] = {0.0, 0.0, 0.0};
    const long long stride = (long long)gridDim.x * kHmfThreads;
    for (long long i = (long long)blockIdx.x * kHmfThreads + threadIdx.x; i < N; i += stride) {
        const double x = a[i];
        r[0] = fma(x, x, r[0]);
        r[1] += x;
        if (b) {
            const double y = b[i];
            r[0] = fma(y, y, r[0]);
            r[2] += y;
        }
    }
    block_sum<kHmfThreads, 3>(r, scratch);
    if (threadIdx.x == 0) {
        part[3 * blockIdx.x + 0] = r[0];
        part[3 * blockIdx.x + 1] = r[1];
        part[3 * blockIdx.x + 2] = r[2];
    }
}

// One CTA: out4 = {K, V, a, b}.
//   kpart: g_k triples from kinetic_partial_kernel.
//   HMF (model 0): mpart = g_m (sum cos, sum sin) partials; V = (N/2)(1 - Mx^2 - My^2), eq.(5) PAPER.md:69;
//                  (a, b) = (Mx, My).
//   pair models:   vpart = g_v partial sums of the pair-potential kernel, already scaled; V = sum;
//                  (a, b) = total momentum.
__global__ void __launch_bounds__(kHmfThreads)
energy_finalize_kernel(int model, long long N, const double* __restrict__ kpart, int g_k,
                       const double2* __restrict__ mpart, int g_m, const double* __restrict__ vpart, int g_v,
                       double* __restrict__ out4) {
    __shared__ double scratch[3 * (kHmfThreads / 32)];
    double r[3] = {0.0, 0.0, 0.0};
    for (int i = threadIdx.x; i < g_k; i += kHmfThreads) {
        r[0] += kpart[3 * i];
        r[1] += kpart[3 * i + 1];
        r[2] += kpart[3 * i + 2];
    }
    block_sum<kHmfThreads, 3>(r, scratch);
    const double K = 0.5 * r[0];
    double V, a = r[1], b = r[2];
    if (model == 0) {
        double Mx, My;
        hmf_magnetisation<kHmfThreads>(mpart, g_m, 1.0 / (double)N, scratch, Mx, My);   // N = all particles
        V = 0.5 * (double)N * (1.0 - Mx * Mx - My * My);
        a = Mx;
        b = My;
    } else {
        double v[1] = {0.0};
        for (int i = threadIdx.x; i < g_v; i += kHmfThreads) v[0] += vpart[i];
        block_sum<kHmfThreads, 1>(v, scratch);
        V = v[0];
    }
    if (threadIdx.x == 0) {
        out4[0] = K;
        out4[1] = V;
        out4[2] = a;
        out4[3] = b;
    }
}

}  // namespace lrmd
