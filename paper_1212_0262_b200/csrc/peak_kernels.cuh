// peak_kernels.cuh — FP64 issue-rate microbenchmark behind lrmd_fp64_peak (hard part 8:
// "the build must measure a DFMA-only peak and the clock held").  It is the measured counterpart of the derived
// `alu` roofline denominator 148 SMs x 64 FP64 lanes x sm_max_mhz that bench.py quotes for the pair kernels
// (the O(N^2) force loop is pure FP64 arithmetic once the j-tile is on chip).
//
// One thread runs 16 independent dependency chains of one FP64 operation (DFMA, DMUL or DADD) and, per group of
// 16 FP64 instructions, XN instructions of another class on their own independent chains.  The mixes answer the
// question the pair kernels' design turns on: how many FP64-pipe issue cycles does a non-FP64 instruction (the
// MUFU seed, a shuffle, a shared-memory load, an integer op) of the same warp cost?
#pragma once

#include "common.cuh"

namespace lrmd {

// op: what the 16 chains execute.  The DFMA flavours differ in how many of the three 64-bit source operands are
// private to the chain (the register file feeds a 3-register DFMA more slowly than a 2-register DMUL / DADD unless
// operands are shared between consecutive instructions or are immediates):
//   kPeakDfma      a = fma(a, m, c)      m, c shared by all chains
//   kPeakDfma3     a = fma(b_k, c_k, a)  three private registers (the accumulate of a pair kernel: fma(dx, y, fx))
//   kPeakDfma2     a = fma(a, b_k, c)    one shared register
//   kPeakDfmaSq    a = fma(a, a, c)      a register used twice (fma(dx, dx, eps))
//   kPeakDfmaImm   a = fma(a, m, 1.0)    immediate addend (fma(-r2, y0, 1.0))
enum { kPeakDfma = 0, kPeakDmul = 1, kPeakDadd = 2, kPeakDfma3 = 3, kPeakDfma2 = 4, kPeakDfmaSq = 5, kPeakDfmaImm = 6 };
enum { kMixNone = 0, kMixInt = 1, kMixMufu = 2, kMixShfl = 3, kMixLds = 4, kMixMufuSeed = 5, kMixMov = 6, kMixSts = 7 };

constexpr int kPeakThreads = 128;
constexpr int kPeakChains = 16;

// out[blockIdx.x * blockDim.x + threadIdx.x] receives a value that depends on every chain (so that nothing is
// eliminated); clk[2 * blockIdx.x + {0, 1}] receive the CTA's elapsed SM cycles (clock64) and nanoseconds
// (globaltimer): their ratio over all CTAs is the SM clock held during the run.
template <int OP, int XK, int XN>
__global__ void __launch_bounds__(kPeakThreads)
fp64_peak_kernel(double* __restrict__ out, const double* __restrict__ seedv, int iters, unsigned long long* __restrict__ clk) {
    __shared__ double sm[kPeakThreads * 2];
    const int tid = threadIdx.x;
    // operands come from memory so that nothing folds at compile time: m ~ 1, c ~ 0
    const double m = seedv[0], c = seedv[1];
    double a[kPeakChains];
#pragma unroll
    for (int k = 0; k < kPeakChains; ++k) a[k] = seedv[2] + (double)(tid + k);
    double pb[kPeakChains], pc[kPeakChains];      // private operands of the kPeakDfma3 / kPeakDfma2 chains
#pragma unroll
    for (int k = 0; k < kPeakChains; ++k) { pb[k] = m + 1e-12 * (double)(tid + k); pc[k] = c * (double)(k + 1) * 1e-3; }
    int xi[8];
    double xd[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) { xi[k] = tid + k; xd[k] = 1.5 + 0.001 * (double)(tid + k); }
    sm[tid] = (double)tid;
    sm[tid + kPeakThreads] = (double)(tid + 1);
    __syncthreads();
    unsigned long long t0, c0;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    c0 = clock64();
#pragma unroll 2
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < kPeakChains; ++k) {
            if (OP == kPeakDfma) a[k] = fma(a[k], m, c);
            else if (OP == kPeakDmul) a[k] = a[k] * m;
            else if (OP == kPeakDadd) a[k] = a[k] + c;
            else if (OP == kPeakDfma3) a[k] = fma(pb[k], pc[k], a[k]);
            else if (OP == kPeakDfma2) a[k] = fma(a[k], pb[k], c);
            else if (OP == kPeakDfmaSq) a[k] = fma(a[k], a[k], c);
            else a[k] = fma(a[k], m, 1.0);
            // the extras are spread evenly between the FP64 instructions
            constexpr int STRIDE = XN > 0 ? kPeakChains / XN : kPeakChains + 1;
            if (XN > 0 && k % STRIDE == 0) {
                const int x = (k / STRIDE) & 7;
                if (XK == kMixInt) {
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(xi[x]) : "r"(it), "r"(tid));   // alu pipe
                } else if (XK == kMixMufu) {
                    asm volatile("rcp.approx.ftz.f64 %0, %0;" : "+d"(xd[x]));   // MUFU.RCP64H (+ the MOV of the low word)
                } else if (XK == kMixMufuSeed) {
                    // the seed as the pair kernels use it: MUFU.RCP64H of a value, consumed by one DFMA
                    double y;
                    asm volatile("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(xd[x]));
                    xd[x] = fma(-xd[x], y, 2.5);
                } else if (XK == kMixShfl) {
                    xi[x] = __shfl_sync(0xffffffffu, xi[x], (tid + 1) & 31);
                } else if (XK == kMixLds) {
                    xd[x] = sm[(tid + (x + it) * 32) & (2 * kPeakThreads - 1)];
                    asm volatile("" : "+d"(xd[x]));
                } else if (XK == kMixMov) {
                    asm volatile("mov.b32 %0, %1;" : "=r"(xi[x]) : "r"(xi[(x + 1) & 7]));
                } else if (XK == kMixSts) {
                    sm[(tid + x * 32) & (2 * kPeakThreads - 1)] = xd[x];
                }
            }
        }
    }
    const unsigned long long c1 = clock64();
    unsigned long long t1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < kPeakChains; ++k) s += a[k];
#pragma unroll
    for (int k = 0; k < 8; ++k) s += xd[k] + (double)xi[k];
#pragma unroll
    for (int k = 0; k < kPeakChains; ++k) s += pb[k] + pc[k];
    s += sm[(tid * 7) & (2 * kPeakThreads - 1)];
    out[(size_t)blockIdx.x * kPeakThreads + tid] = s;
    if (tid == 0) {
        clk[2 * blockIdx.x] = c1 - c0;
        clk[2 * blockIdx.x + 1] = t1 - t0;
    }
}

}  // namespace lrmd
