// trig.cuh — fp64 sincos for the HMF / Ring hot path ("The most demanding part of
// an integration step is the computation of the sine and cosine of the position angles").
//
// 20 FP64-pipe instructions on the fast path and NO fp64<->int conversions (F2I.F64 / I2F.F64 run
// at a fraction of the DFMA rate): the quadrant is rounded with the add-magic-constant trick.
//   k = rint(x * 2/pi)              1 DFMA + 1 DADD
//   r = x - k*pi/2 (3-term FMA)     3 DFMA             |r| <= pi/4 (+ rounding)
//   u = r*r                          1 DMUL
//   sin r = r + (r u) S(u)           5 DFMA + 1 DMUL + 1 DFMA
//   cos r = 1 + u (-1/2 + u C(u))    5 DFMA + 2 DFMA
// Coefficients: gen_trig_coeffs.py (degree-5 Chebyshev fits; approximation error 2^-55 / 2^-59).
// Total error <= ~1 ulp for |x| < 2^30; larger arguments take CUDA's sincos() (Payne-Hanek),
// out of line.
#pragma once

#include <cmath>
#include <cstring>
#include <cuda_runtime.h>

namespace lrmd {

// Bit access that also compiles for the host (csrc/host_check.cu runs this arithmetic on the
// CPU in the -m "not gpu" tests).
__host__ __device__ __forceinline__ int dbl_lo(double x) {
#ifdef __CUDA_ARCH__
    return __double2loint(x);
#else
    unsigned long long b; std::memcpy(&b, &x, 8); return (int)(unsigned)(b & 0xffffffffull);
#endif
}
__host__ __device__ __forceinline__ int dbl_hi(double x) {
#ifdef __CUDA_ARCH__
    return __double2hiint(x);
#else
    unsigned long long b; std::memcpy(&b, &x, 8); return (int)(unsigned)(b >> 32);
#endif
}
__host__ __device__ __forceinline__ double dbl_make(int hi, int lo) {
#ifdef __CUDA_ARCH__
    return __hiloint2double(hi, lo);
#else
    unsigned long long b = ((unsigned long long)(unsigned)hi << 32) | (unsigned)lo;
    double x; std::memcpy(&x, &b, 8); return x;
#endif
}

__host__ __device__ __noinline__ void sincos_huge(double x, double* s, double* c) {
#ifdef __CUDA_ARCH__
    ::sincos(x, s, c);
#else
    *s = std::sin(x); *c = std::cos(x);
#endif
}

__host__ __device__ __forceinline__ void sincos_pi4(double x, double& s, double& c) {
    constexpr double kTwoOverPi = 0x1.45f306dc9c883p-1;
    constexpr double kMagic = 6755399441055744.0;   // 1.5 * 2^52
    constexpr double kPio2Hi = 0x1.921fb54442d18p+0;
    constexpr double kPio2Mid = 0x1.1a62633145c07p-54;
    constexpr double kPio2Lo = -0x1.f1976b7ed8fbcp-110;

    // |x| >= 2^30, inf or NaN: rare, out of line.  Integer compare on the high word (ALU pipe,
    // not a DSETP on the FP64 pipe): 2^30 has high word 0x41D00000.
    if ((dbl_hi(x) & 0x7fffffff) >= 0x41D00000) {
        sincos_huge(x, &s, &c);
        return;
    }
    const double t = fma(x, kTwoOverPi, kMagic);
    const unsigned q = (unsigned)dbl_lo(t);   // k mod 2^32 (two's complement)
    const double k = t - kMagic;
    double r = fma(-k, kPio2Hi, x);
    r = fma(-k, kPio2Mid, r);
    r = fma(-k, kPio2Lo, r);
    const double u = r * r;

    double ps = 0x1.5dfb4dfaf15abp-33;
    ps = fma(ps, u, -0x1.ae5fdeb852566p-26);
    ps = fma(ps, u, 0x1.71de376b9c575p-19);
    ps = fma(ps, u, -0x1.a01a019e623afp-13);
    ps = fma(ps, u, 0x1.1111111110b23p-7);
    ps = fma(ps, u, -0x1.5555555555555p-3);
    const double ru = r * u;
    const double sr = fma(ru, ps, r);

    double pc = -0x1.906dd38cb66a1p-37;
    pc = fma(pc, u, 0x1.1eeb52bea9072p-29);
    pc = fma(pc, u, -0x1.27e4fa025e03dp-22);
    pc = fma(pc, u, 0x1.a01a019f3df42p-16);
    pc = fma(pc, u, -0x1.6c16c16c1691fp-10);
    pc = fma(pc, u, 0x1.5555555555555p-5);
    pc = fma(pc, u, -0.5);
    const double cr = fma(pc, u, 1.0);

    // quadrant: q&1 swaps, sign bits flipped with integer ops (ALU pipe, not FP64)
    const double a = (q & 1) ? cr : sr;    // |sin|
    const double b = (q & 1) ? sr : cr;    // |cos|
    const unsigned sflip = (q & 2u) << 30;           // sin negative in quadrants 2, 3
    const unsigned cflip = ((q + 1u) & 2u) << 30;    // cos negative in quadrants 1, 2
    s = dbl_make((int)((unsigned)dbl_hi(a) ^ sflip), dbl_lo(a));
    c = dbl_make((int)((unsigned)dbl_hi(b) ^ cflip), dbl_lo(b));
}

}  // namespace lrmd
