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
//
// The HMF kernel is bound by instruction issue as much as by HBM once its data movement is
// right, so the constants live in __constant__ memory (an FP64 instruction takes a constant-bank
// operand for free, whereas a 64-bit immediate costs two extra moves each time the register
// allocator rematerialises it), and the range check is hoisted by the callers: sincos_fast() has
// no branch, sincos_is_small() is one integer compare, sincos_any() is the checked form.
#pragma once

#include <cmath>
#include <cstring>
#include <cuda_runtime.h>

namespace lrmd {

// Bit access that also compiles for the host (lrmd_host_sincos runs this arithmetic on the CPU in
// the -m "not gpu" tests).
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

// Constants: [0] 2/pi, [1] 1.5*2^52, [2..4] pi/2 split in three, [5..10] S highest degree first,
// [11..17] C highest degree first followed by -1/2.
#define LRMD_TRIG_TABLE                                                                                     \
    {0x1.45f306dc9c883p-1, 6755399441055744.0, 0x1.921fb54442d18p+0, 0x1.1a62633145c07p-54,                 \
     -0x1.f1976b7ed8fbcp-110, 0x1.5dfb4dfaf15abp-33, -0x1.ae5fdeb852566p-26, 0x1.71de376b9c575p-19,         \
     -0x1.a01a019e623afp-13, 0x1.1111111110b23p-7, -0x1.5555555555555p-3, -0x1.906dd38cb66a1p-37,           \
     0x1.1eeb52bea9072p-29, -0x1.27e4fa025e03dp-22, 0x1.a01a019f3df42p-16, -0x1.6c16c16c1691fp-10,          \
     0x1.5555555555555p-5, -0.5}
static __constant__ double kTrigDev[18] = LRMD_TRIG_TABLE;
static const double kTrigHost[18] = LRMD_TRIG_TABLE;
#ifdef __CUDA_ARCH__
#define LRMD_TRIG(i) kTrigDev[i]
#else
#define LRMD_TRIG(i) kTrigHost[i]
#endif

// |x| < 2^30 (and not inf / NaN): integer compare on the high word (ALU pipe, not a DSETP on the
// FP64 pipe); 2^30 has high word 0x41D00000.
__host__ __device__ __forceinline__ bool sincos_is_small(double x) {
    return (dbl_hi(x) & 0x7fffffff) < 0x41D00000;
}

// Requires sincos_is_small(x).
__host__ __device__ __forceinline__ void sincos_fast(double x, double& s, double& c) {
    const double magic = LRMD_TRIG(1);
    const double t = fma(x, LRMD_TRIG(0), magic);
    const unsigned q = (unsigned)dbl_lo(t);   // k mod 2^32 (two's complement)
    const double k = t - magic;
    double r = fma(-k, LRMD_TRIG(2), x);
    r = fma(-k, LRMD_TRIG(3), r);
    r = fma(-k, LRMD_TRIG(4), r);
    const double u = r * r;

    double ps = LRMD_TRIG(5);
    ps = fma(ps, u, LRMD_TRIG(6));
    ps = fma(ps, u, LRMD_TRIG(7));
    ps = fma(ps, u, LRMD_TRIG(8));
    ps = fma(ps, u, LRMD_TRIG(9));
    ps = fma(ps, u, LRMD_TRIG(10));
    const double ru = r * u;
    const double sr = fma(ru, ps, r);

    double pc = LRMD_TRIG(11);
    pc = fma(pc, u, LRMD_TRIG(12));
    pc = fma(pc, u, LRMD_TRIG(13));
    pc = fma(pc, u, LRMD_TRIG(14));
    pc = fma(pc, u, LRMD_TRIG(15));
    pc = fma(pc, u, LRMD_TRIG(16));
    pc = fma(pc, u, LRMD_TRIG(17));
    const double cr = fma(pc, u, 1.0);

    // quadrant: q&1 swaps, sign bits flipped with integer ops (ALU pipe, not FP64)
    const double a = (q & 1) ? cr : sr;    // |sin|
    const double b = (q & 1) ? sr : cr;    // |cos|
    const unsigned sflip = (q & 2u) << 30;           // sin negative in quadrants 2, 3
    const unsigned cflip = ((q + 1u) & 2u) << 30;    // cos negative in quadrants 1, 2
    s = dbl_make((int)((unsigned)dbl_hi(a) ^ sflip), dbl_lo(a));
    c = dbl_make((int)((unsigned)dbl_hi(b) ^ cflip), dbl_lo(b));
}

// Any argument, out of line: CUDA's sincos (Payne-Hanek reduction for huge |x|, NaN for inf / NaN).
// Returns (sin, cos) in registers.
__host__ __device__ __noinline__ double2 sincos_slow(double x) {
    double2 r;
#ifdef __CUDA_ARCH__
    ::sincos(x, &r.x, &r.y);
#else
    r.x = std::sin(x); r.y = std::cos(x);
#endif
    return r;
}

// Checked form for one-particle-per-thread callers.
__host__ __device__ __forceinline__ void sincos_any(double x, double& s, double& c) {
    if (sincos_is_small(x)) {
        sincos_fast(x, s, c);
    } else {
        const double2 r = sincos_slow(x);
        s = r.x;
        c = r.y;
    }
}

// The checked form as an out-of-line call returning (sin, cos) in registers: the cold path of
// callers that hoist the range check over a group of angles.
__host__ __device__ __noinline__ double2 sincos_any_call(double x) {
    double2 r;
    sincos_any(x, r.x, r.y);
    return r;
}

}  // namespace lrmd
