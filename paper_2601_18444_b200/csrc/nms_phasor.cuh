// nms_phasor.cuh -- the phasor e^{-i Psi} of Eq. 42-47 (L353-L368) from an EXACTLY reduced phase.
//
// The amplitude kernels form the phase in cycles, t = (q / 2 pi) . r, with one fp64 FMA whose addend MAGIC = 1.5 * 2^20
// makes the adder round to a multiple of 2^-32 cycle: the low mantissa word of the result is k = frac(t) * 2^32 as a
// two's-complement integer in [-2^31, 2^31) -- the "t - rint(t)" reduction of the north star done by the rounding of
// the adder, for any |t| < 2^19 cycles, with no fp32 phase rounding.  Two evaluations of {cos, sin}(2 pi k / 2^32):
//
//   phasor_mufu(k)  XU pipe: I2FP, FMUL, sin.approx + cos.approx (MUFU; absolute error <= 2^-21.4 per value, CUDA C
//                   Programming Guide).  6 issue slots, 2 of them on the 16 lanes/clk/SM XU pipe.  Measured on B200
//                   (nms_phasor_selftest): max error 4.3e-7, rms 1.2e-7; the cosine has a MEAN error of +1.2758e-8 (the
//                   sine none), i.e. a constant term e_0 in the phasor that adds e_0 * sum_j w_j to every amplitude (0.2 on
//                   C5's nuclear amplitude).  It is below half an ulp of cos near 1, so it cannot be taken out of the fp32
//                   phasor; subtracting e_0 * (tile weight sums) from the fp64 tile sums at the flush was tried in round 2:
//                   16 % fewer signed-kind misses on the full C5 map (292 -> 246 of 84 976) for 1.5 % of the throughput --
//                   not kept; the polynomial phasor has no such term.  The error is the MUFU tables' own: feeding the
//                   unit a phase whose conversion is exact and rotating by the exactly known remainder (first order)
//                   left max 3.5e-7 / rms 1e-7 unchanged (round-2 experiment).
//   phasor_poly(k)  FMA + ALU pipes: residual from the nearest quarter cycle as ONE shift (k << 2 wraps to
//                   2^34 (f - n/4)), I2FP, x = 2 pi (f - n/4) with 2 pi split into fl32 hi + lo (a single fl32
//                   constant is 2.8e-8 off: a sawtooth phase error that leaks A(-3q), A(5q) into A(q) at 7e-9),
//                   minimax sin (degree 7) and cos (degree 8) on [-pi/4, pi/4] (approximation errors 1.8e-9, 1e-10),
//                   quadrant swap and signs from the top two bits.  Emulated in fp32: max error 8.3e-8, rms 1.8e-8 per
//                   component, every Fourier component of the error function below 5e-10.
//                   19 issue slots, none on the XU pipe.  (Evaluating the same polynomials in fp64 on the FP64 pipe,
//                   idle at 6 % in the accurate recurrence kernel, was measured SLOWER: C5 0.567 -> 0.525 with the step
//                   phasor alone in fp64, 0.483 with both; mixing three-term steps into the rotations gained nothing.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace nms {

typedef unsigned long long u64;

constexpr double MAGIC = 1572864.0;                 // 1.5 * 2^20: ulp = 2^-32 (needs |t| < 2^19 cycles)
constexpr double INV_2PI = 0.15915494309189533577;

__device__ __forceinline__ u64 pack2(float lo, float hi)
{
    u64 d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ void unpack2(u64 v, float& lo, float& hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}

// {cos, sin}(2 pi k / 2^32) on the XU pipe.  (sin.approx / cos.approx multiply x by fl(1 / 2 pi) again -- FMUL.RZ,
// then MUFU on cycles; PTX offers no entry point that skips it.)
__device__ __forceinline__ void sincos_mufu(int k, float& co, float& so)
{
    const float TWO_PI_2M32 = 0x1.921fb6p-30f;   // fl(2 pi) * 2^-32
    const float x = __int2float_rn(k) * TWO_PI_2M32;
    co = __cosf(x);
    so = __sinf(x);
}

// {cos, sin}(2 pi k / 2^32) on the FMA and ALU pipes, to fp32 rounding accuracy.
__device__ __forceinline__ void sincos_poly(int k, float& co, float& so)
{
    const float C_HI = 0x1.921fb6p-32f;          // fl32(2 pi) * 2^-34
    const float C_LO = -0x1.777a5cp-57f;         // (2 pi - fl32(2 pi)) * 2^-34
    const float rf = __int2float_rn(k << 2);     // 2^34 (f - n/4), n = rint(4 f): the shift drops n
    const float x = fmaf(rf, C_HI, rf * C_LO);   // 2 pi (f - n/4) in [-pi/4, pi/4)
    const float z = x * x;
    float s = fmaf(z, fmaf(z, -0x1.98da66p-13f, 0x1.1105b4p-7f), -0x1.555540p-3f);
    s = fmaf(x * z, s, x);                                              // sin x = x + x^3 (s1 + s2 z + s3 z^2)
    float c = fmaf(z, fmaf(z, 0x1.9a025ap-16f, -0x1.6c0c8cp-10f), 0x1.55554ap-5f);
    c = fmaf(z, fmaf(z, c, -0.5f), 1.0f);                               // cos x = 1 - z/2 + z^2 (c2 + c3 z + c4 z^2)
    // phi = x + n pi/2:  n = 0: (c, s);  1: (-s, c);  2: (-c, -s);  3: (s, -c)
    const unsigned q2 = (unsigned)k + 0x20000000u;                      // top two bits: n mod 4
    const unsigned q3 = (unsigned)k + 0x60000000u;                      // top two bits: (n + 1) mod 4
    const bool swap = (q2 & 0x40000000u) != 0u;
    const float cc = swap ? s : c, ss = swap ? c : s;
    co = __uint_as_float(__float_as_uint(cc) ^ (q3 & 0x80000000u));     // cos negative for n in {1, 2}
    so = __uint_as_float(__float_as_uint(ss) ^ (q2 & 0x80000000u));     // sin negative for n in {2, 3}
}

// The same for a phase known to lie within a quarter cycle of zero (|k| < 2^30; the step phasor of the line recurrence
// when d' r_max < 1/4): no quadrant logic, minimax sin (degree 11) and cos (degree 10) on [-pi/2, pi/2] (approximation
// errors 1.7e-11 and 3.9e-10).  15 issue slots.
__device__ __forceinline__ void sincos_poly_half(int k, float& co, float& so)
{
    const float C_HI = 0x1.921fb6p-30f;          // fl32(2 pi) * 2^-32
    const float C_LO = -0x1.777a5cp-55f;         // (2 pi - fl32(2 pi)) * 2^-32
    const float rf = __int2float_rn(k);
    const float x = fmaf(rf, C_HI, rf * C_LO);
    const float z = x * x;
    float s = fmaf(z, -0x1.99aedep-26f, 0x1.7167p-19f);
    s = fmaf(z, s, -0x1.a01782p-13f);
    s = fmaf(z, s, 0x1.11110ap-7f);
    s = fmaf(z, s, -0x1.555556p-3f);
    so = fmaf(x * z, s, x);
    float c = fmaf(z, -0x1.194102p-22f, 0x1.9f8f5ap-16f);
    c = fmaf(z, c, -0x1.6c149cp-10f);
    c = fmaf(z, c, 0x1.555550p-5f);
    co = fmaf(z, fmaf(z, c, -0.5f), 1.0f);
}

// m = fma(q', r, MAGIC) (or a sum rounded at the same place): the low word holds frac(t) * 2^32.  The phasor
// {cos, sin} comes back as one packed register pair (one complex accumulator update = one fma.rn.f32x2).
template <bool POLY>
__device__ __forceinline__ u64 phasor(double m)
{
    float c, s;
    if (POLY) sincos_poly(__double2loint(m), c, s);
    else sincos_mufu(__double2loint(m), c, s);
    return pack2(c, s);
}

}  // namespace nms
