// rad_device.cuh -- device-side building blocks of the sm_100a radiation-integral kernels.
//
// Error-free transforms (double-double), the turn-based sincos, 1-D TMA bulk copies with
// mbarrier completion, and the packed trajectory layout.  CUDA path only; the CPU oracle
// shares nothing with this file.
#pragma once

#include <cstdint>
#include <cuda_runtime.h>

#include "sincos_coeffs.h"

namespace rad {

// ------------------------------------------------------------------ packed layout (HBM + smem)
// The pack kernel rewrites the caller's 11 SoA arrays into chunk records that one TMA
// bulk copy brings into shared memory.  One chunk = header + CH sample records.
//
// header (HDR doubles): [0] P0_b hi  [1] P0_b lo   P0 = t/(2 gamma^2) - dz   (double-double)
//                       [2] t_b      [3] x_b       [4] y_b     (base sample of the chunk)
//                       [5] gamma[0] of the trajectory        [6..7] pad
// sample (REC doubles): [0] D0 = 1/(2 gamma^2) - dvz    [1] vx   [2] vy
//                       [3] w*ax  [4] w*ay  [5] w*az    (w = trapezoid weight)
//                       [6] P0_k - P0_b   [7] t_k - t_b   [8] x_k - x_b   [9] y_k - y_b
// Padding samples of a trajectory's last chunk have D0 = 1 and zeros elsewhere: they
// contribute exactly 0.
constexpr int CH = 128;
constexpr int REC = 10;
constexpr int HDR = 8;
constexpr int CHUNK_DBL = HDR + CH * REC;
constexpr int CHUNK_BYTES = CHUNK_DBL * 8;
static_assert(CHUNK_BYTES % 16 == 0, "TMA bulk copies move multiples of 16 bytes");

// ------------------------------------------------------------------ double-double helpers
struct dd { double hi, lo; };

__device__ __forceinline__ dd two_sum(double a, double b) {
    double s = a + b;
    double bb = s - a;
    double e = (a - (s - bb)) + (b - bb);
    return {s, e};
}
__device__ __forceinline__ dd fast_two_sum(double a, double b) {   // |a| >= |b|
    double s = a + b;
    return {s, b - (s - a)};
}
__device__ __forceinline__ dd two_prod(double a, double b) {
    double p = a * b;
    return {p, fma(a, b, -p)};
}
__device__ __forceinline__ dd dd_add(dd a, dd b) {
    dd s = two_sum(a.hi, b.hi);
    return fast_two_sum(s.hi, s.lo + (a.lo + b.lo));
}
__device__ __forceinline__ dd dd_neg(dd a) { return {-a.hi, -a.lo}; }
__device__ __forceinline__ dd dd_mul_d(dd a, double b) {
    dd p = two_prod(a.hi, b);
    return fast_two_sum(p.hi, fma(a.lo, b, p.lo));
}
__device__ __forceinline__ dd dd_mul(dd a, dd b) {
    dd p = two_prod(a.hi, b.hi);
    return fast_two_sum(p.hi, fma(a.hi, b.lo, fma(a.lo, b.hi, p.lo)));
}
// a / b with b a double-double, a a double: one Newton correction on the IEEE quotient.
__device__ __forceinline__ dd d_div_dd(double a, dd b) {
    double q = a / b.hi;
    double r = fma(-q, b.hi, a);      // exact residual of the leading quotient
    r = fma(-q, b.lo, r);
    return fast_two_sum(q, r / b.hi);
}

// 1/(2 pi) as a double-double
constexpr double INV_2PI_HI = 0x1.45f306dc9c883p-3;
constexpr double INV_2PI_LO = -0x1.6b01ec5417056p-57;

// fractional part (nearest-integer sense, result in [-1/2, 1/2]) of a double-double
__device__ __forceinline__ double dd_frac(dd a) {
    const double M52 = 6755399441055744.0;           // 1.5 * 2^52
    double k = (a.hi + M52) - M52;                   // rint for |a.hi| < 2^51
    return (a.hi - k) + a.lo;
}

// ------------------------------------------------------------------ phasor of a phase in turns
// For |p| < 2^50 turns returns  c = cos(2 pi p)  and  s = sin(2 pi p) / sqrt(2).
// Reduction is exact: k = rint(p) (cvt.rni.f64.f64 = FRND.F64, which does not occupy the FP64 pipe;
// measured +2.4 % / +4.9 % evals/s over the magic-number add it replaced), r = p - k in [-1/2, 1/2].
// Then a = sqrt(2) sin(pi r/2) and b = 2 cos(pi r/2) by two Horner polynomials in r^2, and two
// angle doublings written so that every step is one FP64 instruction:
//     cos(pi r) = 1 - a^2            sqrt(2) sin(pi r) = a b =: S2
//     cos(2 pi r) = 1 - S2^2         sin(2 pi r)/sqrt(2) = S2 cos(pi r)
// No quadrant logic, no selects, no integer instructions: on B200 an ALU instruction issued
// between DFMAs costs FP64 issue time, so the four extra FP64
// instructions are cheaper than the ~10 integer ones of a swap/sign scheme.  The 1/sqrt(2)
// on the sine is carried by the imaginary accumulators and undone in the epilogue.
// Coefficients live in constant memory so that every Horner step is one DFMA with a
// constant-bank operand (no UMOV / MOV to materialise 64-bit immediates in the loop).
__constant__ double SC_S6[7] = RAD_SC_HI_S;
__constant__ double SC_C6[7] = RAD_SC_HI_C;
__constant__ double SC_S5[6] = RAD_SC_LO_S;
__constant__ double SC_C5[6] = RAD_SC_LO_C;

template <int DEG>
__device__ __forceinline__ void sincos_poly(double z, double &ps, double &pc);
template <>
__device__ __forceinline__ void sincos_poly<6>(double z, double &ps, double &pc) {
    ps = SC_S6[6]; pc = SC_C6[6];
#pragma unroll
    for (int i = 5; i >= 0; --i) { ps = fma(ps, z, SC_S6[i]); pc = fma(pc, z, SC_C6[i]); }
}
template <>
__device__ __forceinline__ void sincos_poly<5>(double z, double &ps, double &pc) {
    ps = SC_S5[5]; pc = SC_C5[5];
#pragma unroll
    for (int i = 4; i >= 0; --i) { ps = fma(ps, z, SC_S5[i]); pc = fma(pc, z, SC_C5[i]); }
}
template <int DEG>
__device__ __forceinline__ void phasor_turns(double p, double &c_out, double &s_out) {
#ifndef RAD_MAGIC_REDUCTION
    const double r = p - rint(p);                    // FRND.F64 runs beside the FP64 pipe; the subtraction is exact
#else
    const double M52 = 6755399441055744.0;           // 1.5 * 2^52: ulp = 1 (two more FP64-pipe instructions)
    const double kq = p + M52;
    const double r = p - (kq - M52);
#endif
    double ps, pc;
    sincos_poly<DEG>(r * r, ps, pc);
    const double a = r * ps;
    const double c2 = fma(-a, a, 1.0);
    const double s2 = a * pc;
    c_out = fma(-s2, s2, 1.0);
    s_out = s2 * c2;
}

// 1/(x*x) for x > 0: hardware seed (2^-23) + one cubic step (-> 2^-69) on x^2.
__device__ __forceinline__ double inv_square(double x) {
    double x2 = x * x;
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x2));
    double e = fma(-x2, y, 1.0);
    double e2 = fma(e, e, e);
    return fma(y, e2, y);
}

// ------------------------------------------------------------------ TMA (1-D bulk) + mbarrier
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t phase) {
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(phase)
            : "memory");
    } while (!done);
}
// global -> shared bulk copy (SASS: UBLKCP), completion counted in bytes on `bar`
__device__ __forceinline__ void tma_load_1d(void *dst_smem, const void *src_gmem, uint32_t bytes,
                                            uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(dst_smem)),
        "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

}  // namespace rad
