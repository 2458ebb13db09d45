// ll_device.cuh — device-side arithmetic building blocks of libll_b200 (sm_100a only).
//
// Nothing here is shared with oracle/: the oracle evaluates sinl/cosl of radians in long double, this
// file reduces the phase in *quarter cycles* (the spline is set up on phase * 2/pi) with the
// round-to-integer magic constant and evaluates two short Horner polynomials on the FP64 pipe.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ll {

constexpr double kMagic = 6755399441055744.0;        // 1.5 * 2^52: (y + kMagic) - kMagic == rint(y), |y| < 2^51
constexpr double kTwoOverPi = 0x1.45f306dc9c883p-1;
constexpr double kPi = 3.14159265358979323846;
constexpr double kPio2_1 = 0x1.921fb54442d18p+0;     // pi/2 split in three doubles (Cody-Waite with FMA)
constexpr double kPio2_2 = 0x1.1a62633145c07p-54;
constexpr double kPio2_3 = -0x1.f1976b7ed8fbcp-110;
constexpr double kSixth = 0x1.5555555555555p-3;

// sin(pi r/2) = r * S(r^2), cos(pi r/2) = C(r^2), |r| <= 1/2.  S and C are degree-5 polynomials in r^2
// interpolated at the Chebyshev nodes of [0, 1/4] (gen_sincos_coeffs.py; max error 3.4e-15 (sin), 5.6e-14 (cos)).
// That is far below the rounding of the argument itself (a phase of 1e6-1e7 quarter cycles carries 1e-10-1e-9 of
// absolute error in FP64) and 20x below what the 1e-6 bar on log L needs at <d|h> = 1e6; one more term each would
// cost two FP64 issue slots per bin for nothing measurable.  The coefficients live in constant memory so that every
// Horner step is one DFMA with a constant-bank operand (no UMOV/IMAD.MOV literal rebuilds inside the hot loop).
__constant__ double kSinC[6] = {0x1.921fb54442cfap+0, -0x1.4abbce6257a2ap-1, 0x1.466bc67123fa1p-4,
                                -0x1.32d2c644adc0bp-8, 0x1.5071ce4b47930p-13, -0x1.dd54805f3f706p-19};
__constant__ double kCosC[6] = {0x1.ffffffffffe0bp-1, -0x1.3bd3cc9bd2c35p+0, 0x1.03c1f074ded21p-2,
                                -0x1.55d3ba300cd50p-6, 0x1.e1e7ccccb387ap-11, -0x1.a0ee132c60c1fp-16};

__device__ __forceinline__ void sincos_poly_qc(double r, double &s, double &c)
{
    const double r2 = r * r;
    double ps = fma(kSinC[5], r2, kSinC[4]);
    double pc = fma(kCosC[5], r2, kCosC[4]);
    ps = fma(ps, r2, kSinC[3]);
    pc = fma(pc, r2, kCosC[3]);
    ps = fma(ps, r2, kSinC[2]);
    pc = fma(pc, r2, kCosC[2]);
    ps = fma(ps, r2, kSinC[1]);
    pc = fma(pc, r2, kCosC[1]);
    ps = fma(ps, r2, kSinC[0]);
    pc = fma(pc, r2, kCosC[0]);
    s = ps * r;
    c = pc;
}

// The same functions to the rounding of the arithmetic (degree 7 in r^2: max error 3.4e-17 (sin), 1.5e-17 (cos), and
// C(0) = 1 exactly), for the few evaluations per re-synchronisation of the rotation recurrence whose error is
// AMPLIFIED: a phase error delta in the per-bin rotation w = e^{i D1 Psi} becomes k delta in z after k bins, and
// because D1 Psi drifts slowly the degree-5 polynomial's error (5.6e-14 in cos) has the same sign over thousands of
// consecutive blocks — it was what made the distance from the oracle grow like the re-sync length squared.
__constant__ double kSinA[8] = {0x1.921fb54442d18p+0, -0x1.4abbce625be53p-1, 0x1.466bc6775aad9p-4, -0x1.32d2cce62ac22p-8,
                                0x1.50783485cbd83p-13, -0x1.e3074b4ff3058p-19, 0x1.e8eed12ee00a3p-25, -0x1.6c5b875d4e739p-31};
__constant__ double kCosA[8] = {0x1.0000000000000p+0, -0x1.3bd3cc9be45dep+0, 0x1.03c1f081b5aacp-2, -0x1.55d3c7e3c90f8p-6,
                                0x1.e1f5068355e15p-11, -0x1.a6d1ec7906c20p-16, 0x1.f9cc41140bb60p-22, -0x1.b264ba152378ap-28};
__device__ __forceinline__ void sincos_poly_qc_acc(double r, double &s, double &c)
{
    const double r2 = r * r;
    double ps = fma(kSinA[7], r2, kSinA[6]);
    double pc = fma(kCosA[7], r2, kCosA[6]);
#pragma unroll
    for (int k = 5; k >= 0; --k) {
        ps = fma(ps, r2, kSinA[k]);
        pc = fma(pc, r2, kCosA[k]);
    }
    s = ps * r;
    c = pc;
}

// quadrant bookkeeping: angle = (pi/2)(n + r); q = n mod 4.  Integer-pipe only (selects and sign-bit XORs on
// the high words), so it costs no FP64 issue slot.
__device__ __forceinline__ double flip_sign_if(double x, unsigned mask /* 0 or 0x80000000 */)
{
    return __hiloint2double(__double2hiint(x) ^ (int)mask, __double2loint(x));
}
__device__ __forceinline__ void quadrant_fix(int q, double s, double c, double &sn, double &cs)
{
    const bool sw = q & 1;
    const double a = sw ? c : s;
    const double b = sw ? s : c;
    sn = flip_sign_if(a, ((unsigned)q << 30) & 0x80000000u);
    cs = flip_sign_if(b, ((unsigned)(q + 1) << 30) & 0x80000000u);
}
// as quadrant_fix, but returns e = amp * (cos, sin) with the signs folded into amp and the swap
__device__ __forceinline__ void quadrant_apply(int q, double amp, double s, double c, double &u, double &v)
{
    // sn = sg * a, cs = sg * (sw ? -s : c), sg = (q & 2) ? -1 : 1, a = sw ? c : s
    const bool sw = q & 1;
    const double a = sw ? c : s;
    // b = sw ? -s : c, written on the words so that the negation folds into the select of the high word
    const float bh = sw ? -__int_as_float(__double2hiint(s)) : __int_as_float(__double2hiint(c));
    const double b = __hiloint2double(__float_as_int(bh), sw ? __double2loint(s) : __double2loint(c));
    const double as = flip_sign_if(amp, ((unsigned)q << 30) & 0x80000000u);
    u = as * b;
    v = as * a;
}

// sin and cos of an angle given in quarter cycles (y = angle * 2/pi).
__device__ __forceinline__ void sincos_qc(double y, double &sn, double &cs)
{
    const double sh = __dadd_rn(y, kMagic);
    const int q = __double2loint(sh);
    const double nd = __dadd_rn(sh, -kMagic);
    const double r = __dadd_rn(y, -nd);
    double s, c;
    sincos_poly_qc(r, s, c);
    quadrant_fix(q, s, c, sn, cs);
}
// the same with the degree-7 polynomials (re-synchronisation of the rotation recurrence)
__device__ __forceinline__ void sincos_qc_acc(double y, double &sn, double &cs)
{
    const double sh = __dadd_rn(y, kMagic);
    const int q = __double2loint(sh);
    const double nd = __dadd_rn(sh, -kMagic);
    const double r = __dadd_rn(y, -nd);
    double s, c;
    sincos_poly_qc_acc(r, s, c);
    quadrant_fix(q, s, c, sn, cs);
}
// u - i v = amp * exp(-i (pi/2) y)
__device__ __forceinline__ void amp_expi_qc(double amp, double y, double &u, double &v)
{
    const double sh = __dadd_rn(y, kMagic);
    const int q = __double2loint(sh);
    const double nd = __dadd_rn(sh, -kMagic);
    const double r = __dadd_rn(y, -nd);
    double s, c;
    sincos_poly_qc(r, s, c);
    quadrant_apply(q, amp, s, c, u, v);
}

// ---- FP32-accumulate variant (reading R15) --------------------------------------------------------
// sin x = x + x^3 S1(x^2), cos x = 1 - x^2/2 + x^4 C2(x^2), |x| <= pi/4, binary32.  The leading terms are exact
// in binary and the remaining coefficients were fitted after rounding their predecessors
// (gen_sincos_coeffs.py: max polynomial error 7.0e-11 (sin), 1.1e-10 (cos)), so the only error left at the
// 1e-8 level is the evaluation rounding, which is incoherent from bin to bin.
__device__ __forceinline__ void sincos_poly_f32(float x, float &s, float &c)
{
    const float x2 = x * x;
    float ps = fmaf(0x1.7658e0p-19f, x2, -0x1.a0423ap-13f);
    float pc = fmaf(0x1.99ead0p-16f, x2, -0x1.6c0c2ep-10f);
    ps = fmaf(ps, x2, 0x1.11115ep-7f);
    pc = fmaf(pc, x2, 0x1.55554ap-5f);
    ps = fmaf(ps, x2, -0x1.555556p-3f);
    pc = fmaf(pc, x2, -0.5f);
    s = fmaf(x * x2, ps, x);
    c = fmaf(pc, x2, 1.0f);
}
__device__ __forceinline__ float flip_sign_if_f32(float x, unsigned mask /* 0 or 0x80000000 */)
{
    return __uint_as_float(__float_as_uint(x) ^ mask);
}
// u - i v = amp * exp(-i (pi/2) y): the phase y (quarter cycles) is reduced to [-1/2, 1/2] in FP64, scaled to
// radians in FP64 (so that the pi/2 factor is not rounded to binary32), then everything else is binary32.
__device__ __forceinline__ void amp_expi_qc_f32(float amp, double y, float &u, float &v)
{
    const double sh = __dadd_rn(y, kMagic);
    const int q = __double2loint(sh);
    const double nd = __dadd_rn(sh, -kMagic);
    const double r = __dadd_rn(y, -nd);
    const float x = __double2float_rn(r * kPio2_1);
    float s, c;
    sincos_poly_f32(x, s, c);
    const bool sw = q & 1;
    const float a = sw ? c : s;
    const float b = sw ? -s : c;
    const float as = flip_sign_if_f32(amp, ((unsigned)q << 30) & 0x80000000u);
    u = as * b;
    v = as * a;
}

// packed binary32 pairs (sm_100 f32x2 instructions: one instruction for two bins' worth of FMA)
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
// both lanes: sin x = x + x^3 S1(x^2), cos x = 1 - x^2/2 + x^4 C2(x^2)   (same coefficients as sincos_poly_f32)
__device__ __forceinline__ void sincos_poly_f32x2(f32x2 x, f32x2 &s, f32x2 &c)
{
    const f32x2 x2 = mul2(x, x);
    f32x2 ps = fma2(pack2(0x1.7658e0p-19f, 0x1.7658e0p-19f), x2, pack2(-0x1.a0423ap-13f, -0x1.a0423ap-13f));
    f32x2 pc = fma2(pack2(0x1.99ead0p-16f, 0x1.99ead0p-16f), x2, pack2(-0x1.6c0c2ep-10f, -0x1.6c0c2ep-10f));
    ps = fma2(ps, x2, pack2(0x1.11115ep-7f, 0x1.11115ep-7f));
    pc = fma2(pc, x2, pack2(0x1.55554ap-5f, 0x1.55554ap-5f));
    ps = fma2(ps, x2, pack2(-0x1.555556p-3f, -0x1.555556p-3f));
    pc = fma2(pc, x2, pack2(-0.5f, -0.5f));
    s = fma2(mul2(x, x2), ps, x);
    c = fma2(pc, x2, pack2(1.0f, 1.0f));
}
// FP64 part of amp_expi_qc_f32: quadrant number and reduced angle in radians (binary32)
__device__ __forceinline__ float reduce_qc_to_rad_f32(double y, int &q)
{
    const double sh = __dadd_rn(y, kMagic);
    q = __double2loint(sh);
    const double nd = __dadd_rn(sh, -kMagic);
    const double r = __dadd_rn(y, -nd);
    return __double2float_rn(r * kPio2_1);
}
// quadrant bookkeeping on binary32: amp e^{-i angle} = u - i v with u = as * b, v = as * a
__device__ __forceinline__ void quadrant_f32(int q, float amp, float s, float c, float &as, float &a, float &b)
{
    const bool sw = q & 1;
    a = sw ? c : s;
    b = sw ? -s : c;
    as = flip_sign_if_f32(amp, ((unsigned)q << 30) & 0x80000000u);
}

// sin and cos of an angle in radians, accurate for |x| up to ~1e9 (three-term Cody-Waite with FMA; the
// reduced argument is then handed to the quarter-cycle polynomials).
__device__ __forceinline__ void sincos_rad(double x, double &sn, double &cs)
{
    const double sh = __dadd_rn(x * kTwoOverPi, kMagic);
    const int q = __double2loint(sh);
    const double nd = __dadd_rn(sh, -kMagic);
    double r = fma(-nd, kPio2_1, x);
    r = fma(-nd, kPio2_2, r);
    r = fma(-nd, kPio2_3, r);
    double s, c;
    sincos_poly_qc(r * kTwoOverPi, s, c);
    quadrant_fix(q, s, c, sn, cs);
}

// taper(x) = 1 (x <= 1); s^3 (10 - 15 s + 6 s^2), s = (1 + kappa - x)/kappa (1 < x < 1 + kappa); 0 beyond.
// (reading R9; BASELINE.json "tapered to zero above f_ISCO")
__device__ __forceinline__ double taper(double x, double kappa, double inv_kappa)
{
    if (x <= 1.0) return 1.0;
    if (x >= 1.0 + kappa) return 0.0;
    const double s = (1.0 + kappa - x) * inv_kappa;
    return s * s * s * fma(s, fma(6.0, s, -15.0), 10.0);
}

// the same function without branches: s clamped to [0, 1] gives exactly 1 at s = 1 (1 * (6 - 15 + 10)) and 0 at s = 0
__device__ __forceinline__ double taper_nobranch(double x, double kappa, double inv_kappa)
{
    const double s = fmin(fmax((1.0 + kappa - x) * inv_kappa, 0.0), 1.0);
    return s * s * s * fma(s, fma(6.0, s, -15.0), 10.0);
}

// frequency of dense bin i, exactly as the grid is defined (reading R3): f_i = (double)(k_min + i) * df
__host__ __device__ __forceinline__ double bin_freq(long long k_min, long long i, double df)
{
    return (double)(k_min + i) * df;
}

// smallest i in [0, n_f] with f_i >= f  (n_f if none)
__host__ __device__ inline long long first_bin_ge(double f, long long k_min, long long n_f, double df)
{
    double est = ceil(f / df) - (double)k_min;
    if (!(est > 0.0)) est = 0.0;
    if (est > (double)n_f) est = (double)n_f;
    long long i = (long long)est;
    while (i > 0 && bin_freq(k_min, i - 1, df) >= f) --i;
    while (i < n_f && bin_freq(k_min, i, df) < f) ++i;
    return i;
}

// smallest i in [0, n_f] with f_i > f  (n_f if none)
__host__ __device__ inline long long first_bin_gt(double f, long long k_min, long long n_f, double df)
{
    double est = floor(f / df) + 1.0 - (double)k_min;
    if (!(est > 0.0)) est = 0.0;
    if (est > (double)n_f) est = (double)n_f;
    long long i = (long long)est;
    while (i > 0 && bin_freq(k_min, i - 1, df) > f) --i;
    while (i < n_f && bin_freq(k_min, i, df) <= f) ++i;
    return i;
}

// ---------------------------------------------------------------------------------------------------
// mbarrier + 1-D bulk TMA (cp.async.bulk) helpers; SASS: SYNCS.* / UBLKCP.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!done);
}
__device__ __forceinline__ void tma_load_1d(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

} // namespace ll
