// sc_math.cuh — fp64 building blocks of the march kernel (sm_100a).
//
// The march is bound by the FP64 pipe, so every transcendental is written out as a short
// DFMA sequence seeded by the MUFU approximations (MUFU.RCP64H / MUFU.RSQ64H, reached through
// rcp.approx.ftz.f64 / rsqrt.approx.ftz.f64) instead of the IEEE-rounded library routines:
//   reciprocal        1 MUFU + 3 DFMA   (cubic Newton step)
//   rsqrt             1 MUFU + 5 FP64
//   exp / expm1       range reduction by ln2 + degree-13 polynomial, 2^k by exponent arithmetic
//   sin / cos         |y| <= pi/4 polynomial kernels (the arguments are 2*l*Im(Omega) << 1); library
//                     sincos on the rare warp that exceeds it
// Accuracy (measured by sc_debug_math, tests/test_gpu_parity.py): <= 4 ulp each.
#pragma once
#include <cuda_runtime.h>

namespace scm {

// polynomial coefficients live in constant memory so that the DFMAs take them as c[bank][offset] operands
// instead of re-materialising 64-bit immediates with two UMOVs each
__constant__ double kExp[12] = {1.6059043836821613e-10, 2.08767569878681e-09, 2.505210838544172e-08, 2.755731922398589e-07,
                                2.7557319223985893e-06, 2.48015873015873e-05, 1.984126984126984e-04, 1.388888888888889e-03,
                                8.333333333333333e-03, 4.1666666666666664e-02, 1.6666666666666666e-01, 0.5};   // 1/13! .. 1/2!
__constant__ double kSin[6] = {1.58969099521155010221e-10, -2.50507602534068634195e-08, 2.75573137070700676789e-06,
                               -1.98412698298579493134e-04, 8.33333333332248946124e-03, -1.66666666666666324348e-01};
__constant__ double kCos[6] = {-1.13596475577881948265e-11, 2.08757232129817482790e-09, -2.75573143513906633035e-07,
                               2.48015872894767294178e-05, -1.38888888888741095749e-03, 4.16666666666666019037e-02};
__constant__ double kRed[4] = {1.4426950408889634074, 6.93147180369123816490e-01, 1.90821492927058770002e-10, 6755399441055744.0};

struct cplx { double re, im; };

__device__ __forceinline__ cplx mk(double a, double b) { cplx r; r.re = a; r.im = b; return r; }

__device__ __forceinline__ double rcp_nr(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
#ifdef SC_MATH_EXTRA_NEWTON
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
#endif
    const double t = fma(e, e, e);
    return fma(y, t, y);
}

__device__ __forceinline__ double rsqrt_nr(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
#ifdef SC_MATH_EXTRA_NEWTON
    {
        const double t0 = x * y;
        const double e0 = fma(-t0, y, 1.0);
        y = fma(0.5 * y, e0, y);
    }
#endif
    const double t = x * y;
    const double e = fma(-t, y, 1.0);          // 1 - x y^2
    const double p = fma(0.375, e, 0.5);       // y (1 + e/2 + 3 e^2/8)
    const double ye = y * e;
    return fma(ye, p, y);
}

// ex = exp(x), xm1 = exp(x) - 1 without cancellation, for x <= ~0 (any x > -700 works; x <= -700 -> 0, -1)
__device__ __forceinline__ void exp_pair(double x, double& ex, double& xm1) {
    const double L2E = kRed[0], LN2_HI = kRed[1], LN2_LO = kRed[2], MAGIC = kRed[3];   // MAGIC = 1.5 * 2^52
    x = fmax(x, -700.0);
    double kf = fma(x, L2E, MAGIC);
    const int k = __double2loint(kf);
    kf -= MAGIC;
    double r = fma(-kf, LN2_HI, x);
    r = fma(-kf, LN2_LO, r);
    // expm1(r) = r + r^2 (1/2 + r/6 + ... + r^11/13!), |r| <= ln2/2: truncation < 5e-18
    double p = kExp[0];
#pragma unroll
    for (int i = 1; i < 12; ++i) p = fma(p, r, kExp[i]);
    const double r2 = r * r;
    p = fma(p, r2, r);                                  // expm1(r)
    const double s = __hiloint2double((k + 1023) << 20, 0);   // 2^k, k in [-1010, 0]
    xm1 = fma(s, p, s - 1.0);
    ex = fma(s, p, s);
}

// s = sin(y), cm1 = cos(y) - 1 for |y| <= pi/4 (minimax kernels of the classic fdlibm k_sin/k_cos)
__device__ __forceinline__ void sincos_small(double y, double& s, double& cm1) {
    const double z = y * y;
    double ps = kSin[0], pc = kCos[0];
#pragma unroll
    for (int i = 1; i < 6; ++i) { ps = fma(ps, z, kSin[i]); pc = fma(pc, z, kCos[i]); }
    s = fma(y * z, ps, y);
    cm1 = fma(z * z, pc, -0.5 * z);
}

// Principal square root Omega of w (Re Omega >= 0) and rq = 1/|Omega|^2 (so that 1/Omega = conj(Omega) rq).
__device__ __forceinline__ void csqrt_inv(double wr, double wi, double& sr, double& si, double& rq) {
    const double q = fma(wr, wr, wi * wi);
    rq = rsqrt_nr(q);                  // 1/|w| = 1/|Omega|^2
    const double m = q * rq;           // |w|
    const double p = 0.5 * (m + fabs(wr));
    const double rp = rsqrt_nr(p);
    const double a = p * rp;           // sqrt(p)
    const double b = 0.5 * fabs(wi) * rp;
    sr = wr >= 0.0 ? a : b;
    si = copysign(wr >= 0.0 ? b : a, wi);
}

// Step coefficient T = tanh(Omega l)/Omega, Omega = sqrt(|De|^2 - z^2): the closed-form step
// of PAPER.md:982 is the Moebius map gamma' = [gamma + iT(z gamma + De)] / [1 - iT(z + conj(De) gamma)].
// T depends on De only through |De|^2, so gamma (De) and gamma-tilde (-conj De) share it.
__device__ __forceinline__ cplx coef_T(double d2, double zr, double zi, double len) {
    const double wr = fma(zi, zi, fma(-zr, zr, d2));
    const double wi = -2.0 * zr * zi;
    double sr, si, rq;
    csqrt_inv(wr, wi, sr, si, rq);
    const double m2l = -2.0 * len;
    const double x = m2l * sr, y = m2l * si;
    double ex, xm1, s, cm1;
    exp_pair(x, ex, xm1);
    if (__any_sync(0xffffffffu, fabs(y) > 0.78539816339744830962)) {
        double cc;
        sincos(y, &s, &cc);
        cm1 = cc - 1.0;
    } else {
        sincos_small(y, s, cm1);
    }
    // E - 1 = (e^x - 1) cos y + (cos y - 1) + i e^x sin y
    const double er = fma(xm1, cm1, xm1) + cm1;
    const double ei = ex * s;
    const double fr = 2.0 + er;                         // 1 + E
    const double rf = rcp_nr(fma(fr, fr, ei * ei));
    // tanh(Omega l) = -(E-1)/(E+1) = -(E-1) conj(E+1) / |E+1|^2
    const double tr = -fma(er, fr, ei * ei) * rf;
    const double ti = fma(er, ei, -ei * fr) * rf;
    const double ir = sr * rq, ii = -si * rq;           // 1/Omega
    return mk(fma(tr, ir, -ti * ii), fma(tr, ii, ti * ir));
}

// One closed-form step given T: 27 fp64 instructions + 1 MUFU.
__device__ __forceinline__ cplx step_T(cplx g, double Dr, double Di, double zr, double zi, cplx T) {
    const double ur = fma(zr, g.re, fma(-zi, g.im, Dr));        // u = z g + De
    const double ui = fma(zr, g.im, fma(zi, g.re, Di));
    const double Nr = fma(-T.re, ui, fma(-T.im, ur, g.re));     // N = g + i T u
    const double Ni = fma(T.re, ur, fma(-T.im, ui, g.im));
    const double vr = fma(Dr, g.re, fma(Di, g.im, zr));         // v = z + conj(De) g
    const double vi = fma(Dr, g.im, fma(-Di, g.re, zi));
    const double Qr = fma(T.re, vi, fma(T.im, vr, 1.0));        // Q = 1 - i T v
    const double Qi = fma(-T.re, vr, T.im * vi);
    const double rq = rcp_nr(fma(Qr, Qr, Qi * Qi));
    return mk(fma(Nr, Qr, Ni * Qi) * rq, fma(Ni, Qr, -Nr * Qi) * rq);
}

// Local homogeneous solution gamma_h = -De/(z + i Omega) (start values, boundary reset): rare, library math.
__device__ __forceinline__ cplx gamma_hom(double Dr, double Di, double zr, double zi) {
    const double wr = Dr * Dr + Di * Di - (zr * zr - zi * zi), wi = -2.0 * zr * zi;
    const double m = hypot(wr, wi);
    double sr, si;
    if (wr >= 0.0) { sr = sqrt(0.5 * (m + wr)); si = wi / (2.0 * sr); }
    else { const double a = sqrt(0.5 * (m - wr)); sr = fabs(wi) / (2.0 * a); si = copysign(a, wi); }
    const double br = zr - si, bi = zi + sr;              // z + i Omega
    const double d = br * br + bi * bi;
    return mk(-(Dr * br + Di * bi) / d, -(Di * br - Dr * bi) / d);
}

}  // namespace scm
