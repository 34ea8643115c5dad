// sc_math.cuh — arithmetic building blocks of the march kernel (sm_100a), fp64 and fp32.
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
// The optional FP32 mode (opts.precision = 32) uses the same formulas on float: MUFU.RCP / MUFU.RSQ directly
// (1-2 ulp), degree-7 expm1 and degree-4 sin/cos kernels.  Everything above the primitives is one template.
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

template <typename R> struct cplx_t { R re, im; };
using cplx = cplx_t<double>;
using cplxf = cplx_t<float>;

template <typename R>
__device__ __forceinline__ cplx_t<R> mk(R a, R b) { cplx_t<R> r; r.re = a; r.im = b; return r; }

__device__ __forceinline__ double mad(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float mad(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double absr(double a) { return fabs(a); }
__device__ __forceinline__ float absr(float a) { return fabsf(a); }
__device__ __forceinline__ double cpsign(double a, double b) { return copysign(a, b); }
__device__ __forceinline__ float cpsign(float a, float b) { return copysignf(a, b); }
__device__ __forceinline__ double maxr(double a, double b) { return fmax(a, b); }
__device__ __forceinline__ float maxr(float a, float b) { return fmaxf(a, b); }

// ---------------------------------------------------------------------------------------------- fp64 primitives
__device__ __forceinline__ double rcp_nr(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    const double t = fma(e, e, e);
    return fma(y, t, y);
}

__device__ __forceinline__ double rsqrt_nr(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
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
__device__ __forceinline__ void sincos_lib(double y, double& s, double& cm1) { double c; sincos(y, &s, &c); cm1 = c - 1.0; }

// ---------------------------------------------------------------------------------------------- fp32 primitives
__device__ __forceinline__ float rcp_nr(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rsqrt_nr(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

__device__ __forceinline__ void exp_pair(float x, float& ex, float& xm1) {
    x = fmaxf(x, -80.0f);
    float kf = fmaf(x, 1.4426950408889634f, 12582912.0f);            // 1.5 * 2^23
    const int k = __float_as_int(kf) - 0x4B400000;
    kf -= 12582912.0f;
    float r = fmaf(-kf, 0.693145751953125f, x);
    r = fmaf(-kf, 1.42860682030941723212e-6f, r);
    // expm1(r) = r + r^2 (1/2 + r/6 + ... + r^5/7!), |r| <= ln2/2: truncation < 2e-8 relative
    float p = 1.9841270e-4f;
    p = fmaf(p, r, 1.3888889e-3f); p = fmaf(p, r, 8.3333333e-3f); p = fmaf(p, r, 4.1666667e-2f);
    p = fmaf(p, r, 1.6666667e-1f); p = fmaf(p, r, 0.5f);
    p = fmaf(p, r * r, r);
    const float s = __int_as_float((k + 127) << 23);                  // 2^k, k in [-116, 0]
    xm1 = fmaf(s, p, s - 1.0f);
    ex = fmaf(s, p, s);
}

__device__ __forceinline__ void sincos_small(float y, float& s, float& cm1) {
    const float z = y * y;
    float ps = 2.7183114939898219064e-6f, pc = 2.43904487962774090654e-5f;
    ps = fmaf(ps, z, -1.98393348360966317347e-4f); ps = fmaf(ps, z, 8.3333293858894631756e-3f); ps = fmaf(ps, z, -1.66666666416265235595e-1f);
    pc = fmaf(pc, z, -1.38867637746099294692e-3f); pc = fmaf(pc, z, 4.16666233237390631894e-2f);
    s = fmaf(y * z, ps, y);
    cm1 = fmaf(z * z, pc, -0.5f * z);
}
__device__ __forceinline__ void sincos_lib(float y, float& s, float& cm1) { float c; sincosf(y, &s, &c); cm1 = c - 1.0f; }

// ---------------------------------------------------------------------------------------------- the step
// Principal square root Omega of w (Re Omega >= 0) and rq = 1/|Omega|^2 (so that 1/Omega = conj(Omega) rq).
template <typename R>
__device__ __forceinline__ void csqrt_inv(R wr, R wi, R& sr, R& si, R& rq) {
    const R q = mad(wr, wr, wi * wi);
    rq = rsqrt_nr(q);                  // 1/|w| = 1/|Omega|^2
    const R m = q * rq;                // |w|
    const R p = R(0.5) * (m + absr(wr));
    const R rp = rsqrt_nr(p);
    const R a = p * rp;                // sqrt(p)
    const R b = R(0.5) * absr(wi) * rp;
    sr = wr >= R(0) ? a : b;
    si = cpsign(wr >= R(0) ? b : a, wi);
}

// Step coefficient T = tanh(Omega l)/Omega, Omega = sqrt(|De|^2 - z^2): the closed-form step
// of PAPER.md:982 is the Moebius map gamma' = [gamma + iT(z gamma + De)] / [1 - iT(z + conj(De) gamma)].
// T depends on De only through |De|^2, so gamma (De) and gamma-tilde (-conj De) share it.
template <typename R>
__device__ __forceinline__ cplx_t<R> coef_T(R d2, R zr, R zi, R len) {
    const R wr = mad(zi, zi, mad(-zr, zr, d2));
    const R wi = R(-2) * zr * zi;
    R sr, si, rq;
    csqrt_inv(wr, wi, sr, si, rq);
    const R m2l = R(-2) * len;
    const R x = m2l * sr, y = m2l * si;
    R ex, xm1, s, cm1;
    exp_pair(x, ex, xm1);
    if (__any_sync(0xffffffffu, absr(y) > R(0.78539816339744830962))) sincos_lib(y, s, cm1);
    else sincos_small(y, s, cm1);
    // E - 1 = (e^x - 1) cos y + (cos y - 1) + i e^x sin y
    const R er = mad(xm1, cm1, xm1) + cm1;
    const R ei = ex * s;
    const R fr = R(2) + er;                             // 1 + E
    const R rf = rcp_nr(mad(fr, fr, ei * ei));
    // tanh(Omega l) = -(E-1)/(E+1) = -(E-1) conj(E+1) / |E+1|^2
    const R tr = -mad(er, fr, ei * ei) * rf;
    const R ti = mad(er, ei, -ei * fr) * rf;
    const R ir = sr * rq, ii = -si * rq;                // 1/Omega
    return mk(mad(tr, ir, -ti * ii), mad(tr, ii, ti * ir));
}

// Out-of-line copy of the exp-based evaluation: the march's hot loop evaluates T by the Taylor table below and only
// calls this for the two end pieces of a trajectory and for pieces outside the table's radius.
template <typename R>
__device__ __noinline__ cplx_t<R> coef_T_slow(R d2, R zr, R zi, R len) { return coef_T(d2, zr, zi, len); }

// T as a function of w = Omega^2 is meromorphic: T(w) = tanh(l sqrt w)/sqrt w = sum_k (2/l)/(w + (2k+1)^2 wp),
// wp = (pi/2l)^2, poles on the negative real axis only.  For an energy z0 (Matsubara i*eps, or eps + i*delta) and a
// piece of the common length l = h with Doppler shift a,
//     w = |De|^2 - (z0 + a)^2 = w0 + dw,   w0 = -z0^2,   dw = (|De|^2 - a^2) - 2 z0 a,
// and |dw| is small against the distance from w0 to the nearest pole (eps^2 + wp on the imaginary axis; the ratio
// is at most |a| 2h/pi + |De|^2/wp at ANY Matsubara energy), so T is a short Taylor polynomial in dw whose
// coefficients c_k(z0) = T^(k)(w0)/k! the host tabulates per energy (sc_api.cu taylor_table).  On the imaginary
// axis w0 is real and the c_k are REAL (T is real on the real axis): a real-coefficient polynomial at a complex point
// costs 2 FMAs per term — divide by the real quadratic (x - dw)(x - conj dw) = x^2 - r x + s; the remainder
// b1 x + (b0 - r b1) at x = dw is (b0 - b1 Re dw) + i b1 Im dw.  Off the axis (sc_ldos) the c_k are complex: Horner.
// K and the radius fraction: truncation <= RMAX^(K+1) relative.  K = 5 at 0.01 of the radius bounds it by 1e-12; the
// bound is only approached at the highest energies (|dw| ~ 2 eps |a|), where one step already contracts a perturbation
// of gamma by e^{-2 eps h}; at the low energies that carry a long memory |dw|/radius ~ |De|^2/wp ~ 1e-4 and the
// truncation is below 1e-20.  The parity budget is 1e-9.
template <typename R> struct TaylorK;
template <> struct TaylorK<double> { static constexpr int K = 5; static constexpr double RMAX = 0.01; };                                // 0.01^6 = 1e-12
template <> struct TaylorK<float> { static constexpr int K = 3; static constexpr double RMAX = 0.012; };                                // 0.012^4 = 2e-8
template <typename R, int K>
__device__ __forceinline__ cplx_t<R> taylor_real(const R (&c)[K + 1], R dwr, R dwi, R s) {
    const R r = dwr + dwr;
    R b2 = c[K];
    R b1 = mad(r, b2, c[K - 1]);
#pragma unroll
    for (int k = K - 2; k >= 0; --k) {
        const R b0 = mad(r, b1, mad(-s, b2, c[k]));
        b2 = b1; b1 = b0;
    }
    return mk(mad(-b2, dwr, b1), b2 * dwi);              // here b1 holds b_0 and b2 holds b_1
}
// The same with the nearest pole taken out in closed form (energies on the imaginary axis only): the rest,
// R(w) = T(w) - (2/h)/(w + wp), converges out to the SECOND pole, |dw| < w0 + 9 wp — three times the reach in |a|:
//     T = (2/h)/(w0 + wp + dw) + sum_k r_k dw^k,   r_k real.
// Used by the rounds that spill T (strong vector potentials), where T is evaluated once per piece.
template <typename R> struct TaylorPoleK;
template <> struct TaylorPoleK<double> { static constexpr int K = 8; static constexpr double RMAX = 0.012; };   // 0.012^9 = 5e-18
template <> struct TaylorPoleK<float> { static constexpr int K = 4; static constexpr double RMAX = 0.03; };      // 0.03^5  = 2e-8
// ... and a short version of it for rounds that re-evaluate T in pass 2 but whose |a| is beyond the pole-free table
// (same truncation rule as TaylorK: RMAX^(K+1))
template <typename R> struct TaylorPoleShortK;
template <> struct TaylorPoleShortK<double> { static constexpr int K = 5; static constexpr double RMAX = 0.01; };   // 1e-12
template <> struct TaylorPoleShortK<float> { static constexpr int K = 3; static constexpr double RMAX = 0.012; };
template <typename R, int K>
__device__ __forceinline__ cplx_t<R> taylor_pole(const R (&c)[K + 1], R pole_a, R pole_res, R dwr, R dwi, R s) {
    const R r = dwr + dwr;
    R b2 = c[K];
    R b1 = mad(r, b2, c[K - 1]);
#pragma unroll
    for (int k = K - 2; k >= 0; --k) {
        const R b0 = mad(r, b1, mad(-s, b2, c[k]));
        b2 = b1; b1 = b0;
    }
    // here b1 holds b_0 and b2 holds b_1;  pole term: res / (A + dw) = res conj(A + dw) / |A + dw|^2
    const R pr = pole_a + dwr;
    const R q = pole_res * rcp_nr(mad(pr, pr, dwi * dwi));
    return mk(mad(pr, q, mad(-b2, dwr, b1)), mad(-dwi, q, b2 * dwi));
}
template <typename R, int K>
__device__ __forceinline__ cplx_t<R> taylor_cplx(const R (&cr)[K + 1], const R (&ci)[K + 1], R dwr, R dwi) {
    R pr = cr[K], pi = ci[K];
#pragma unroll
    for (int k = K - 1; k >= 0; --k) {
        const R qr = mad(pr, dwr, mad(-pi, dwi, cr[k]));
        pi = mad(pr, dwi, mad(pi, dwr, ci[k]));
        pr = qr;
    }
    return mk(pr, pi);
}

// One closed-form step given T: 27 arithmetic instructions + 1 MUFU.
template <typename R>
__device__ __forceinline__ cplx_t<R> step_T(cplx_t<R> g, R Dr, R Di, R zr, R zi, cplx_t<R> T) {
    const R ur = mad(zr, g.re, mad(-zi, g.im, Dr));        // u = z g + De
    const R ui = mad(zr, g.im, mad(zi, g.re, Di));
    const R Nr = mad(-T.re, ui, mad(-T.im, ur, g.re));     // N = g + i T u
    const R Ni = mad(T.re, ur, mad(-T.im, ui, g.im));
    const R vr = mad(Dr, g.re, mad(Di, g.im, zr));         // v = z + conj(De) g
    const R vi = mad(Dr, g.im, mad(-Di, g.re, zi));
    const R Qr = mad(T.re, vi, mad(T.im, vr, R(1)));       // Q = 1 - i T v
    const R Qi = mad(-T.re, vr, T.im * vi);
    const R rq = rcp_nr(mad(Qr, Qr, Qi * Qi));
    return mk(mad(Nr, Qr, Ni * Qi) * rq, mad(Ni, Qr, -Nr * Qi) * rq);
}

// Implicit mid-point step (PAPER.md C4-C9 :984-1001, v_F = 1): gamma' = gamma + l f((gamma + gamma')/2) with
// f = i[conj(De) g^2 + 2 z g + De] is the quadratic c2 g'^2 + c1 g' + c0 = 0; the root that tends to gamma as
// l -> 0 is g' = 2 c0 / (-c1 + sqrt(c1^2 - 4 c2 c0)) with the principal square root (-c1 ~ 1, sqrt ~ 1: the
// denominator never cancels).  No exponential, no T to share: ~63 arithmetic instructions + 3 MUFU per step.
template <typename R>
__device__ __forceinline__ cplx_t<R> step_mid(cplx_t<R> g, R Dr, R Di, R zr, R zi, R len) {
    const R q = R(0.25) * len;
    const R c2r = q * Di, c2i = q * Dr;                      // c2 = i (l/4) conj(De)
    const R pr = mad(c2r, g.re, -c2i * g.im);                // c2 g
    const R pi = mad(c2r, g.im, c2i * g.re);
    const R lr = -len * zi, li = len * zr;                   // i l z
    const R c1r = mad(R(2), pr, lr) - R(1), c1i = mad(R(2), pi, li);
    const R ar = pr + lr + R(1), ai = pi + li;               // c1 - c2 g + 2
    const R c0r = mad(ar, g.re, mad(-ai, g.im, R(-4) * c2r)); // (c1 - c2 g + 2) g - 4 conj(c2)
    const R c0i = mad(ar, g.im, mad(ai, g.re, R(4) * c2i));
    const R mr = mad(c2r, c0r, -c2i * c0i), mi = mad(c2r, c0i, c2i * c0r);      // c2 c0
    const R dr = mad(c1r, c1r, mad(-c1i, c1i, R(-4) * mr));  // c1^2 - 4 c2 c0
    const R di = mad(R(2) * c1r, c1i, R(-4) * mi);
    R sr, si, rq;
    csqrt_inv(dr, di, sr, si, rq);
    const R er = sr - c1r, ei = si - c1i;                    // -c1 + sqrt(.)
    const R rd = R(2) * rcp_nr(mad(er, er, ei * ei));
    return mk(mad(c0r, er, c0i * ei) * rd, mad(c0i, er, -c0r * ei) * rd);
}

// Local homogeneous solution gamma_h = -De/(z + i Omega) (start values, boundary reset): rare, library math,
// always evaluated in fp64.
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
