// sc_kernels.cuh — sm_100a kernels of the Riccati sweep.
//
//   rotate_in_kernel     a2: Delta, A on the reference grid -> node coefficients on every trajectory
//   reset_store_kernel   R8: boundary stores := local homogeneous solution
//   march_kernel         a3+a4+a5: boundary gather, gamma-tilde down (stores gamma-tilde per node), gamma up,
//                        node products, reduction over energies
//   rotate_back_kernel   a6+a7: masked-bilinear gather of the per-angle sums to the grid, angle sum, finalise
//
// One warp owns one trajectory of one angle pair (k, k+N/2); its 32 lanes are 32 energies.  Delta and A
// at the nodes are warp-uniform, every scratch access is a 512-byte contiguous warp transaction, the
// energy sum is a shared-memory transpose + column sum (no atomics anywhere on the data path), and the
// sums of successive 32-energy rounds are accumulated by the same warp in the per-pair partial array.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "sc_math.cuh"

namespace sck {
using scm::cplx;
using scm::cplxf;
using scm::cplx_t;
using scm::mk;

// vector types of the march's working precision R (opts.precision: 64 -> double, 32 -> float)
template <typename R> struct VT;
template <> struct VT<double> { using V2 = double2; using V4 = double4; };
template <> struct VT<float> { using V2 = float2; using V4 = float4; };
__device__ __forceinline__ double2 mk2(double a, double b) { return make_double2(a, b); }
__device__ __forceinline__ float2 mk2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ double4 mk4(double a, double b, double c, double d) { return make_double4(a, b, c, d); }
__device__ __forceinline__ float4 mk4(float a, float b, float c, float d) { return make_float4(a, b, c, d); }

// kernels of this library launched by the calling host thread (one context per host thread) since the last
// sc_debug_launch_count; library routines (cuFFT, cuBLAS, cuSOLVER) and memsets / copies are not counted
inline thread_local long long g_launches = 0;

constexpr int MAX_COMP = 4;        // order-parameter components Delta_G (Eq. 1 :37)
struct GridDev {
    int nx, ny; double h;
    const unsigned char* mask;
    const double2* delta; const double* Ax; const double* Ay;   // delta: [ncomp][ny][nx]; Ax/Ay may be null
    int ncomp;
};

struct TrajDev {                 // physical trajectories (angles k < N/2), struct of arrays
    int n;                       // count
    const int* k; const int* t; const int* jf; const int* nn;
    const double* l0; const double* l1;
    const long long* noff;       // first node in the node arrays
    const int* dF; const int* dB;   // store rows: (k,t) and its mirror (k+N/2, N_rot-1-t)
};

// tc: per-energy Taylor table of the step coefficient T (sc_math.cuh), [ne][TC_LD] = Re c_0..c_8, Im c_0..c_8,
// (distance from w0 = -z0^2 to the nearest pole of T)^2.  tmode 1: every energy on the imaginary axis (real c_k);
// 2: general energies in the upper half plane (complex c_k).
// tcp (tmode 1 only): the pole-subtracted table, [ne][TCP_LD] = r_0..r_8, (distance to the second pole)^2, w0 + wp, 2/h.
constexpr int TC_KMAX = 8;
constexpr int TC_LD = 2 * (TC_KMAX + 1) + 2;
constexpr int TCP_LD = 12;
struct EnergyDev { int ne; const double* zr; const double* zi; const double* w; const int* partner; const double* tc; const double* tcp; int tmode; };

// ------------------------------------------------------------------------------------------------
// masked bilinear interpolation of Delta (R5) and plain bilinear of A at a point
// ------------------------------------------------------------------------------------------------
// R5 fallback (rare, out of line): no corner in the mask -> nearest mask point within 2 cells
__device__ __noinline__ int nearest_mask_point(const unsigned char* mask, int nx, int ny, double gx, double gy, int i0, int j0) {
    double bd = 1e300; int best = -1;
    for (int jj = j0 - 2; jj <= j0 + 3; ++jj)
        for (int ii = i0 - 2; ii <= i0 + 3; ++ii) {
            if (ii < 0 || ii >= nx || jj < 0 || jj >= ny || !mask[(size_t)jj * nx + ii]) continue;
            const double d = (gx - ii) * (gx - ii) + (gy - jj) * (gy - jj);
            if (d < bd) { bd = d; best = jj * nx + ii; }
        }
    return best;
}
__device__ __forceinline__ bool interp_delta(const GridDev& G, const double2* __restrict__ F, double x, double y, double& dr, double& di) {
    const double gx = x / G.h + 0.5 * (G.nx - 1), gy = y / G.h + 0.5 * (G.ny - 1);
    const int i0 = (int)floor(gx), j0 = (int)floor(gy);
    const double fx = gx - i0, fy = gy - j0;
    double sw = 0.0, ar = 0.0, ai = 0.0;
#pragma unroll
    for (int b = 0; b < 2; ++b)
#pragma unroll
        for (int a = 0; a < 2; ++a) {
            const int ii = min(max(i0 + a, 0), G.nx - 1), jj = min(max(j0 + b, 0), G.ny - 1);
            const double w = (a ? fx : 1.0 - fx) * (b ? fy : 1.0 - fy);
            const size_t q = (size_t)jj * G.nx + ii;
            if (G.mask[q]) { const double2 d = F[q]; sw += w; ar += w * d.x; ai += w * d.y; }
        }
    if (sw > 1e-12) { dr = ar / sw; di = ai / sw; return true; }
    const int best = nearest_mask_point(G.mask, G.nx, G.ny, gx, gy, i0, j0);
    if (best < 0) { dr = di = 0.0; return false; }
    const double2 d = F[best];
    dr = d.x; di = d.y;
    return true;
}
// Delta(p_F, R) = sum_G eta_G Delta_G(R) (Eq. 1 :37) at a point; eta: the ncomp basis-function values of the direction,
// `stride` apart
__device__ __forceinline__ bool interp_gap(const GridDev& G, const double* eta, int stride, double x, double y, double& dr, double& di) {
    const size_t ng = (size_t)G.nx * G.ny;
    bool ok = true;
    dr = di = 0.0;
    for (int c = 0; c < G.ncomp; ++c) {
        double r, i;
        ok = interp_delta(G, G.delta + c * ng, x, y, r, i) && ok;
        const double e = eta[(size_t)c * stride];
        dr = fma(e, r, dr); di = fma(e, i, di);
    }
    return ok;
}

__device__ __forceinline__ double interp_plain(const GridDev& G, const double* F, double x, double y) {
    if (!F) return 0.0;
    const double gx = x / G.h + 0.5 * (G.nx - 1), gy = y / G.h + 0.5 * (G.ny - 1);
    const int i0 = (int)floor(gx), j0 = (int)floor(gy);
    const double fx = gx - i0, fy = gy - j0;
    double acc = 0.0;
#pragma unroll
    for (int b = 0; b < 2; ++b)
#pragma unroll
        for (int a = 0; a < 2; ++a) {
            const int ii = min(max(i0 + a, 0), G.nx - 1), jj = min(max(j0 + b, 0), G.ny - 1);
            acc += (a ? fx : 1.0 - fx) * (b ? fy : 1.0 - fy) * F[(size_t)jj * G.nx + ii];
        }
    return acc;
}

// a2: one warp per trajectory, lanes over nodes (coalesced along the trajectory).  Also writes the PIECE
// coefficients the march consumes: piece p of a trajectory with nn nodes (p = 0..nn) is {Re De, Im De, a, |De|^2 - a^2}
// with De, a the half-step values by linear interpolation and nearest-neighbour extrapolation at both ends
// (reading R4); its length is l0 (p = 0), l1 (p = nn) or h.  Piece records of trajectory g start at
// noff[g] + g.  The fourth entry is the energy-independent part of the argument of the T table (sc_math.cuh).
template <typename R>
__global__ void __launch_bounds__(256, 3) rotate_in_kernel(GridDev G, TrajDev T, const double* vx, const double* vy, const double* eta /*[ncomp][nphi]*/,
                                 int nphi, double c, int sigma, double2* nd_D, double* nd_a, typename VT<R>::V2* nd_Dr,
                                 typename VT<R>::V4* pc, float2* pmax, int* n_bad) {
    const int g = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (g >= T.n) return;
    const int lane = threadIdx.x & 31;
    const int k = T.k[g];
    const double cx = vx[k], cy = vy[k], w = (T.t[g] - c) * G.h;
    const int jf = T.jf[g], nn = T.nn[g];
    const long long off = T.noff[g];
#pragma unroll 1
    for (int m = lane; m < nn; m += 32) {
        const double u = (jf + m - c) * G.h;
        const double x = u * cx - w * cy, y = u * cy + w * cx;
        double dr, di;
        if (!interp_gap(G, eta + k, nphi, x, y, dr, di)) atomicAdd(n_bad, 1);
        nd_D[off + m] = make_double2(dr, di);
        if (sizeof(R) == 4) nd_Dr[off + m] = mk2((R)dr, (R)di);                  // fp32 mode: the march reads a float copy
        nd_a[off + m] = sigma * (cx * interp_plain(G, G.Ax, x, y) + cy * interp_plain(G, G.Ay, x, y));
    }
    __syncwarp();
    typename VT<R>::V4* P = pc + off + g;
    float wmax = 0.f, amax = 0.f;        // bounds on | |De|^2 - a^2 | and |a| over the trajectory's pieces (rounded up)
    for (int p = lane; p <= nn; p += 32) {
        const int lo = p > 0 ? p - 1 : 0, hi = p < nn ? p : nn - 1;
        const double2 Dl = nd_D[off + lo], Dh = nd_D[off + hi];
        const double al = nd_a[off + lo], ah = nd_a[off + hi];
        const double dx = lo == hi ? Dl.x : 0.5 * (Dl.x + Dh.x), dy = lo == hi ? Dl.y : 0.5 * (Dl.y + Dh.y);
        const double am = lo == hi ? al : 0.5 * (al + ah);
        const typename VT<R>::V4 rec = mk4((R)dx, (R)dy, (R)am, (R)(dx * dx + dy * dy - am * am));
        P[p] = rec;
        wmax = fmaxf(wmax, __double2float_ru(fabs((double)rec.w))); amax = fmaxf(amax, __double2float_ru(fabs((double)rec.z)));
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) { wmax = fmaxf(wmax, __shfl_xor_sync(0xffffffffu, wmax, o)); amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o)); }
    if (lane == 0) pmax[g] = make_float2(wmax, amax);
}

// fallback coefficients for boundary points that have no valid specular partner (R6 fallback):
// Delta(R_min) eta(mirrored direction) and sigma v_in . A(R_min)
__global__ void fallback_kernel(GridDev G, int nfb, const int* rows, const double* px, const double* py,
                                const double* dx, const double* dy, const double* eta_m /*[ncomp][nfb]*/, int sigma,
                                double2* fb_D, double* fb_a) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nfb) return;
    double dr, di;
    interp_gap(G, eta_m + i, nfb, px[i], py[i], dr, di);
    fb_D[rows[i]] = make_double2(dr, di);
    fb_a[rows[i]] = sigma * (dx[i] * interp_plain(G, G.Ax, px[i], py[i]) + dy[i] * interp_plain(G, G.Ay, px[i], py[i]));
}

// R8: store[dF][n] = gamma_h(last piece); store[dB][partner n] = conj(gamma-tilde_h(first piece)).
template <typename R>
__global__ void reset_store_kernel(TrajDev T, EnergyDev E, const typename VT<R>::V4* pc, typename VT<R>::V2* store) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)T.n * E.ne) return;
    const int g = (int)(idx / E.ne), n = (int)(idx % E.ne);
    const typename VT<R>::V4* P = pc + T.noff[g] + g;
    const typename VT<R>::V4 cl = P[T.nn[g]], c0 = P[0];
    const cplx ge = scm::gamma_hom(cl.x, cl.y, E.zr[n] + cl.z, E.zi[n]);
    store[(size_t)T.dF[g] * E.ne + n] = mk2((R)ge.re, (R)ge.im);
    const cplx gt = scm::gamma_hom(-(double)c0.x, c0.y, E.zr[n] + c0.z, E.zi[n]);
    store[(size_t)T.dB[g] * E.ne + E.partner[n]] = mk2((R)gt.re, (R)-gt.im);
}

// ------------------------------------------------------------------------------------------------
// the march (working precision R = double, or float with opts.precision = 32)
// ------------------------------------------------------------------------------------------------
template <typename R>
struct MarchArgsT {
    using V2 = typename VT<R>::V2; using V4 = typename VT<R>::V4;
    TrajDev T;
    EnergyDev E;
    const int* order; int n_items;          // longest-first work list
    const V2* nd_D;                         // node coefficients Delta_j eta_k           [node]
    const V4* pc;                           // piece coefficients {Re De, Im De, a, |De|^2 - a^2} [node + g]
    const float2* pmax;                     // per trajectory: max | |De|^2 - a^2 |, max |a| over its pieces
    double h;                               // length of every interior piece
    int bc_mode;
    const int* ga_idx; const double* ga_w; const unsigned char* ga_n;   // entry gathers per store row [row][4]
    const double2* fb_D; const double* fb_a;
    const V2* store_old; V2* store_new;
    char* scr; long long scr_stride;        // per warp slot: scr_stride bytes = (smax+2) rows of 32 entries of 4 R
    double* part;                           // MODE 0: [node][6] = SF.re, SF.im, X2.re, X2.im, SG/2, SI
    double* ldos;                           // MODE 1: [node][ne] = Re g_n
    int* counter;
    double* stat_max2;                      // per warp slot: max |gamma|^2 seen (optional)
    unsigned long long* n_stored;           // [0] running count of (piece, energy) units marched by rounds that spilled T,
                                            // [1] by rounds that re-evaluated T from the pole-subtracted table
};
using MarchArgs = MarchArgsT<double>;

constexpr int MARCH_WARPS = 8;               // warps per CTA
constexpr int MARCH_MIN_CTAS = 2;            // resident CTAs per SM the fp64 register budget is sized for (128 registers per thread)
constexpr int P1_UNROLL = 2;                 // pass 1: pieces per unrolled loop body
constexpr int PF_DIST = 16;                  // pass 2: scratch lines are pulled into L2 this many nodes ahead
constexpr int RED_NODES = 4;                 // nodes per shared-memory reduction batch
constexpr int RED_VALS = 6;
constexpr int STAGE_LD = 34;                 // padded row of the transpose stage: 16-byte aligned rows, conflict-free 128-bit column reads

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
// warp-uniform coefficient record (read-only path)
__device__ __forceinline__ double4 ldu(const double4* p) {
    double4 v;
    asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ float4 ldu(const float4* p) { return __ldg(p); }

template <typename R>
__device__ __forceinline__ cplx_t<R> gather_start(const MarchArgsT<R>& A, int row, int n) {
    const int cnt = A.ga_n[row];
    R sr = R(0), si = R(0);
    for (int i = 0; i < cnt; ++i) {
        const R w = (R)A.ga_w[4 * row + i];
        const typename VT<R>::V2 v = A.store_old[(size_t)A.ga_idx[4 * row + i] * A.E.ne + n];
        sr = scm::mad(w, v.x, sr); si = scm::mad(w, v.y, si);
    }
    return mk(sr, si);
}
template <typename R>
__device__ __forceinline__ cplx_t<R> hom_start(double Dr, double Di, double zr, double zi) {   // rare: fp64 library math
    const cplx s = scm::gamma_hom(Dr, Di, zr, zi);
    return mk((R)s.re, (R)s.im);
}

// products at one node (Eq. 24 :165): P = gamma gamma~, 1/(1+P); writes the six weighted terms of the
// energy sums into rows r..r+5 of the warp's transpose stage (MODE 0), or returns Re g (MODE 1)
// UW: every weight of the energy table is 1 and every lane is active (plain Matsubara sums over a multiple of 32 energies):
// the two multiplications by w_n are compiled out (bitwise the same result)
template <int MODE, bool STATS, typename R, bool UW>
__device__ __forceinline__ R node_products(cplx_t<R> gm, R gtr, R gti, typename VT<R>::V2 Dn, R wn, R* st, R& max2) {
    using scm::mad;
    const R Pr = mad(gm.re, gtr, -gm.im * gti), Pi = mad(gm.re, gti, gm.im * gtr);
    const R qr = R(1) + Pr;
    const R rq = scm::rcp_nr(mad(qr, qr, Pi * Pi));
    if (STATS) max2 = scm::maxr(max2, scm::maxr(mad(gm.re, gm.re, gm.im * gm.im), mad(gtr, gtr, gti * gti)));
    if (MODE == 0) {
        const R wq = UW ? rq : wn * rq;
        const R wr = qr * wq, wi = -Pi * wq;                 // w/(1+P)
        st[0 * STAGE_LD] = mad(gm.re, wr, -gm.im * wi);      // SF  = w gamma/(1+P)
        st[1 * STAGE_LD] = mad(gm.re, wi, gm.im * wr);
        st[2 * STAGE_LD] = mad(gtr, wr, -gti * wi);          // X2  = w gamma~/(1+P)  (SF of k+N/2 = conj)
        st[3 * STAGE_LD] = mad(gtr, wi, gti * wr);
        st[4 * STAGE_LD] = wi;                               // SG/2 = w Im 1/(1+P) (Im g = 2 Im 1/(1+P): doubled in rotate-back)
        const R si = mad(Dn.x, gm.im - gti, -Dn.y * (gm.re + gtr));
        st[5 * STAGE_LD] = UW ? si : wn * si;   // SI (Eq. 19 :128 numerator)
    }
    return mad(R(2) * qr, rq, R(-1));                        // Re g = 2 Re 1/(1+P) - 1
}

// column sums of the stage: lane c < cnt sums row c over the 32 lanes — 8 partial sums of 4 values each, then a
// fixed tree (31 additions, dependency depth 6)
template <typename R>
__device__ __forceinline__ double stage_colsum(const R* stage, int lane) {
    using V2 = typename VT<R>::V2;
    const V2* col = reinterpret_cast<const V2*>(stage + lane * STAGE_LD);
    R s[8];
#pragma unroll
    for (int q = 0; q < 4; ++q) { const V2 a = col[q]; s[2 * q] = a.x; s[2 * q + 1] = a.y; }
#pragma unroll
    for (int i = 4; i < 16; i += 4)
#pragma unroll
        for (int q = 0; q < 4; ++q) { const V2 a = col[i + q]; s[2 * q] += a.x; s[2 * q + 1] += a.y; }
    return (double)(((s[0] + s[1]) + (s[2] + s[3])) + ((s[4] + s[5]) + (s[6] + s[7])));
}

// Scratch between the two passes, one entry per (piece or node, lane), a warp's 32 entries contiguous.
//   ST = false ("recompute"): entry m = gamma~(node m) = 2 R.  T is NOT spilled: re-evaluating it from the table in
//        pass 2 costs 18 FP64 instructions against 32 B of HBM traffic (~70 instruction slots at the machine balance).
//        Chosen per (trajectory, 32-energy round) when every piece is inside the table's radius (bound from pmax).
//   ST = true  ("stored"):    entry p = {T_p, gamma~(node p-1)} = 4 R, one 256-bit (fp64) / 128-bit (fp32) access:
//        T is evaluated once per piece, from the table where a warp vote allows, from exp/sqrt elsewhere.
//   STEP 1 (mid-point) has no T: always the 2 R layout.
template <typename R> struct Ent { R tr, ti, gr, gi; };
template <typename R, bool ST> struct ScrT { static constexpr int BYTES = (ST ? 4 : 2) * (int)sizeof(R); static constexpr int ROW = 32 * BYTES; };
template <bool ST>
__device__ __forceinline__ Ent<double> ld_ent(const char* p, double) {
    Ent<double> e;
    if (ST) asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(e.tr), "=d"(e.ti), "=d"(e.gr), "=d"(e.gi) : "l"(p));
    else { asm volatile("ld.global.v2.f64 {%0,%1}, [%2];" : "=d"(e.gr), "=d"(e.gi) : "l"(p)); e.tr = e.ti = 0.0; }
    return e;
}
template <bool ST>
__device__ __forceinline__ Ent<float> ld_ent(const char* p, float) {
    Ent<float> e;
    if (ST) asm volatile("ld.global.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(e.tr), "=f"(e.ti), "=f"(e.gr), "=f"(e.gi) : "l"(p));
    else { asm volatile("ld.global.v2.f32 {%0,%1}, [%2];" : "=f"(e.gr), "=f"(e.gi) : "l"(p)); e.tr = e.ti = 0.f; }
    return e;
}
template <bool ST>
__device__ __forceinline__ void st_ent(char* p, cplx T, cplx gt) {
    if (ST) asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(T.re), "d"(T.im), "d"(gt.re), "d"(gt.im) : "memory");
    else asm volatile("st.global.v2.f64 [%0], {%1,%2};" ::"l"(p), "d"(gt.re), "d"(gt.im) : "memory");
}
template <bool ST>
__device__ __forceinline__ void st_ent(char* p, cplxf T, cplxf gt) {
    if (ST) asm volatile("st.global.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(T.re), "f"(T.im), "f"(gt.re), "f"(gt.im) : "memory");
    else asm volatile("st.global.v2.f32 [%0], {%1,%2};" ::"l"(p), "f"(gt.re), "f"(gt.im) : "memory");
}

// Per-lane Taylor table of T about this lane's energy (TM 1: real coefficients, 2: complex) and its evaluation for
// one piece record.
template <typename R, int TM>
struct TTab {
    static constexpr int K = scm::TaylorK<R>::K;
    static constexpr bool IMAG = TM == 1;       // every energy on the imaginary axis: Re z = a exactly
    R cr[K + 1]; R ci[TM == 2 ? K + 1 : 1];
    R thr2, m2zr, m2zi;
    __device__ __forceinline__ void load(const EnergyDev& E, int n) {
        const double* row = E.tc + (size_t)n * TC_LD;
#pragma unroll
        for (int k = 0; k <= K; ++k) { cr[k] = (R)row[k]; if (TM == 2) ci[k] = (R)row[TC_KMAX + 1 + k]; }
        if (TM != 2) ci[0] = R(0);
        thr2 = (R)(row[2 * (TC_KMAX + 1)] * (scm::TaylorK<R>::RMAX * scm::TaylorK<R>::RMAX));
        m2zr = (R)(-2.0 * E.zr[n]); m2zi = (R)(-2.0 * E.zi[n]);
    }
    // every piece of a trajectory with the bounds pm is inside the radius of energy n (conservative; 1e-3 covers rounding)
    static __device__ __forceinline__ bool covers(const EnergyDev& E, int n, float2 pm) {
        const R thr = (R)(E.tc[(size_t)n * TC_LD + 2 * (TC_KMAX + 1)] * (scm::TaylorK<R>::RMAX * scm::TaylorK<R>::RMAX));
        const R br = (R)pm.x + (R)(2.0 * fabs(E.zr[n])) * (R)pm.y, bi = (R)(2.0 * E.zi[n]) * (R)pm.y;
        return scm::mad(br, br, bi * bi) * R(1.001) <= thr;
    }
    // dw = (|De|^2 - a^2) - 2 z0 a
    __device__ __forceinline__ cplx_t<R> taylor(const typename VT<R>::V4& cc, R dwr, R dwi, R s2) const {
        if constexpr (TM == 2) return scm::taylor_cplx<R, K>(cr, ci, dwr, dwi);
        else return scm::taylor_real<R, K>(cr, dwr, dwi, s2);
    }
    // known to be inside the radius
    __device__ __forceinline__ cplx_t<R> fast(const typename VT<R>::V4& cc) const {
        const R dwr = TM == 2 ? scm::mad(m2zr, cc.z, cc.w) : cc.w, dwi = m2zi * cc.z;
        return taylor(cc, dwr, dwi, scm::mad(dwr, dwr, dwi * dwi));
    }
    // one warp vote per piece: table inside the radius, exp-based evaluation outside
    __device__ __forceinline__ cplx_t<R> voted(const typename VT<R>::V4& cc, R zr0, R zi0, R len) const {
        const R dwr = TM == 2 ? scm::mad(m2zr, cc.z, cc.w) : cc.w, dwi = m2zi * cc.z;
        const R s2 = scm::mad(dwr, dwr, dwi * dwi);
        if (!__any_sync(0xffffffffu, !(s2 <= thr2))) return taylor(cc, dwr, dwi, s2);
        return scm::coef_T_slow(scm::mad(cc.x, cc.x, cc.y * cc.y), zr0 + cc.z, zi0, len);
    }
};
// Pole-subtracted table (energies on the imaginary axis): three times the radius.  KC = TaylorPoleK (degree 8) for the
// rounds that spill T (one warp vote per piece, exp-based evaluation outside the radius); KC = TaylorPoleShortK
// (degree 5) for rounds that re-evaluate T in pass 2 and are known to be inside its radius.
template <typename R, typename KC>
struct TTabPole {
    static constexpr int K = KC::K;
    static constexpr bool IMAG = true;
    R c[K + 1]; R thr2, pole_a, pole_res, m2zi;
    __device__ __forceinline__ void load(const EnergyDev& E, int n) {
        const double* row = E.tcp + (size_t)n * TCP_LD;
#pragma unroll
        for (int k = 0; k <= K; ++k) c[k] = (R)row[k];
        thr2 = (R)(row[9] * (KC::RMAX * KC::RMAX));
        pole_a = (R)row[10]; pole_res = (R)row[11]; m2zi = (R)(-2.0 * E.zi[n]);
    }
    static __device__ __forceinline__ bool covers(const EnergyDev& E, int n, float2 pm) {
        const R thr = (R)(E.tcp[(size_t)n * TCP_LD + 9] * (KC::RMAX * KC::RMAX));
        const R br = (R)pm.x, bi = (R)(2.0 * E.zi[n]) * (R)pm.y;
        return scm::mad(br, br, bi * bi) * R(1.001) <= thr;
    }
    __device__ __forceinline__ cplx_t<R> fast(const typename VT<R>::V4& cc) const {
        const R dwr = cc.w, dwi = m2zi * cc.z;
        return scm::taylor_pole<R, K>(c, pole_a, pole_res, dwr, dwi, scm::mad(dwr, dwr, dwi * dwi));
    }
    __device__ __forceinline__ cplx_t<R> voted(const typename VT<R>::V4& cc, R zr0, R zi0, R len) const {
        const R dwr = cc.w, dwi = m2zi * cc.z;
        const R s2 = scm::mad(dwr, dwr, dwi * dwi);
        if (!__any_sync(0xffffffffu, !(s2 <= thr2))) return scm::taylor_pole<R, K>(c, pole_a, pole_res, dwr, dwi, s2);
        return scm::coef_T_slow(scm::mad(cc.x, cc.x, cc.y * cc.y), zr0 + cc.z, zi0, len);
    }
};
// T of an end piece (length != h): exp-based
template <typename R>
__device__ __forceinline__ cplx_t<R> end_T(const typename VT<R>::V4& cc, R zr0, R zi0, R len) {
    return scm::coef_T_slow(scm::mad(cc.x, cc.x, cc.y * cc.y), zr0 + cc.z, zi0, len);
}

// ---- coefficient staging: the warp-uniform piece / node records of a trajectory are streamed through shared
// memory in chunks of 32 (one record per lane, coalesced cp.async, double-buffered one chunk ahead), so that no
// step ever waits on a global load of its coefficients; the step loop reads them with broadcast LDS.
constexpr int CHUNK = 32;
static_assert(CHUNK % RED_NODES == 0, "a reduction batch must not straddle two coefficient chunks (the running sums are fetched one batch ahead)");
template <typename R> __host__ __device__ constexpr int march_stage_bytes() { return RED_NODES * RED_VALS * STAGE_LD * (int)sizeof(R); }   // per warp
template <typename R> __host__ __device__ constexpr int march_coef_bytes() { return 2 * CHUNK * 6 * (int)sizeof(R); }                      // per warp: pc[2][32] V4 + nd[2][32] V2
template <typename R> __host__ __device__ constexpr int march_smem() { return MARCH_WARPS * (march_stage_bytes<R>() + march_coef_bytes<R>()); }   // fp64: 75264 B (opt-in)

template <int BYTES>
__device__ __forceinline__ void cp_async(void* smem, const void* gmem) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    if (BYTES == 32) {
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa + 16), "l"((const char*)gmem + 16) : "memory");
    } else if (BYTES == 16) {
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
    } else {
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(gmem) : "memory");
    }
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// state of one warp while it works on one trajectory
template <typename R>
struct WarpJob {
    using V2 = typename VT<R>::V2; using V4 = typename VT<R>::V4;
    int lane, nn, dF, dB, ne; long long noff;
    R len0, len1, hlen;
    const V2* ND; const V4* PC; double* PART;
    R* stage; V4* pcb; V2* ndb;
    char* scr_w;                             // this warp slot's scratch
};

// One 32-energy round of one trajectory: pass 1 (gamma-tilde from u_out down to u_in, spilled per node), pass 2
// (gamma from u_in up to u_out, node products, reduction over the 32 energies).
// MODE 0: Matsubara sums; 1: per-energy Re g (LDOS); 2: boundary values only.
// STEP 0: closed-form step; 1: implicit mid-point rule (C4-C9 :984-1001).
// ST: T spilled with gamma-tilde (see ScrT).  TM: layout of the T table.
template <int MODE, bool STATS, int STEP, typename R, bool ST, bool UW, typename TAB>
__device__ __forceinline__ void march_round(const MarchArgsT<R>& A, const WarpJob<R>& J, const TAB& tab, int n0, R& max2) {
    using V2 = typename VT<R>::V2; using V4 = typename VT<R>::V4;
    constexpr int ROW = ScrT<R, ST>::ROW, BYTES = ScrT<R, ST>::BYTES;
    constexpr int NB = ST ? 1 : 0;                          // ST: node m lives in entry m+1 (entry p = piece p)
    // HALF: only every second gamma~ is spilled (odd nodes, and the last node); pass 2 steps the stored value of node
    // m+1 down across piece m+1 — with the T it evaluates anyway for gamma's step up across the same piece — to get
    // gamma~ at the even node m: one more Moebius step per two units (13.5 FP64 instructions per unit) for half the
    // scratch traffic (16 instead of 32 B per unit).  Entry m>>1 holds node m+1 (m even, m+1 < nn) or the last node.
    constexpr bool HALF = !ST && STEP == 0;
    constexpr int PFROWS = HALF ? RED_NODES / 2 : RED_NODES;   // scratch rows one reduction batch consumes
    const int lane = J.lane, nn = J.nn, ne = J.ne;
    char* const scr = J.scr_w + lane * BYTES;               // entry e of this lane: scr + e*ROW
    const bool pf_lane = lane * 128 < PFROWS * ROW;         // lanes that cover a batch's rows in 128-byte lines
    const bool act = n0 + lane < ne;
    const int n = act ? n0 + lane : ne - 1;
    const R zr0 = (R)A.E.zr[n], zi0 = (R)A.E.zi[n];
    const R wn = act ? (R)A.E.w[n] : R(0);
    const int nb = A.E.partner[n];
    const V4* __restrict__ PC = J.PC; const V2* __restrict__ ND = J.ND;
    V4* const pcb = J.pcb; V2* const ndb = J.ndb;
    const int npart = nn * RED_VALS;

    // T of piece cc and the step across it
    auto coefT = [&](const V4& cc, bool interior, R len) -> cplx_t<R> {
        if (STEP != 0) return mk(R(0), R(0));
        if (!interior) return end_T<R>(cc, zr0, zi0, len);
        if (ST) return tab.voted(cc, zr0, zi0, len);
        return tab.fast(cc);
    };
    auto stepT = [&](cplx_t<R> g, R sgn, const V4& cc, cplx_t<R> T, R len) -> cplx_t<R> {
        if (STEP == 0) return scm::step_T(g, sgn * cc.x, cc.y, TAB::IMAG ? cc.z : zr0 + cc.z, zi0, T);
        return scm::step_mid(g, sgn * cc.x, cc.y, zr0 + cc.z, zi0, len);
    };

    // ---------------- pass 1: gamma-tilde from u_out down to u_in ----------------
    const int ctop = nn >> 5;                                  // chunk c holds pieces 32c .. 32c+31
    if (ctop * CHUNK + lane <= nn) cp_async<sizeof(V4)>(pcb + (ctop & 1) * CHUNK + lane, PC + ctop * CHUNK + lane);
    cp_commit();
    cplx_t<R> gt;
    if (A.bc_mode == 1) {
        const V4 c4 = ldu(PC + nn);
        gt = hom_start<R>(-(double)c4.x, c4.y, A.E.zr[n] + c4.z, A.E.zi[n]);
    } else if (A.ga_n[J.dB]) {
        const cplx_t<R> s = gather_start(A, J.dB, nb);            // gamma of the mirrored trajectory at its entry
        gt = mk(s.re, -s.im);
    } else {
        const cplx_t<R> s = hom_start<R>(A.fb_D[J.dB].x, A.fb_D[J.dB].y, A.E.zr[nb] + A.fb_a[J.dB], A.E.zi[nb]);
        gt = mk(s.re, -s.im);
    }
    cplx_t<R> T0 = mk(R(0), R(0));                             // T of the entry piece, kept for pass 2 when not spilled
    {
        // the step across piece p lands on node p-1: entry p (ST) or entry p-1 (gamma~ only)
        char* e = scr + (size_t)(HALF ? (nn - 1) >> 1 : nn - 1 + NB) * ROW;   // HALF: successive spills go to successive lower rows
        int p = nn;
        for (int c = ctop; c >= 0; --c) {
            if (c > 0) {
                cp_async<sizeof(V4)>(pcb + ((c - 1) & 1) * CHUNK + lane, PC + (c - 1) * CHUNK + lane);
                cp_commit();
                cp_wait<1>();
            } else {
                cp_wait<0>();
            }
            __syncwarp();
            const V4* __restrict__ buf = pcb + (c & 1) * CHUNK;
            const int plo = max(c * CHUNK, 1);
            if (p == nn) {                                      // exit piece (length l1)
                const V4 cc = buf[p & (CHUNK - 1)];
                const cplx_t<R> T = coefT(cc, false, J.len1);
                gt = stepT(gt, R(-1), cc, T, J.len1);
                if (MODE != 2 || ST) st_ent<ST>(e, T, gt);      // (HALF: the last node is always spilled)
                e -= ROW; --p;
            }
            const V4* __restrict__ bp = buf + (p & (CHUNK - 1));
#pragma unroll P1_UNROLL
            for (; p >= plo; --p, --bp) {
                const V4 cc = *bp;
                const cplx_t<R> T = coefT(cc, true, J.hlen);
                gt = stepT(gt, R(-1), cc, T, J.hlen);
                if (HALF) { if (!(p & 1)) { if (MODE != 2) st_ent<ST>(e, T, gt); e -= ROW; } }   // landed on the odd node p-1: row (p-1)>>1
                else { if (MODE != 2 || ST) st_ent<ST>(e, T, gt); e -= ROW; }
            }
            if (c == 0) {                                       // entry piece (length l0); its gamma~ is the end value
                const V4 cc = buf[0];
                T0 = coefT(cc, false, J.len0);
                gt = stepT(gt, R(-1), cc, T0, J.len0);
            }
            __syncwarp();                                       // chunk c is free for the load issued next round
        }
        if (act) A.store_new[(size_t)J.dB * ne + nb] = mk2(gt.re, -gt.im);
    }

    // ---------------- pass 2: gamma from u_in up to u_out; products and energy reduction ------------
    // chunk c of pass 2 holds, for nodes m = 32c .. 32c+31, the piece m+1 (the step that leaves the node) and Delta_m
    const int nchunk = (nn + CHUNK - 1) >> 5;
    cplx_t<R> gm;
    {
        const V4 c0 = pcb[0];                                   // piece 0 is still in buffer 0 (last chunk of pass 1)
        __syncwarp();
        if (lane < nn) {
            cp_async<sizeof(V4)>(pcb + CHUNK + lane, PC + 1 + lane);      // pass-2 chunk 0 goes to buffer 1
            cp_async<sizeof(V2)>(ndb + CHUNK + lane, ND + lane);
        }
        cp_commit();
        if (A.bc_mode == 1) gm = hom_start<R>(c0.x, c0.y, A.E.zr[n] + c0.z, A.E.zi[n]);
        else if (A.ga_n[J.dF]) gm = gather_start(A, J.dF, n);
        else gm = hom_start<R>(A.fb_D[J.dF].x, A.fb_D[J.dF].y, A.E.zr[n] + A.fb_a[J.dF], A.E.zi[n]);
        gm = stepT(gm, R(1), c0, T0, J.len0);
    }
    constexpr bool LD = ST || MODE != 2;        // pass 2 reads the scratch (burn-in sweeps without spilled T do not)
    const char* e = scr + NB * ROW;             // entry of node 0
    if (LD)
        for (int q = RED_NODES; q < PF_DIST && q < nn; q += RED_NODES)
            if (pf_lane) prefetch_l2(J.scr_w + (size_t)(HALF ? q >> 1 : q + NB) * ROW + lane * 128);
    Ent<R> En{}, En2{};                          // the next two entries (register look-ahead over the HBM latency)
    if (LD) { En = ld_ent<ST>(e, R(0)); En2 = ld_ent<ST>(e + ROW, R(0)); }
    cplx_t<R> gt_odd = mk(R(0), R(0));           // HALF: gamma~ of the odd node, held from the even node before it
    double part_nxt = 0.0;                       // running sums of the earlier energy rounds, fetched one batch ahead
    if (MODE == 0 && n0 && lane < RED_NODES * RED_VALS && lane < npart) part_nxt = J.PART[lane];
    int m = 0;
    // node m: products with gamma~(m) from its entry, then the step across piece m+1 (T from entry m+1 when spilled)
    auto node = [&](int b, const V4* pbuf, const V2* dbuf, bool exitp) {
        const V4 cc = pbuf[b]; const V2 dc = dbuf[b];              // pbuf, dbuf: the batch's first records in the staged chunk
        const R len = exitp ? J.len1 : J.hlen;
        if (HALF) {                                            // batches start on even nodes: the parity of m+b is that of b
            const cplx_t<R> T = coefT(cc, !exitp, len);
            cplx_t<R> gth = gt_odd;
            if (!(b & 1)) {
                const cplx_t<R> G = mk(En.gr, En.gi);          // entry (m+b)>>1: node m+b+1, or the last node itself
                if (LD) { En = En2; En2 = ld_ent<ST>(e + ((b >> 1) + 2) * ROW, R(0)); }
                gt_odd = G;
                gth = exitp ? G : stepT(G, R(-1), cc, T, len);
            }
            if (MODE != 2) {
                const R rg = node_products<MODE, STATS, R, UW>(gm, gth.re, gth.im, dc, wn, J.stage + b * RED_VALS * STAGE_LD + lane, max2);
                if (MODE == 1 && act) A.ldos[(size_t)(J.noff + m + b) * ne + n] = (double)rg;
            }
            gm = stepT(gm, R(1), cc, T, len);
            return;
        }
        const Ent<R> Ec = En;
        if (LD) { En = En2; En2 = ld_ent<ST>(e + (b + 2) * ROW, R(0)); }   // two entries ahead (the scratch has spare rows)
        if (MODE != 2) {
            const R rg = node_products<MODE, STATS, R, UW>(gm, Ec.gr, Ec.gi, dc, wn, J.stage + b * RED_VALS * STAGE_LD + lane, max2);
            if (MODE == 1 && act) A.ldos[(size_t)(J.noff + m + b) * ne + n] = (double)rg;
        }
        // ST: the entry of node m+b is the entry of piece m+b+1, the step that leaves the node: it holds that T
        const cplx_t<R> T = ST ? mk(Ec.tr, Ec.ti) : coefT(cc, !exitp, len);
        gm = stepT(gm, R(1), cc, T, len);
    };
    for (int c = 0; c < nchunk; ++c) {
        const int bsel = (c + 1) & 1;                           // chunk c lives in buffer (c+1)&1
        if (c + 1 < nchunk) {
            const int q = (c + 1) * CHUNK + lane;
            if (q < nn) {
                cp_async<sizeof(V4)>(pcb + (bsel ^ 1) * CHUNK + lane, PC + 1 + q);
                cp_async<sizeof(V2)>(ndb + (bsel ^ 1) * CHUNK + lane, ND + q);
            }
            cp_commit();
            cp_wait<1>();
        } else {
            cp_wait<0>();
        }
        __syncwarp();
        const V4* __restrict__ pbuf = pcb + bsel * CHUNK;
        const V2* __restrict__ dbuf = ndb + bsel * CHUNK;
        const int mhi = min(nn, (c + 1) * CHUNK);
        // full batches that do not end the trajectory; the last batch (exit piece) goes through the compact tail code below, so
        // that the unrolled batch exists once, not twice, in the instruction stream (rounds of different kinds share the I-cache)
        const int mfull = min(mhi, nn - 1);
        for (; m + RED_NODES <= mfull; m += RED_NODES) {
            if (LD && pf_lane && m + PF_DIST < nn) prefetch_l2(J.scr_w + (size_t)(HALF ? (m + PF_DIST) >> 1 : m + PF_DIST + NB) * ROW + lane * 128);
            const double part_old = part_nxt;
            if (MODE == 0 && n0 && lane < RED_NODES * RED_VALS && (m + RED_NODES) * RED_VALS + lane < npart)
                part_nxt = J.PART[(m + RED_NODES) * RED_VALS + lane];
            const V4* __restrict__ pb = pbuf + (m & (CHUNK - 1)); const V2* __restrict__ db = dbuf + (m & (CHUNK - 1));
#pragma unroll
            for (int b = 0; b < RED_NODES; ++b) node(b, pb, db, false);
            e += PFROWS * ROW;
            if (MODE == 0) {
                __syncwarp();
                if (lane < RED_NODES * RED_VALS) {
                    double s = stage_colsum(J.stage, lane);
                    if (n0) s += part_old;
                    J.PART[m * RED_VALS + lane] = s;
                }
                __syncwarp();
            }
        }
        if (m < mhi) {                                       // the last 1..4 nodes of the trajectory (last chunk only)
            const int rem = mhi - m;
            const double part_old = part_nxt;
            const V4* __restrict__ pb = pbuf + (m & (CHUNK - 1)); const V2* __restrict__ db = dbuf + (m & (CHUNK - 1));
#pragma unroll 1
            for (int b = 0; b < rem - 1; ++b) node(b, pb, db, false);
            node(rem - 1, pb, db, true);                         // m + rem == nn: the exit piece, with its own length
            if (MODE == 0) {
                __syncwarp();
                if (lane < rem * RED_VALS) {
                    double s = stage_colsum(J.stage, lane);
                    if (n0) s += part_old;
                    J.PART[m * RED_VALS + lane] = s;
                }
                __syncwarp();
            }
            m = mhi;
        }
        __syncwarp();                                           // this chunk's buffer is free for the next load
    }
    if (act) A.store_new[(size_t)J.dF * ne + n] = mk2(gm.re, gm.im);
}

// ---- TWO energies per lane (n0 + lane and n0 + 32 + lane) of one trajectory in one pass: the warp-uniform coefficient
// loads, the loop bookkeeping, the shared-memory transpose and the running sums are shared by the two energies (their
// six summands are added in registers before the stage), and the two independent dependency chains of a lane interleave.
// Only the common case: Matsubara sums (MODE 0), closed-form step, every piece inside the pole-free table for all 64
// energies, unit weights, no stats.  gamma~ of every second node is spilled as one 256-bit entry {gt(n), gt(n+32)}.
template <typename R>
__device__ __forceinline__ void node_terms(cplx_t<R> gm, cplx_t<R> gt, typename VT<R>::V2 Dn, R (&o)[6]) {
    using scm::mad;
    const R Pr = mad(gm.re, gt.re, -gm.im * gt.im), Pi = mad(gm.re, gt.im, gm.im * gt.re);
    const R qr = R(1) + Pr;
    const R rq = scm::rcp_nr(mad(qr, qr, Pi * Pi));
    const R wr = qr * rq, wi = -Pi * rq;                      // 1/(1+P)
    o[0] = mad(gm.re, wr, -gm.im * wi);                      // SF
    o[1] = mad(gm.re, wi, gm.im * wr);
    o[2] = mad(gt.re, wr, -gt.im * wi);                      // X2
    o[3] = mad(gt.re, wi, gt.im * wr);
    o[4] = wi;                                               // SG/2 (doubled in rotate-back)
    o[5] = mad(Dn.x, gm.im - gt.im, -Dn.y * (gm.re + gt.re));   // SI
}

// the same six terms of a second energy, accumulated onto o (each sum rides on the last FMA of its term)
template <typename R>
__device__ __forceinline__ void node_terms_acc(cplx_t<R> gm, cplx_t<R> gt, typename VT<R>::V2 Dn, R (&o)[6]) {
    using scm::mad;
    const R Pr = mad(gm.re, gt.re, -gm.im * gt.im), Pi = mad(gm.re, gt.im, gm.im * gt.re);
    const R qr = R(1) + Pr;
    const R rq = scm::rcp_nr(mad(qr, qr, Pi * Pi));
    const R wr = qr * rq, wi = -Pi * rq;
    o[0] = mad(gm.re, wr, mad(-gm.im, wi, o[0]));
    o[1] = mad(gm.re, wi, mad(gm.im, wr, o[1]));
    o[2] = mad(gt.re, wr, mad(-gt.im, wi, o[2]));
    o[3] = mad(gt.re, wi, mad(gt.im, wr, o[3]));
    o[4] += wi;
    o[5] = mad(Dn.x, gm.im - gt.im, mad(-Dn.y, gm.re + gt.re, o[5]));
}

template <typename R, typename TAB>
__device__ __forceinline__ void march_round2(const MarchArgsT<R>& A, const WarpJob<R>& J, int n0) {
    using V2 = typename VT<R>::V2; using V4 = typename VT<R>::V4;
    constexpr int BYTES = 4 * (int)sizeof(R), ROW = 32 * BYTES;   // one entry = both energies' gamma~ of one node
    constexpr int PFROWS = RED_NODES / 2;
    const int lane = J.lane, nn = J.nn, ne = J.ne;
    char* const scr = J.scr_w + lane * BYTES;
    const bool pf_lane = lane * 128 < PFROWS * ROW;
    const int na = n0 + lane, nb = n0 + 32 + lane;             // both < ne (whole double rounds only)
    TAB ta, tb; ta.load(A.E, na); tb.load(A.E, nb);
    const R zia = (R)A.E.zi[na], zib = (R)A.E.zi[nb];
    const int pa = A.E.partner[na], pb = A.E.partner[nb];
    const V4* __restrict__ PC = J.PC; const V2* __restrict__ ND = J.ND;
    V4* const pcb = J.pcb; V2* const ndb = J.ndb;
    const int npart = nn * RED_VALS;

    // ---------------- pass 1: gamma-tilde from u_out down to u_in ----------------
    const int ctop = nn >> 5;
    if (ctop * CHUNK + lane <= nn) cp_async<sizeof(V4)>(pcb + (ctop & 1) * CHUNK + lane, PC + ctop * CHUNK + lane);
    cp_commit();
    cplx_t<R> gta, gtb;
    if (A.bc_mode == 1) {
        const V4 c4 = ldu(PC + nn);
        gta = hom_start<R>(-(double)c4.x, c4.y, A.E.zr[na] + c4.z, A.E.zi[na]);
        gtb = hom_start<R>(-(double)c4.x, c4.y, A.E.zr[nb] + c4.z, A.E.zi[nb]);
    } else if (A.ga_n[J.dB]) {
        const cplx_t<R> sa = gather_start(A, J.dB, pa), sb = gather_start(A, J.dB, pb);
        gta = mk(sa.re, -sa.im); gtb = mk(sb.re, -sb.im);
    } else {
        const cplx_t<R> sa = hom_start<R>(A.fb_D[J.dB].x, A.fb_D[J.dB].y, A.E.zr[pa] + A.fb_a[J.dB], A.E.zi[pa]);
        const cplx_t<R> sb = hom_start<R>(A.fb_D[J.dB].x, A.fb_D[J.dB].y, A.E.zr[pb] + A.fb_a[J.dB], A.E.zi[pb]);
        gta = mk(sa.re, -sa.im); gtb = mk(sb.re, -sb.im);
    }
    cplx_t<R> T0a = mk(R(0), R(0)), T0b = T0a;
    {
        char* e = scr + (size_t)((nn - 1) >> 1) * ROW;
        int p = nn;
        for (int c = ctop; c >= 0; --c) {
            if (c > 0) {
                cp_async<sizeof(V4)>(pcb + ((c - 1) & 1) * CHUNK + lane, PC + (c - 1) * CHUNK + lane);
                cp_commit();
                cp_wait<1>();
            } else {
                cp_wait<0>();
            }
            __syncwarp();
            const V4* __restrict__ buf = pcb + (c & 1) * CHUNK;
            const int plo = max(c * CHUNK, 1);
            if (p == nn) {                                      // exit piece (length l1); the last node is always spilled
                const V4 cc = buf[p & (CHUNK - 1)];
                const cplx_t<R> Ta = end_T<R>(cc, R(0), zia, J.len1), Tb = end_T<R>(cc, R(0), zib, J.len1);
                gta = scm::step_T(gta, -cc.x, cc.y, cc.z, zia, Ta);
                gtb = scm::step_T(gtb, -cc.x, cc.y, cc.z, zib, Tb);
                st_ent<true>(e, gta, gtb);
                e -= ROW; --p;
            }
            const V4* __restrict__ bp = buf + (p & (CHUNK - 1));
#pragma unroll 2
            for (; p >= plo; --p, --bp) {
                const V4 cc = *bp;
                const cplx_t<R> Ta = ta.fast(cc), Tb = tb.fast(cc);
                gta = scm::step_T(gta, -cc.x, cc.y, cc.z, zia, Ta);
                gtb = scm::step_T(gtb, -cc.x, cc.y, cc.z, zib, Tb);
                if (!(p & 1)) { st_ent<true>(e, gta, gtb); e -= ROW; }      // landed on the odd node p-1: row (p-1)>>1
            }
            if (c == 0) {                                       // entry piece (length l0)
                const V4 cc = buf[0];
                T0a = end_T<R>(cc, R(0), zia, J.len0); T0b = end_T<R>(cc, R(0), zib, J.len0);
                gta = scm::step_T(gta, -cc.x, cc.y, cc.z, zia, T0a);
                gtb = scm::step_T(gtb, -cc.x, cc.y, cc.z, zib, T0b);
            }
            __syncwarp();
        }
        A.store_new[(size_t)J.dB * ne + pa] = mk2(gta.re, -gta.im);
        A.store_new[(size_t)J.dB * ne + pb] = mk2(gtb.re, -gtb.im);
    }

    // ---------------- pass 2: gamma from u_in up to u_out; products and energy reduction ------------
    const int nchunk = (nn + CHUNK - 1) >> 5;
    cplx_t<R> ga, gb;
    {
        const V4 c0 = pcb[0];
        __syncwarp();
        if (lane < nn) {
            cp_async<sizeof(V4)>(pcb + CHUNK + lane, PC + 1 + lane);
            cp_async<sizeof(V2)>(ndb + CHUNK + lane, ND + lane);
        }
        cp_commit();
        if (A.bc_mode == 1) {
            ga = hom_start<R>(c0.x, c0.y, A.E.zr[na] + c0.z, A.E.zi[na]);
            gb = hom_start<R>(c0.x, c0.y, A.E.zr[nb] + c0.z, A.E.zi[nb]);
        } else if (A.ga_n[J.dF]) {
            ga = gather_start(A, J.dF, na); gb = gather_start(A, J.dF, nb);
        } else {
            ga = hom_start<R>(A.fb_D[J.dF].x, A.fb_D[J.dF].y, A.E.zr[na] + A.fb_a[J.dF], A.E.zi[na]);
            gb = hom_start<R>(A.fb_D[J.dF].x, A.fb_D[J.dF].y, A.E.zr[nb] + A.fb_a[J.dF], A.E.zi[nb]);
        }
        ga = scm::step_T(ga, c0.x, c0.y, c0.z, zia, T0a);
        gb = scm::step_T(gb, c0.x, c0.y, c0.z, zib, T0b);
    }
    const char* e = scr;                         // entry of nodes 0 / 1
    for (int q = RED_NODES; q < PF_DIST && q < nn; q += RED_NODES)
        if (pf_lane) prefetch_l2(J.scr_w + (size_t)(q >> 1) * ROW + lane * 128);
    // {gt_a, gt_b} of the next two spilled nodes: E0 serves nodes 4i, 4i+1, E1 nodes 4i+2, 4i+3, each reloaded (two entries ahead) once
    // its pair is done, so that neither the entries nor the gamma~ of the odd node are ever copied between registers
    Ent<R> E0 = ld_ent<true>(e, R(0)), E1 = ld_ent<true>(e + ROW, R(0));
    double part_nxt = 0.0;
    if (n0 && lane < RED_NODES * RED_VALS && lane < npart) part_nxt = J.PART[lane];
    int m = 0;
    auto node = [&](int b, const V4* pbuf, const V2* dbuf, bool exitp, const Ent<R>& E) {
        const V4 cc = pbuf[b]; const V2 dc = dbuf[b];
        const R len = exitp ? J.len1 : J.hlen;
        const cplx_t<R> Ta = exitp ? end_T<R>(cc, R(0), zia, len) : ta.fast(cc);
        const cplx_t<R> Tb = exitp ? end_T<R>(cc, R(0), zib, len) : tb.fast(cc);
        cplx_t<R> ha = mk(E.tr, E.ti), hb = mk(E.gr, E.gi);      // entry (m+b)>>1: gamma~ of the odd node m+b | 1, or of the last node itself
        if (!(b & 1) && !exitp) {                                 // even node: one step down from the odd node above it
            ha = scm::step_T(ha, -cc.x, cc.y, cc.z, zia, Ta);
            hb = scm::step_T(hb, -cc.x, cc.y, cc.z, zib, Tb);
        }
        R sa[6];
        node_terms<R>(ga, ha, dc, sa); node_terms_acc<R>(gb, hb, dc, sa);
        R* st = J.stage + b * RED_VALS * STAGE_LD + lane;
#pragma unroll
        for (int v = 0; v < 6; ++v) st[v * STAGE_LD] = sa[v];
        ga = scm::step_T(ga, cc.x, cc.y, cc.z, zia, Ta);
        gb = scm::step_T(gb, cc.x, cc.y, cc.z, zib, Tb);
    };
    for (int c = 0; c < nchunk; ++c) {
        const int bsel = (c + 1) & 1;
        if (c + 1 < nchunk) {
            const int q = (c + 1) * CHUNK + lane;
            if (q < nn) {
                cp_async<sizeof(V4)>(pcb + (bsel ^ 1) * CHUNK + lane, PC + 1 + q);
                cp_async<sizeof(V2)>(ndb + (bsel ^ 1) * CHUNK + lane, ND + q);
            }
            cp_commit();
            cp_wait<1>();
        } else {
            cp_wait<0>();
        }
        __syncwarp();
        const V4* __restrict__ pbuf = pcb + bsel * CHUNK;
        const V2* __restrict__ dbuf = ndb + bsel * CHUNK;
        const int mhi = min(nn, (c + 1) * CHUNK);
        const int mfull = min(mhi, nn - 1);                     // the last batch goes through the tail code (see march_round)
        for (; m + RED_NODES <= mfull; m += RED_NODES) {
            if (pf_lane && m + PF_DIST < nn) prefetch_l2(J.scr_w + (size_t)((m + PF_DIST) >> 1) * ROW + lane * 128);
            const double part_old = part_nxt;
            if (n0 && lane < RED_NODES * RED_VALS && (m + RED_NODES) * RED_VALS + lane < npart)
                part_nxt = J.PART[(m + RED_NODES) * RED_VALS + lane];
            const V4* __restrict__ pb = pbuf + (m & (CHUNK - 1)); const V2* __restrict__ db = dbuf + (m & (CHUNK - 1));
            static_assert(RED_NODES == 4, "two pairs of nodes per block");
            node(0, pb, db, false, E0); node(1, pb, db, false, E0);
            E0 = ld_ent<true>(e + 2 * ROW, R(0));
            node(2, pb, db, false, E1); node(3, pb, db, false, E1);
            E1 = ld_ent<true>(e + 3 * ROW, R(0));
            e += PFROWS * ROW;
            __syncwarp();
            if (lane < RED_NODES * RED_VALS) {
                double s = stage_colsum(J.stage, lane);
                if (n0) s += part_old;
                J.PART[m * RED_VALS + lane] = s;
            }
            __syncwarp();
        }
        if (m < mhi) {                                       // the last 1..4 nodes of the trajectory (last chunk only)
            const int rem = mhi - m;
            const double part_old = part_nxt;
            const V4* __restrict__ pb = pbuf + (m & (CHUNK - 1)); const V2* __restrict__ db = dbuf + (m & (CHUNK - 1));
#pragma unroll 1
            for (int b = 0; b < rem - 1; ++b) node(b, pb, db, false, b < 2 ? E0 : E1);
            node(rem - 1, pb, db, true, rem <= 2 ? E0 : E1);     // m + rem == nn: the exit piece, with its own length
            __syncwarp();
            if (lane < rem * RED_VALS) {
                double s = stage_colsum(J.stage, lane);
                if (n0) s += part_old;
                J.PART[m * RED_VALS + lane] = s;
            }
            __syncwarp();
            m = mhi;
        }
        __syncwarp();
    }
    A.store_new[(size_t)J.dF * ne + na] = mk2(ga.re, ga.im);
    A.store_new[(size_t)J.dF * ne + nb] = mk2(gb.re, gb.im);
}

// The plain Matsubara sweep (MODE 0, closed-form step, imaginary-axis energies, unit weights, no stats) marches two
// energies per lane (march_round2, with the pole-free or the pole-subtracted table).  Like every other instantiation it is
// compiled for two CTAs of 8 warps per SM (128 registers per thread: the node loops hold no spill; left alone the compiler
// takes 240 registers to hoist loads, and four warps per scheduler hide that latency better — fp64 1.6 %, fp32 9 % faster).
template <int MODE, bool STATS, int STEP, int TM, bool UW> constexpr bool kTwoEnergies = MODE == 0 && !STATS && STEP == 0 && TM == 1 && UW;
template <int MODE, bool STATS, int STEP, int TM, bool UW> constexpr int kMarchCtasPerSm = MARCH_MIN_CTAS;
template <int MODE, bool STATS, int STEP, typename R, int TM, bool UW = false>
__global__ void __launch_bounds__(MARCH_WARPS * 32, (kMarchCtasPerSm<MODE, STATS, STEP, TM, UW>)) march_kernel(MarchArgsT<R> A) {
    using V2 = typename VT<R>::V2; using V4 = typename VT<R>::V4;
    extern __shared__ double4 smem_raw[];
    WarpJob<R> J;
    J.lane = threadIdx.x & 31;
    const int wib = threadIdx.x >> 5, slot = blockIdx.x * MARCH_WARPS + wib;
    char* const smem_w = reinterpret_cast<char*>(smem_raw) + wib * (march_stage_bytes<R>() + march_coef_bytes<R>());
    J.stage = reinterpret_cast<R*>(smem_w);                                        // [4 nodes][6 values][33]
    J.pcb = reinterpret_cast<V4*>(smem_w + march_stage_bytes<R>());               // [2][CHUNK] piece records
    J.ndb = reinterpret_cast<V2*>(J.pcb + 2 * CHUNK);                             // [2][CHUNK] node Delta
    J.scr_w = A.scr + (size_t)slot * A.scr_stride;
    J.ne = A.E.ne; J.hlen = (R)A.h;
    R max2 = R(0);
    unsigned long long nst = 0, npl = 0;

    for (;;) {
        int item = 0;
        if (J.lane == 0) item = atomicAdd(A.counter, 1);
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= A.n_items) break;
        const int g = A.order[item];
        J.nn = A.T.nn[g]; J.noff = A.T.noff[g];
        J.dF = A.T.dF[g]; J.dB = A.T.dB[g];
        J.len0 = (R)A.T.l0[g]; J.len1 = (R)A.T.l1[g];
        J.ND = A.nd_D + J.noff; J.PC = A.pc + J.noff + g;
        J.PART = A.part + (size_t)J.noff * RED_VALS;
        const float2 pm = A.pmax[g];

        for (int n0 = 0; n0 < J.ne; n0 += 32) {
            if constexpr (kTwoEnergies<MODE, STATS, STEP, TM, UW>) {
                // a whole double round inside the pole-free table: both energies of every lane in one pass
                if (n0 + 64 <= J.ne) {
                    const int na = n0 + J.lane, nb = n0 + 32 + J.lane;
                    if (!__any_sync(0xffffffffu, !TTab<R, 1>::covers(A.E, na, pm) || !TTab<R, 1>::covers(A.E, nb, pm))) {
                        march_round2<R, TTab<R, 1>>(A, J, n0);
                        n0 += 32;
                        continue;
                    }
                    // beyond the pole-free table but inside the pole-subtracted one: the same double round with that table
                    using Short = TTabPole<R, scm::TaylorPoleShortK<R>>;
                    if (!__any_sync(0xffffffffu, !Short::covers(A.E, na, pm) || !Short::covers(A.E, nb, pm))) {
                        march_round2<R, Short>(A, J, n0);
                        npl += (unsigned long long)(J.nn + 1) * 64;
                        n0 += 32;
                        continue;
                    }
                }
            }
            const int n = min(n0 + J.lane, J.ne - 1);
            // STEP 0: T is re-evaluated in pass 2 if every piece is inside a table's radius for all 32 lanes, else spilled
            if (STEP == 0 && __any_sync(0xffffffffu, !TTab<R, TM>::covers(A.E, n, pm))) {
                if constexpr (TM == 1) {
                    using Short = TTabPole<R, scm::TaylorPoleShortK<R>>;
                    if (!__any_sync(0xffffffffu, !Short::covers(A.E, n, pm))) {
                        Short tab; tab.load(A.E, n);
                        march_round<MODE, STATS, STEP, R, false, UW>(A, J, tab, n0, max2);
                        npl += (unsigned long long)(J.nn + 1) * min(32, J.ne - n0);
                    } else {
                        TTabPole<R, scm::TaylorPoleK<R>> tab; tab.load(A.E, n);
                        march_round<MODE, STATS, STEP, R, true, UW>(A, J, tab, n0, max2);
                        nst += (unsigned long long)(J.nn + 1) * min(32, J.ne - n0);
                    }
                } else {
                    TTab<R, TM> tab; tab.load(A.E, n);
                    march_round<MODE, STATS, STEP, R, true, UW>(A, J, tab, n0, max2);
                    nst += (unsigned long long)(J.nn + 1) * min(32, J.ne - n0);
                }
            } else {
                TTab<R, TM> tab;
                if (STEP == 0) tab.load(A.E, n);
                march_round<MODE, STATS, STEP, R, false, UW>(A, J, tab, n0, max2);
            }
        }
    }
    if (STATS) {
        double mx = (double)max2;
#pragma unroll
        for (int o = 16; o; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        if (J.lane == 0) A.stat_max2[slot] = mx;
    }
    if (J.lane == 0 && nst) atomicAdd(A.n_stored, nst);
    if (J.lane == 0 && npl) atomicAdd(A.n_stored + 1, npl);
}

// ------------------------------------------------------------------------------------------------
// a6 + a7: rotate back, sum over angles, finalise
// ------------------------------------------------------------------------------------------------
struct BackArgs {
    GridDev G;
    int nphi, nrot; double c;
    const double* vx; const double* vy; const double* eta /*[ncomp][nphi]*/; const double* W;
    const int* line_g;           // [pair][t] -> first physical trajectory on that lattice line, or -1
    const int* line_n;           // [pair][t] -> number of trajectories (inside intervals) on that line
    TrajDev T;
    const double* part;          // [node][6]
    double t; double D[MAX_COMP]; int sigma;      // D_G = ln(T/T_c^G) + sum_n w_n t/eps_n (Eq. 22 :144)
    double2* delta_new;          // [ncomp][ny][nx]
    double* jx; double* jy; double* feI;
    int* n_bad;
    double* raw;                 // non-null: write the 2 ncomp + 3 un-finalised accumulators [..][ny][nx] instead (energy-sharded
                                 // sweep): Re, Im of every component's numerator, then Jx, Jy, I
};

// weights of the (up to 4) valid lattice nodes around a grid point for pair p; returns count
__device__ __forceinline__ int back_weights(const BackArgs& B, int p, double x, double y, long long node[4], double w[4]) {
    const double cx = B.vx[p], cy = B.vy[p];
    const double uu = (x * cx + y * cy) / B.G.h + B.c, ww = (-x * cy + y * cx) / B.G.h + B.c;
    const int j0 = (int)floor(uu), t0 = (int)floor(ww);
    const double fu = uu - j0, fw = ww - t0;
    const int* lg = B.line_g + (size_t)p * B.nrot;
    const int* ln = B.line_n + (size_t)p * B.nrot;
    int n = 0; double sw = 0.0;
#pragma unroll
    for (int b = 0; b < 2; ++b) {
        const int tt = t0 + b;
        if (tt < 0 || tt >= B.nrot) continue;
        const int g0 = lg[tt];
        if (g0 < 0) continue;
        for (int g = g0; g < g0 + ln[tt]; ++g) {               // one interval unless the grain has holes / is concave
            const int jf = B.T.jf[g], nn = B.T.nn[g];
#pragma unroll
            for (int a = 0; a < 2; ++a) {
                const int jj = j0 + a;
                if (jj < jf || jj >= jf + nn) continue;
                const double wt = (a ? fu : 1.0 - fu) * (b ? fw : 1.0 - fw);
                node[n] = B.T.noff[g] + (jj - jf); w[n] = wt; sw += wt; ++n;
            }
        }
    }
    if (sw > 1e-12) { const double r = 1.0 / sw; for (int i = 0; i < n; ++i) w[i] *= r; return n; }
    double bd = 1e300; long long best = -1;
    for (int tt = t0 - 2; tt <= t0 + 3; ++tt) {
        if (tt < 0 || tt >= B.nrot) continue;
        const int g0 = lg[tt];
        if (g0 < 0) continue;
        for (int g = g0; g < g0 + ln[tt]; ++g) {
            const int jf = B.T.jf[g], nn = B.T.nn[g];
            for (int jj = j0 - 2; jj <= j0 + 3; ++jj) {
                if (jj < jf || jj >= jf + nn) continue;
                const double d = (uu - jj) * (uu - jj) + (ww - tt) * (ww - tt);
                if (d < bd) { bd = d; best = B.T.noff[g] + (jj - jf); }
            }
        }
    }
    if (best < 0) return 0;
    node[0] = best; w[0] = 1.0;
    return 1;
}

// 2-D thread tiles (BACK_TX x BACK_TY grid points): neighbouring points share lattice nodes, so a compact tile re-uses
// the gathered `part` lines in L1 instead of fetching them again from L2
constexpr int BACK_TX = 16, BACK_TY = 8;
__global__ void __launch_bounds__(BACK_TX * BACK_TY) rotate_back_kernel(BackArgs B) {
    const int i = blockIdx.x * BACK_TX + threadIdx.x, j = blockIdx.y * BACK_TY + threadIdx.y;
    if (i >= B.G.nx || j >= B.G.ny) return;
    const size_t q = (size_t)j * B.G.nx + i;
    const int nc = B.G.ncomp;
    double nr[MAX_COMP], ni[MAX_COMP], sjx = 0.0, sjy = 0.0, sI = 0.0;
#pragma unroll
    for (int c = 0; c < MAX_COMP; ++c) nr[c] = ni[c] = 0.0;
    if (B.G.mask[q]) {
        const double x = (i - 0.5 * (B.G.nx - 1)) * B.G.h, y = (j - 0.5 * (B.G.ny - 1)) * B.G.h;
        const int H = B.nphi / 2;
        for (int p = 0; p < H; ++p) {
            long long node[4]; double w[4];
            const int n = back_weights(B, p, x, y, node, w);
            if (n == 0) { atomicAdd(B.n_bad, 1); continue; }
            double f0 = 0, f1 = 0, f2 = 0, f3 = 0, f4 = 0, f5 = 0;
            for (int s = 0; s < n; ++s) {
                const double* v = B.part + (size_t)node[s] * RED_VALS;
                f0 = fma(w[s], v[0], f0); f1 = fma(w[s], v[1], f1); f2 = fma(w[s], v[2], f2);
                f3 = fma(w[s], v[3], f3); f4 = fma(w[s], v[4], f4); f5 = fma(w[s], v[5], f5);
            }
            // angle k = p: SF = (f0,f1), SG = f4, SI = f5;  angle k+H: SF = conj(X2) = (f2,-f3), SG' v' = SG v, SI' = SI
            const double Wk = B.W[p], Wk2 = B.W[p + H];
#pragma unroll
            for (int c = 0; c < MAX_COMP; ++c)
                if (c < nc) {                                 // projection on eta_G (real): Eq. 22 numerator of component G
                    const double ek = B.eta[(size_t)c * B.nphi + p], ek2 = B.eta[(size_t)c * B.nphi + p + H];
                    nr[c] += Wk * ek * f0 + Wk2 * ek2 * f2;
                    ni[c] += Wk * ek * f1 - Wk2 * ek2 * f3;
                }
            const double wj = 2.0 * (Wk + Wk2) * f4;        // f4 = sum of Im 1/(1+P); Im g = 2 Im 1/(1+P)
            sjx = fma(wj, B.vx[p], sjx); sjy = fma(wj, B.vy[p], sjy);
            sI += (Wk + Wk2) * f5;
        }
    }
    const size_t ng = (size_t)B.G.nx * B.G.ny;
    if (B.raw) {
#pragma unroll
        for (int c = 0; c < MAX_COMP; ++c) if (c < nc) { B.raw[(2 * c) * ng + q] = nr[c]; B.raw[(2 * c + 1) * ng + q] = ni[c]; }
        B.raw[(2 * nc) * ng + q] = sjx; B.raw[(2 * nc + 1) * ng + q] = sjy; B.raw[(2 * nc + 2) * ng + q] = sI;
        return;
    }
    // Delta_new = -2 i t Num / D (Eq. 22 with f = -2 pi i gamma/(1+P)); j = 2 sigma t J (Eq. 8); I = t I (Eq. 19)
    if (B.delta_new) {
#pragma unroll
        for (int c = 0; c < MAX_COMP; ++c) if (c < nc) { const double s = 2.0 * B.t / B.D[c]; B.delta_new[c * ng + q] = make_double2(s * ni[c], -s * nr[c]); }
    }
    if (B.jx) B.jx[q] = 2.0 * B.sigma * B.t * sjx;
    if (B.jy) B.jy[q] = 2.0 * B.sigma * B.t * sjy;
    if (B.feI) B.feI[q] = B.t * sI;
}

// a7 alone, after the accumulators of all energy shards have been summed
struct FinArgs { double D[MAX_COMP]; };
__global__ void finalise_kernel(size_t ng, int nc, const double* raw, double t, FinArgs F, int sigma,
                                double2* delta_new, double* jx, double* jy, double* feI) {
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= ng) return;
    if (delta_new)
        for (int c = 0; c < nc; ++c) { const double s = 2.0 * t / F.D[c]; delta_new[c * ng + q] = make_double2(s * raw[(2 * c + 1) * ng + q], -s * raw[(2 * c) * ng + q]); }
    if (jx) jx[q] = 2.0 * sigma * t * raw[(2 * nc) * ng + q];
    if (jy) jy[q] = 2.0 * sigma * t * raw[(2 * nc + 1) * ng + q];
    if (feI) feI[q] = t * raw[(2 * nc + 2) * ng + q];
}

// counts the non-finite values of a reduced field (SC_ERR_NUMERIC; only run when the caller asked for stats)
__global__ void nonfinite_kernel(size_t n, const double* a, int* count) {
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q < n && !isfinite(a[q])) atomicAdd(count, 1);
}

// LDOS rotate-back: thread per (grid point, energy); energies fastest so the gathers coalesce.
struct BackLdosArgs {
    BackArgs B;
    int ne_out; const int* out_idx;     // internal index of output energy m
    const int* partner;
    int ne;                             // internal energy count
    const double* ldos_nodes;           // [node][ne]
    double* out;                        // [ne_out][ny][nx]
    int p0, p1; int accumulate;         // pair range of this batch
};

__global__ void rotate_back_ldos_kernel(BackLdosArgs L) {
    const BackArgs& B = L.B;
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    const int i = blockIdx.y, j = blockIdx.z;
    if (m >= L.ne_out) return;
    const size_t q = (size_t)j * B.G.nx + i;
    double acc = 0.0;
    if (B.G.mask[q]) {
        const double x = (i - 0.5 * (B.G.nx - 1)) * B.G.h, y = (j - 0.5 * (B.G.ny - 1)) * B.G.h;
        const int H = B.nphi / 2;
        const int n1 = L.out_idx[m], n2 = L.partner[n1];
        for (int p = L.p0; p < L.p1; ++p) {
            long long node[4]; double w[4];
            const int n = back_weights(B, p, x, y, node, w);
            if (n == 0) { if (m == 0) atomicAdd(B.n_bad, 1); continue; }
            double a1 = 0.0, a2 = 0.0;
            for (int s = 0; s < n; ++s) {
                const double* v = L.ldos_nodes + (size_t)node[s] * L.ne;
                a1 = fma(w[s], v[n1], a1); a2 = fma(w[s], v[n2], a2);
            }
            // Re g(k, eps) = value at eps; Re g(k+H, eps) = value of angle k at the partner energy -eps
            acc += B.W[p] * a1 + B.W[p + H] * a2;
        }
        if (L.accumulate) acc += L.out[(size_t)m * B.G.nx * B.G.ny + q];
    }
    L.out[(size_t)m * B.G.nx * B.G.ny + q] = acc;
}

// ------------------------------------------------------------------------------------------------
// debug / measurement kernels
// ------------------------------------------------------------------------------------------------
// re-march one trajectory for one energy with the same device functions; writes gamma, gamma-tilde per node
template <typename R, int TM>
__device__ void debug_traj_body(const MarchArgsT<R>& A, int stepper, int g, int n, double2* outG, double2* outGT) {
    using V4 = typename VT<R>::V4;
    const int nn = A.T.nn[g];
    const V4* PC = A.pc + A.T.noff[g] + g;
    const int nb = A.E.partner[n];
    const R zr0 = (R)A.E.zr[n], zi0 = (R)A.E.zi[n];
    const int dF = A.T.dF[g], dB = A.T.dB[g];
    const R hlen = (R)A.h, len0 = (R)A.T.l0[g], len1 = (R)A.T.l1[g];
    cplx_t<R> gt;
    if (A.bc_mode == 1) gt = hom_start<R>(-(double)PC[nn].x, PC[nn].y, A.E.zr[n] + PC[nn].z, A.E.zi[n]);
    else if (A.ga_n[dB]) { cplx_t<R> s = gather_start(A, dB, nb); gt = mk(s.re, -s.im); }
    else { cplx_t<R> s = hom_start<R>(A.fb_D[dB].x, A.fb_D[dB].y, A.E.zr[nb] + A.fb_a[dB], A.E.zi[nb]); gt = mk(s.re, -s.im); }
    // a table evaluation of T as in the march (per-piece vote; the march's choice between the two tables of an
    // imaginary-axis energy depends on the other 31 lanes of its round, so this tap may take the other one: both are
    // accurate to rounding)
    TTab<R, TM> tab; tab.load(A.E, n);
    auto step = [&](cplx_t<R> x, R sgn, int p) {
        const R len = p == 0 ? len0 : (p == nn ? len1 : hlen);
        if (stepper == 1) return scm::step_mid(x, sgn * PC[p].x, PC[p].y, zr0 + PC[p].z, zi0, len);
        const cplx_t<R> T = p > 0 && p < nn ? tab.voted(PC[p], zr0, zi0, len) : end_T<R>(PC[p], zr0, zi0, len);
        return scm::step_T(x, sgn * PC[p].x, PC[p].y, zr0 + PC[p].z, zi0, T);
    };
    for (int p = nn; p >= 1; --p) { gt = step(gt, R(-1), p); outGT[p - 1] = make_double2(gt.re, gt.im); }
    cplx_t<R> gm;
    if (A.bc_mode == 1) gm = hom_start<R>(PC[0].x, PC[0].y, A.E.zr[n] + PC[0].z, A.E.zi[n]);
    else if (A.ga_n[dF]) gm = gather_start(A, dF, n);
    else gm = hom_start<R>(A.fb_D[dF].x, A.fb_D[dF].y, A.E.zr[n] + A.fb_a[dF], A.E.zi[n]);
    for (int p = 0; p < nn; ++p) { gm = step(gm, R(1), p); outG[p] = make_double2(gm.re, gm.im); }
}
template <typename R>
__global__ void debug_traj_kernel(MarchArgsT<R> A, int stepper, int g, int n, double2* outG, double2* outGT) {
    // a full warp runs the same trajectory and energy (the table evaluation votes across the warp); lane 0 writes
    if (blockIdx.x != 0 || threadIdx.x >= 32) return;
    if (A.E.tmode == 2) debug_traj_body<R, 2>(A, stepper, g, n, outG, outGT);
    else debug_traj_body<R, 1>(A, stepper, g, n, outG, outGT);
}

// max relative error of the math building blocks vs the CUDA library on pseudo-random arguments
__global__ void math_test_kernel(int n, double* err /*6*/) {
    double e[6] = {0, 0, 0, 0, 0, 0};
    unsigned long long s = 0x9E3779B97F4A7C15ull * (blockIdx.x * blockDim.x + threadIdx.x + 1);
    for (int i = 0; i < n; ++i) {
        s = s * 6364136223846793005ull + 1442695040888963407ull;
        const double u1 = (double)(s >> 11) * (1.0 / 9007199254740992.0);
        s = s * 6364136223846793005ull + 1442695040888963407ull;
        const double u2 = (double)(s >> 11) * (1.0 / 9007199254740992.0);
        const double x = exp(40.0 * (u1 - 0.5));                       // 2e-9 .. 5e8
        e[0] = fmax(e[0], fabs(scm::rcp_nr(x) * x - 1.0));
        e[1] = fmax(e[1], fabs(scm::rsqrt_nr(x) * sqrt(x) - 1.0));
        const double a = -30.0 * u2;                                    // exp argument
        double ex, xm1; scm::exp_pair(a, ex, xm1);
        e[2] = fmax(e[2], fabs(ex / exp(a) - 1.0));
        e[3] = fmax(e[3], fabs(xm1 / expm1(a) - 1.0));
        const double y = 1.5707963 * (u1 - 0.5);                        // |y| <= pi/4
        double sn, cm1; scm::sincos_small(y, sn, cm1);
        e[4] = fmax(e[4], fabs(sn - sin(y)) / fmax(fabs(sin(y)), 1e-300));
        const double sh = sin(0.5 * y), cref = -2.0 * sh * sh;              // cos y - 1 without cancellation
        e[5] = fmax(e[5], fabs(cm1 - cref) / fmax(fabs(cref), 1e-300));
    }
    for (int c = 0; c < 6; ++c) {
        double v = e[c];
        for (int o = 16; o; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
        if ((threadIdx.x & 31) == 0) atomicMax((unsigned long long*)&err[c], (unsigned long long)__double_as_longlong(v));
    }
}

// register-resident DFMA loop: 8 independent chains per thread
__global__ void fp64_peak_kernel(int iters, double* sink) {
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double b = 0.999999, c = 1e-7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
            a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
        }
    }
    const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 123.456) sink[0] = s;
}

// register-resident FFMA loop (fp32 pipe: the peak of the fp32 march), 8 independent chains per thread
__global__ void fp32_peak_kernel(int iters, float* sink) {
    float a0 = threadIdx.x * 1e-6f, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const float b = 0.9999f, c = 1e-4f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = fmaf(a0, b, c); a1 = fmaf(a1, b, c); a2 = fmaf(a2, b, c); a3 = fmaf(a3, b, c);
            a4 = fmaf(a4, b, c); a5 = fmaf(a5, b, c); a6 = fmaf(a6, b, c); a7 = fmaf(a7, b, c);
        }
    }
    const float s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 123.456f) sink[0] = s;
}
// MUFU issue rate (the "SFU" of north_star): the reciprocal seeds of the march are MUFU.RCP (fp32) / MUFU.RCP64H (fp64).
// 8 independent chains per thread of MUFU.RCP64H (F64) or MUFU.RSQ (fp32: same unit and rate as MUFU.RCP); the values stay finite.
template <bool F64>
__global__ void mufu_peak_kernel(int iters, float* sink) {
    float a[8]; double d[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) { a[u] = 1.5f + threadIdx.x * 1e-3f + u; d[u] = 1.5 + threadIdx.x * 1e-3 + u; }
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                if constexpr (F64) asm volatile("rcp.approx.ftz.f64 %0, %1;" : "=d"(d[u]) : "d"(d[u]));
                else asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(a[u]) : "f"(a[u]));     // (a chain of rcp.approx is folded away: 1/(1/x) = x)
            }
    }
    float s = 0.f;
#pragma unroll
    for (int u = 0; u < 8; ++u) s += F64 ? (float)d[u] : a[u];
    if (s == 123.456f) sink[0] = s;
}

}  // namespace sck
