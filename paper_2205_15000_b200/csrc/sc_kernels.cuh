// sc_kernels.cuh — sm_100a kernels of the Riccati sweep.
//
//   rotate_in_kernel     a2: Delta, A on the reference grid -> node coefficients on every trajectory
//   reset_store_kernel   R8: boundary stores := local homogeneous solution
//   march_kernel         a3+a4+a5: boundary gather, gamma-tilde down (stores T and gamma-tilde per node),
//                        gamma up (re-uses T), node products, reduction over energies
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

struct GridDev {
    int nx, ny; double h;
    const unsigned char* mask;
    const double2* delta; const double* Ax; const double* Ay;   // Ax/Ay may be null
};

struct TrajDev {                 // physical trajectories (angles k < N/2), struct of arrays
    int n;                       // count
    const int* k; const int* t; const int* jf; const int* nn;
    const double* l0; const double* l1;
    const long long* noff;       // first node in the node arrays
    const int* dF; const int* dB;   // store rows: (k,t) and its mirror (k+N/2, N_rot-1-t)
};

// tc: per-energy table of the step coefficient T (sc_math.cuh taylor_T), [ne][TC_LD] = r_0..r_8, (w0 + 9 wp)^2,
// w0 + wp, 2/h; null when the energy table is not on the imaginary axis (then every piece takes the exp-based evaluation)
constexpr int TC_LD = 12;
struct EnergyDev { int ne; const double* zr; const double* zi; const double* w; const int* partner; const double* tc; };

// ------------------------------------------------------------------------------------------------
// masked bilinear interpolation of Delta (R5) and plain bilinear of A at a point
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool interp_delta(const GridDev& G, double x, double y, double& dr, double& di) {
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
            if (G.mask[q]) { const double2 d = G.delta[q]; sw += w; ar += w * d.x; ai += w * d.y; }
        }
    if (sw > 1e-12) { dr = ar / sw; di = ai / sw; return true; }
    double bd = 1e300; int bi = -1, bj = -1;
    for (int jj = j0 - 2; jj <= j0 + 3; ++jj)
        for (int ii = i0 - 2; ii <= i0 + 3; ++ii) {
            if (ii < 0 || ii >= G.nx || jj < 0 || jj >= G.ny || !G.mask[(size_t)jj * G.nx + ii]) continue;
            const double d = (gx - ii) * (gx - ii) + (gy - jj) * (gy - jj);
            if (d < bd) { bd = d; bi = ii; bj = jj; }
        }
    if (bi < 0) { dr = di = 0.0; return false; }
    const double2 d = G.delta[(size_t)bj * G.nx + bi];
    dr = d.x; di = d.y;
    return true;
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
// coefficients the march consumes: piece p of a trajectory with nn nodes (p = 0..nn) is {Re De, Im De, a, length}
// with De, a the half-step values by linear interpolation and nearest-neighbour extrapolation at both ends
// (reading R4).  Piece records of trajectory g start at noff[g] + g.
template <typename R>
__global__ void rotate_in_kernel(GridDev G, TrajDev T, const double* vx, const double* vy, const double* eta,
                                 double c, int sigma, double2* nd_D, double* nd_a, typename VT<R>::V2* nd_Dr,
                                 typename VT<R>::V4* pc, int* n_bad) {
    const int g = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (g >= T.n) return;
    const int lane = threadIdx.x & 31;
    const int k = T.k[g];
    const double cx = vx[k], cy = vy[k], e = eta[k], w = (T.t[g] - c) * G.h;
    const int jf = T.jf[g], nn = T.nn[g];
    const long long off = T.noff[g];
    for (int m = lane; m < nn; m += 32) {
        const double u = (jf + m - c) * G.h;
        const double x = u * cx - w * cy, y = u * cy + w * cx;
        double dr, di;
        if (!interp_delta(G, x, y, dr, di)) atomicAdd(n_bad, 1);
        nd_D[off + m] = make_double2(e * dr, e * di);
        if (sizeof(R) == 4) nd_Dr[off + m] = mk2((R)(e * dr), (R)(e * di));      // fp32 mode: the march reads a float copy
        nd_a[off + m] = sigma * (cx * interp_plain(G, G.Ax, x, y) + cy * interp_plain(G, G.Ay, x, y));
    }
    __syncwarp();
    typename VT<R>::V4* P = pc + off + g;
    for (int p = lane; p <= nn; p += 32) {
        const int lo = p > 0 ? p - 1 : 0, hi = p < nn ? p : nn - 1;
        const double2 Dl = nd_D[off + lo], Dh = nd_D[off + hi];
        const double al = nd_a[off + lo], ah = nd_a[off + hi];
        const double len = p == 0 ? T.l0[g] : (p == nn ? T.l1[g] : G.h);
        P[p] = lo == hi ? mk4((R)Dl.x, (R)Dl.y, (R)al, (R)len)
                        : mk4((R)(0.5 * (Dl.x + Dh.x)), (R)(0.5 * (Dl.y + Dh.y)), (R)(0.5 * (al + ah)), (R)len);
    }
}

// fallback coefficients for boundary points that have no valid specular partner (R6 fallback):
// Delta(R_min) eta(mirrored direction) and sigma v_in . A(R_min)
__global__ void fallback_kernel(GridDev G, int nfb, const int* rows, const double* px, const double* py,
                                const double* dx, const double* dy, const double* eta_m, int sigma,
                                double2* fb_D, double* fb_a) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nfb) return;
    double dr, di;
    interp_delta(G, px[i], py[i], dr, di);
    fb_D[rows[i]] = make_double2(eta_m[i] * dr, eta_m[i] * di);
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
    const V4* pc;                           // piece coefficients {Re De, Im De, a, len} [node + g]
    int bc_mode;
    const int* ga_idx; const double* ga_w; const unsigned char* ga_n;   // entry gathers per store row [row][4]
    const double2* fb_D; const double* fb_a;
    const V2* store_old; V2* store_new;
    char* scr; long long scr_stride;        // per warp slot: scr_stride bytes = (smax+2) rows of 32 entries
    double* part;                           // MODE 0: [node][6] = SF.re, SF.im, X2.re, X2.im, SG, SI
    double* ldos;                           // MODE 1: [node][ne] = Re g_n
    int* counter;
    double* stat_max2;                      // per warp slot: max |gamma|^2 seen (optional)
};
using MarchArgs = MarchArgsT<double>;

constexpr int MARCH_WARPS = 8;               // warps per CTA
#ifndef SC_MARCH_MIN_CTAS
#define SC_MARCH_MIN_CTAS 2
#endif
constexpr int MARCH_MIN_CTAS = SC_MARCH_MIN_CTAS;   // resident CTAs per SM the fp64 register budget is sized for
constexpr int PF_DIST = 12;                  // pass 2: scratch lines are pulled into L2 this many nodes ahead
#ifndef SC_PF1_DIST
#define SC_PF1_DIST 0
#endif
constexpr int PF1_DIST = SC_PF1_DIST;        // ... and into L1 this many nodes ahead (0: off); the register look-ahead is one node
constexpr int RED_NODES = 4;                 // nodes per shared-memory reduction batch
constexpr int RED_VALS = 6;
constexpr int STAGE_LD = 33;                 // padded row of the transpose stage: conflict-free rows AND columns

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
// 256-bit global accesses (LDG.E.ENL2.256 / STG.E.ENL2.256 on sm_100a): one fp64 scratch entry per lane per instruction
__device__ __forceinline__ double4 ld256(const double4* p) {
    double4 v;
    asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ void st256(double4* p, double a, double b, double c, double d) {
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}
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
template <int MODE, bool STATS, typename R>
__device__ __forceinline__ R node_products(cplx_t<R> gm, R gtr, R gti, typename VT<R>::V2 Dn, R wn, R* st, R& max2) {
    using scm::mad;
    const R Pr = mad(gm.re, gtr, -gm.im * gti), Pi = mad(gm.re, gti, gm.im * gtr);
    const R qr = R(1) + Pr;
    const R rq = scm::rcp_nr(mad(qr, qr, Pi * Pi));
    const R ir = qr * rq, ii = -Pi * rq;               // 1/(1+P)
    if (STATS) max2 = scm::maxr(max2, scm::maxr(mad(gm.re, gm.re, gm.im * gm.im), mad(gtr, gtr, gti * gti)));
    if (MODE == 0) {
        const R wr = wn * ir, wi = wn * ii;
        st[0 * STAGE_LD] = mad(gm.re, wr, -gm.im * wi);      // SF  = w gamma/(1+P)
        st[1 * STAGE_LD] = mad(gm.re, wi, gm.im * wr);
        st[2 * STAGE_LD] = mad(gtr, wr, -gti * wi);          // X2  = w gamma~/(1+P)  (SF of k+N/2 = conj)
        st[3 * STAGE_LD] = mad(gtr, wi, gti * wr);
        st[4 * STAGE_LD] = R(2) * wi;                        // SG  = w Im g = 2 w Im 1/(1+P)
        st[5 * STAGE_LD] = wn * mad(Dn.x, gm.im - gti, -Dn.y * (gm.re + gtr));   // SI (Eq. 19 :128 numerator)
    }
    return mad(R(2), ir, R(-1));                             // Re g = 2 Re 1/(1+P) - 1
}

// column sums of the stage: lane c < cnt sums row c over the 32 lanes (4 partial sums, fixed order)
template <typename R>
__device__ __forceinline__ double stage_colsum(const R* stage, int lane) {
    const R* col = stage + lane * STAGE_LD;
    R s0 = R(0), s1 = R(0), s2 = R(0), s3 = R(0);
#pragma unroll
    for (int i = 0; i < 32; i += 4) { s0 += col[i]; s1 += col[i + 1]; s2 += col[i + 2]; s3 += col[i + 3]; }
    return (double)((s0 + s1) + (s2 + s3));
}

// Scratch entry of one (piece, lane): STEP 0 (closed form) {T.re, T.im, gt.re, gt.im} = 4 R, one 256-bit (fp64) or
// 128-bit (fp32) access; STEP 1 (mid-point) {gt.re, gt.im} = 2 R.  A warp's 32 entries of a piece are contiguous.
template <typename R> struct Ent { R tr, ti, gr, gi; };
template <typename R, int STEP> struct ScrT {
    static constexpr int BYTES = (STEP == 0 ? 4 : 2) * (int)sizeof(R); static constexpr int ROW = 32 * BYTES;
};
template <int STEP>
__device__ __forceinline__ Ent<double> ld_ent(const char* p, double) {
    Ent<double> e;
    if (STEP == 0) { const double4 v = ld256((const double4*)p); e.tr = v.x; e.ti = v.y; e.gr = v.z; e.gi = v.w; }
    else {
        asm volatile("ld.global.v2.f64 {%0,%1}, [%2];" : "=d"(e.gr), "=d"(e.gi) : "l"(p));
        e.tr = e.ti = 0.0;
    }
    return e;
}
template <int STEP>
__device__ __forceinline__ Ent<float> ld_ent(const char* p, float) {
    Ent<float> e;
    if (STEP == 0) asm volatile("ld.global.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(e.tr), "=f"(e.ti), "=f"(e.gr), "=f"(e.gi) : "l"(p));
    else {
        asm volatile("ld.global.v2.f32 {%0,%1}, [%2];" : "=f"(e.gr), "=f"(e.gi) : "l"(p));
        e.tr = e.ti = 0.f;
    }
    return e;
}
template <int STEP>
__device__ __forceinline__ void st_ent(char* p, cplx T, cplx gt) {
    if (STEP == 0) st256((double4*)p, T.re, T.im, gt.re, gt.im);
    else asm volatile("st.global.v2.f64 [%0], {%1,%2};" ::"l"(p), "d"(gt.re), "d"(gt.im) : "memory");
}
template <int STEP>
__device__ __forceinline__ void st_ent(char* p, cplxf T, cplxf gt) {
    if (STEP == 0) asm volatile("st.global.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(T.re), "f"(T.im), "f"(gt.re), "f"(gt.im) : "memory");
    else asm volatile("st.global.v2.f32 [%0], {%1,%2};" ::"l"(p), "f"(gt.re), "f"(gt.im) : "memory");
}
// one step of gamma with piece record cc; STEP 0 re-uses the stored T of the piece
template <int STEP, typename R>
__device__ __forceinline__ cplx_t<R> step_up(cplx_t<R> g, const typename VT<R>::V4& cc, R zr0, R zi0, const Ent<R>& E) {
    if (STEP == 0) return scm::step_T(g, cc.x, cc.y, zr0 + cc.z, zi0, mk(E.tr, E.ti));
    return scm::step_mid(g, cc.x, cc.y, zr0 + cc.z, zi0, cc.w);
}

// ---- coefficient staging: the warp-uniform piece / node records of a trajectory are streamed through shared
// memory in chunks of 32 (one record per lane, coalesced cp.async, double-buffered one chunk ahead), so that no
// step ever waits on a global load of its coefficients; the step loop reads them with broadcast LDS.
constexpr int CHUNK = 32;
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

// MODE 0: Matsubara sums; 1: per-energy Re g (LDOS); 2: boundary values only.
// STEP 0: closed-form step; 1: implicit mid-point rule (C4-C9 :984-1001).
template <int MODE, bool STATS, int STEP, typename R>
__global__ void __launch_bounds__(MARCH_WARPS * 32, MARCH_MIN_CTAS) march_kernel(MarchArgsT<R> A) {
    using V2 = typename VT<R>::V2; using V4 = typename VT<R>::V4;
    extern __shared__ double4 smem_raw[];
    constexpr int ROW = ScrT<R, STEP>::ROW, BYTES = ScrT<R, STEP>::BYTES;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int slot = blockIdx.x * MARCH_WARPS + wib;
    char* const smem_w = reinterpret_cast<char*>(smem_raw) + wib * (march_stage_bytes<R>() + march_coef_bytes<R>());
    R* const stage = reinterpret_cast<R*>(smem_w);                                        // [4 nodes][6 values][33]
    V4* const pcb = reinterpret_cast<V4*>(smem_w + march_stage_bytes<R>());               // [2][CHUNK] piece records
    V2* const ndb = reinterpret_cast<V2*>(pcb + 2 * CHUNK);                               // [2][CHUNK] node Delta
    char* const scr = A.scr + (size_t)slot * A.scr_stride + lane * BYTES;   // entry e of this lane: scr + e*ROW
    const int ne = A.E.ne;
    R max2 = R(0);

    for (;;) {
        int item = 0;
        if (lane == 0) item = atomicAdd(A.counter, 1);
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= A.n_items) break;
        const int g = A.order[item];
        const int nn = A.T.nn[g];
        const long long noff = A.T.noff[g];
        const int dF = A.T.dF[g], dB = A.T.dB[g];
        const V2* __restrict__ ND = A.nd_D + noff;
        const V4* __restrict__ PC = A.pc + noff + g;
        double* __restrict__ const PART = A.part + (size_t)noff * RED_VALS;
        const int npart = nn * RED_VALS;

        for (int n0 = 0; n0 < ne; n0 += 32) {
            const bool act = n0 + lane < ne;
            const int n = act ? n0 + lane : ne - 1;
            const R zr0 = (R)A.E.zr[n], zi0 = (R)A.E.zi[n];
            const R wn = act ? (R)A.E.w[n] : R(0);
            const int nb = A.E.partner[n];
            // Taylor table of T about this lane's energy (interior pieces all have length h)
            constexpr int KT = scm::TaylorK<R>::K;
            const bool tay = STEP == 0 && A.E.tc != nullptr;
            R tcf[KT + 1]; R thr2 = R(-1), pole_a = R(1), pole_res = R(0);
            if (tay) {
#pragma unroll
                for (int k = 0; k <= KT; ++k) tcf[k] = (R)A.E.tc[(size_t)n * TC_LD + k];
                thr2 = (R)(A.E.tc[(size_t)n * TC_LD + 9] * scm::TaylorK<R>::RMAX2);
                pole_a = (R)A.E.tc[(size_t)n * TC_LD + 10]; pole_res = (R)A.E.tc[(size_t)n * TC_LD + 11];
            }
            const R m2zi = R(-2) * zi0;

            // ---------------- pass 1: gamma-tilde from u_out down to u_in; entry p = {T_p, gamma~(node p-1)} ----------
            const int ctop = nn >> 5;                                  // chunk c holds pieces 32c .. 32c+31
            if (ctop * CHUNK + lane <= nn) cp_async<sizeof(V4)>(pcb + (ctop & 1) * CHUNK + lane, PC + ctop * CHUNK + lane);
            cp_commit();
            cplx_t<R> gt;
            if (A.bc_mode == 1) {
                const V4 c4 = ldu(PC + nn);
                gt = hom_start<R>(-(double)c4.x, c4.y, A.E.zr[n] + c4.z, A.E.zi[n]);
            } else if (A.ga_n[dB]) {
                const cplx_t<R> s = gather_start(A, dB, nb);            // gamma of the mirrored trajectory at its entry
                gt = mk(s.re, -s.im);
            } else {
                const cplx_t<R> s = hom_start<R>(A.fb_D[dB].x, A.fb_D[dB].y, A.E.zr[nb] + A.fb_a[dB], A.E.zi[nb]);
                gt = mk(s.re, -s.im);
            }
            {
                char* e = scr + (size_t)nn * ROW;
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
                    const int plo = c * CHUNK;
#pragma unroll 2
                    for (; p >= plo; --p) {
                        const V4 cc = buf[p & (CHUNK - 1)];
                        const R zr = zr0 + cc.z;
                        cplx_t<R> T = mk(R(0), R(0));
                        if (STEP == 0) {
                            const R d2 = scm::mad(cc.x, cc.x, cc.y * cc.y);
                            // w = |De|^2 - z^2 = zi0^2 + dw,  dw = (|De|^2 - a^2) - 2 i zi0 a   (z = i zi0 + a)
                            const R dwr = scm::mad(-cc.z, cc.z, d2), dwi = m2zi * cc.z;
                            const R s2 = scm::mad(dwr, dwr, dwi * dwi);
                            const bool interior = p > 0 && p < nn;
                            if (interior && !__any_sync(0xffffffffu, !(s2 <= thr2))) T = scm::taylor_T<R, KT>(tcf, pole_a, pole_res, dwr, dwi, s2);
                            else T = scm::coef_T_slow(d2, zr, zi0, cc.w);
                            gt = scm::step_T(gt, -cc.x, cc.y, zr, zi0, T);
                        } else {
                            gt = scm::step_mid(gt, -cc.x, cc.y, zr, zi0, cc.w);
                        }
                        st_ent<STEP>(e, T, gt);
                        e -= ROW;
                    }
                    __syncwarp();                                       // chunk c is free for the load issued next round
                }
                if (act) A.store_new[(size_t)dB * ne + nb] = mk2(gt.re, -gt.im);
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
                else if (A.ga_n[dF]) gm = gather_start(A, dF, n);
                else gm = hom_start<R>(A.fb_D[dF].x, A.fb_D[dF].y, A.E.zr[n] + A.fb_a[dF], A.E.zi[n]);
                const Ent<R> e0 = ld_ent<STEP>(scr, R(0));
                gm = step_up<STEP, R>(gm, c0, zr0, zi0, e0);
            }
            const char* e = scr + ROW;                  // entry of node 0
            for (int q = 4; q < PF_DIST && q < nn; q += 4) prefetch_l2(e - lane * BYTES + (size_t)q * ROW + lane * 128);
            Ent<R> En = ld_ent<STEP>(e, R(0));
            double part_nxt = 0.0;                       // running sums of the earlier energy rounds, fetched one batch ahead
            if (MODE == 0 && n0 && lane < RED_NODES * RED_VALS && lane < npart) part_nxt = PART[lane];
            int m = 0;
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
                for (; m + RED_NODES <= mhi; m += RED_NODES) {
                    if (m + PF_DIST < nn) prefetch_l2(e - lane * BYTES + (size_t)PF_DIST * ROW + lane * 128);
                    if (PF1_DIST && m + PF1_DIST < nn) prefetch_l1(e - lane * BYTES + (size_t)PF1_DIST * ROW + lane * 128);
                    const double part_old = part_nxt;
                    if (MODE == 0 && n0 && lane < RED_NODES * RED_VALS && (m + RED_NODES) * RED_VALS + lane < npart)
                        part_nxt = PART[(m + RED_NODES) * RED_VALS + lane];
#pragma unroll
                    for (int b = 0; b < RED_NODES; ++b) {
                        const Ent<R> Ec = En;
                        const V4 cc = pbuf[(m + b) & (CHUNK - 1)]; const V2 dc = dbuf[(m + b) & (CHUNK - 1)];
                        En = ld_ent<STEP>(e + (b + 1) * ROW, R(0));          // one node ahead (scratch has 2 spare entries)
                        if (MODE != 2) {
                            const R rg = node_products<MODE, STATS, R>(gm, Ec.gr, Ec.gi, dc, wn, stage + b * RED_VALS * STAGE_LD + lane, max2);
                            if (MODE == 1 && act) A.ldos[(size_t)(noff + m + b) * ne + n] = (double)rg;
                        }
                        gm = step_up<STEP, R>(gm, cc, zr0, zi0, Ec);
                    }
                    e += RED_NODES * ROW;
                    if (MODE == 0) {
                        __syncwarp();
                        if (lane < RED_NODES * RED_VALS) {
                            double s = stage_colsum(stage, lane);
                            if (n0) s += part_old;
                            PART[m * RED_VALS + lane] = s;
                        }
                        __syncwarp();
                    }
                }
                if (m < mhi) {                                       // ragged tail: 1..3 nodes (last chunk only)
                    const int rem = mhi - m;
                    const double part_old = part_nxt;
                    for (int b = 0; b < rem; ++b) {
                        const Ent<R> Ec = En;
                        const V4 cc = pbuf[(m + b) & (CHUNK - 1)]; const V2 dc = dbuf[(m + b) & (CHUNK - 1)];
                        En = ld_ent<STEP>(e + (b + 1) * ROW, R(0));
                        if (MODE != 2) {
                            const R rg = node_products<MODE, STATS, R>(gm, Ec.gr, Ec.gi, dc, wn, stage + b * RED_VALS * STAGE_LD + lane, max2);
                            if (MODE == 1 && act) A.ldos[(size_t)(noff + m + b) * ne + n] = (double)rg;
                        }
                        gm = step_up<STEP, R>(gm, cc, zr0, zi0, Ec);
                    }
                    if (MODE == 0) {
                        __syncwarp();
                        if (lane < rem * RED_VALS) {
                            double s = stage_colsum(stage, lane);
                            if (n0) s += part_old;
                            PART[m * RED_VALS + lane] = s;
                        }
                        __syncwarp();
                    }
                    m = mhi;
                }
                __syncwarp();                                           // this chunk's buffer is free for the next load
            }
            if (act) A.store_new[(size_t)dF * ne + n] = mk2(gm.re, gm.im);
        }
    }
    if (STATS) {
        double mx = (double)max2;
#pragma unroll
        for (int o = 16; o; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        if (lane == 0) A.stat_max2[slot] = mx;
    }
}

// ------------------------------------------------------------------------------------------------
// a6 + a7: rotate back, sum over angles, finalise
// ------------------------------------------------------------------------------------------------
struct BackArgs {
    GridDev G;
    int nphi, nrot; double c;
    const double* vx; const double* vy; const double* eta; const double* W;
    const int* line_g;           // [pair][t] -> first physical trajectory on that lattice line, or -1
    const int* line_n;           // [pair][t] -> number of trajectories (inside intervals) on that line
    TrajDev T;
    const double* part;          // [node][6]
    double t, D; int sigma;
    double2* delta_new; double* jx; double* jy; double* feI;
    int* n_bad;
    double* raw;                 // non-null: write the 5 un-finalised accumulators [5][ny][nx] instead (energy-sharded sweep)
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

__global__ void rotate_back_kernel(BackArgs B) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= B.G.nx) return;
    const size_t q = (size_t)j * B.G.nx + i;
    double nr = 0.0, ni = 0.0, sjx = 0.0, sjy = 0.0, sI = 0.0;
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
            const double Wk = B.W[p], Wk2 = B.W[p + H], ek = B.eta[p], ek2 = B.eta[p + H];
            nr += Wk * ek * f0 + Wk2 * ek2 * f2;
            ni += Wk * ek * f1 - Wk2 * ek2 * f3;
            const double wj = (Wk + Wk2) * f4;
            sjx = fma(wj, B.vx[p], sjx); sjy = fma(wj, B.vy[p], sjy);
            sI += (Wk + Wk2) * f5;
        }
    }
    if (B.raw) {
        const size_t ng = (size_t)B.G.nx * B.G.ny;
        B.raw[q] = nr; B.raw[ng + q] = ni; B.raw[2 * ng + q] = sjx; B.raw[3 * ng + q] = sjy; B.raw[4 * ng + q] = sI;
        return;
    }
    // Delta_new = -2 i t Num / D (Eq. 22 with f = -2 pi i gamma/(1+P)); j = 2 sigma t J (Eq. 8); I = t I (Eq. 19)
    const double s = 2.0 * B.t / B.D;
    if (B.delta_new) B.delta_new[q] = make_double2(s * ni, -s * nr);
    if (B.jx) B.jx[q] = 2.0 * B.sigma * B.t * sjx;
    if (B.jy) B.jy[q] = 2.0 * B.sigma * B.t * sjy;
    if (B.feI) B.feI[q] = B.t * sI;
}

// a7 alone, after the accumulators of all energy shards have been summed
__global__ void finalise_kernel(size_t ng, const double* raw, double t, double D, int sigma,
                                double2* delta_new, double* jx, double* jy, double* feI) {
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= ng) return;
    const double s = 2.0 * t / D;
    if (delta_new) delta_new[q] = make_double2(s * raw[ng + q], -s * raw[q]);
    if (jx) jx[q] = 2.0 * sigma * t * raw[2 * ng + q];
    if (jy) jy[q] = 2.0 * sigma * t * raw[3 * ng + q];
    if (feI) feI[q] = t * raw[4 * ng + q];
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
template <typename R>
__global__ void debug_traj_kernel(MarchArgsT<R> A, int stepper, int g, int n, double2* outG, double2* outGT) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    using V4 = typename VT<R>::V4;
    const int nn = A.T.nn[g];
    const V4* PC = A.pc + A.T.noff[g] + g;
    const int nb = A.E.partner[n];
    const R zr0 = (R)A.E.zr[n], zi0 = (R)A.E.zi[n];
    const int dF = A.T.dF[g], dB = A.T.dB[g];
    cplx_t<R> gt;
    if (A.bc_mode == 1) gt = hom_start<R>(-(double)PC[nn].x, PC[nn].y, A.E.zr[n] + PC[nn].z, A.E.zi[n]);
    else if (A.ga_n[dB]) { cplx_t<R> s = gather_start(A, dB, nb); gt = mk(s.re, -s.im); }
    else { cplx_t<R> s = hom_start<R>(A.fb_D[dB].x, A.fb_D[dB].y, A.E.zr[nb] + A.fb_a[dB], A.E.zi[nb]); gt = mk(s.re, -s.im); }
    // the same evaluation of T as the march: Taylor table for interior pieces inside its radius, exp-based otherwise
    constexpr int KT = scm::TaylorK<R>::K;
    R tcf[KT + 1]; R thr2 = R(-1), pole_a = R(1), pole_res = R(0);
    if (A.E.tc) {
        for (int k = 0; k <= KT; ++k) tcf[k] = (R)A.E.tc[(size_t)n * TC_LD + k];
        thr2 = (R)(A.E.tc[(size_t)n * TC_LD + 9] * scm::TaylorK<R>::RMAX2);
        pole_a = (R)A.E.tc[(size_t)n * TC_LD + 10]; pole_res = (R)A.E.tc[(size_t)n * TC_LD + 11];
    }
    auto coefT = [&](const V4& c, int p) {
        const R d2 = scm::mad(c.x, c.x, c.y * c.y);
        const R dwr = scm::mad(-c.z, c.z, d2), dwi = R(-2) * zi0 * c.z;
        const R s2 = scm::mad(dwr, dwr, dwi * dwi);
        if (p > 0 && p < nn && s2 <= thr2) return scm::taylor_T<R, KT>(tcf, pole_a, pole_res, dwr, dwi, s2);
        return scm::coef_T(d2, zr0 + c.z, zi0, c.w);
    };
    for (int p = nn; p >= 1; --p) {
        const V4 c = PC[p];
        if (stepper == 1) gt = scm::step_mid(gt, -c.x, c.y, zr0 + c.z, zi0, c.w);
        else { const cplx_t<R> T = coefT(c, p); gt = scm::step_T(gt, -c.x, c.y, zr0 + c.z, zi0, T); }
        outGT[p - 1] = make_double2(gt.re, gt.im);
    }
    cplx_t<R> gm;
    if (A.bc_mode == 1) gm = hom_start<R>(PC[0].x, PC[0].y, A.E.zr[n] + PC[0].z, A.E.zi[n]);
    else if (A.ga_n[dF]) gm = gather_start(A, dF, n);
    else gm = hom_start<R>(A.fb_D[dF].x, A.fb_D[dF].y, A.E.zr[n] + A.fb_a[dF], A.E.zi[n]);
    for (int p = 0; p < nn; ++p) {
        const V4 c = PC[p];
        if (stepper == 1) gm = scm::step_mid(gm, c.x, c.y, zr0 + c.z, zi0, c.w);
        else { const cplx_t<R> T = coefT(c, p); gm = scm::step_T(gm, c.x, c.y, zr0 + c.z, zi0, T); }
        outG[p] = make_double2(gm.re, gm.im);
    }
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

}  // namespace sck
