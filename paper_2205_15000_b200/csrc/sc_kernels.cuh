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
using scm::mk;

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

struct EnergyDev { int ne; const double* zr; const double* zi; const double* w; const int* partner; };

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

// a2: one warp per trajectory, lanes over nodes (coalesced along the trajectory).
__global__ void rotate_in_kernel(GridDev G, TrajDev T, const double* vx, const double* vy, const double* eta,
                                 double c, int sigma, double2* nd_D, double* nd_a, int* n_bad) {
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
        nd_a[off + m] = sigma * (cx * interp_plain(G, G.Ax, x, y) + cy * interp_plain(G, G.Ay, x, y));
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
__global__ void reset_store_kernel(TrajDev T, EnergyDev E, const double2* nd_D, const double* nd_a, double2* store) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)T.n * E.ne) return;
    const int g = (int)(idx / E.ne), n = (int)(idx % E.ne);
    const long long off = T.noff[g];
    const int nn = T.nn[g];
    const double2 Dl = nd_D[off + nn - 1], D0 = nd_D[off];
    const cplx ge = scm::gamma_hom(Dl.x, Dl.y, E.zr[n] + nd_a[off + nn - 1], E.zi[n]);
    store[(size_t)T.dF[g] * E.ne + n] = make_double2(ge.re, ge.im);
    const cplx gt = scm::gamma_hom(-D0.x, D0.y, E.zr[n] + nd_a[off], E.zi[n]);
    store[(size_t)T.dB[g] * E.ne + E.partner[n]] = make_double2(gt.re, -gt.im);
}

// ------------------------------------------------------------------------------------------------
// the march
// ------------------------------------------------------------------------------------------------
struct MarchArgs {
    TrajDev T;
    EnergyDev E;
    const int* order; int n_items;          // longest-first work list
    double h;
    const double2* nd_D; const double* nd_a;
    int bc_mode;
    const int* ga_idx; const double* ga_w; const unsigned char* ga_n;   // entry gathers per store row [row][4]
    const double2* fb_D; const double* fb_a;
    const double2* store_old; double2* store_new;
    double2* scr_T; double2* scr_G; long long scr_stride;   // per warp slot: (smax+1)*32 double2 each
    double* part;                            // MODE 0: [node][6] = SF.re, SF.im, X2.re, X2.im, SG, SI
    double* ldos;                            // MODE 1: [node][ne] = Re g_n
    int* counter;
    double* stat_max2;                       // per warp slot: max |gamma|^2 seen (optional)
};

constexpr int MARCH_WARPS = 8;               // warps per CTA
constexpr int RED_NODES = 4;                 // nodes per shared-memory reduction batch
constexpr int RED_VALS = 6;

__device__ __forceinline__ cplx gather_start(const MarchArgs& A, int row, int n) {
    const int cnt = A.ga_n[row];
    double sr = 0.0, si = 0.0;
    for (int i = 0; i < cnt; ++i) {
        const double w = A.ga_w[4 * row + i];
        const double2 v = A.store_old[(size_t)A.ga_idx[4 * row + i] * A.E.ne + n];
        sr = fma(w, v.x, sr); si = fma(w, v.y, si);
    }
    return mk(sr, si);
}

// MODE 0: Matsubara sums; 1: per-energy Re g (LDOS); 2: boundary values only.
template <int MODE, bool STATS>
__global__ void __launch_bounds__(MARCH_WARPS * 32, 2) march_kernel(MarchArgs A) {
    __shared__ double stage_all[MARCH_WARPS][RED_NODES * RED_VALS][32];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int slot = blockIdx.x * MARCH_WARPS + wib;
    double (*stage)[32] = stage_all[wib];
    double2* __restrict__ sT = A.scr_T + (size_t)slot * A.scr_stride;
    double2* __restrict__ sG = A.scr_G + (size_t)slot * A.scr_stride;
    const int ne = A.E.ne;
    double max2 = 0.0;

    for (;;) {
        int item = 0;
        if (lane == 0) item = atomicAdd(A.counter, 1);
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= A.n_items) break;
        const int g = A.order[item];
        const int nn = A.T.nn[g];
        const long long noff = A.T.noff[g];
        const double l0 = A.T.l0[g], l1 = A.T.l1[g];
        const int dF = A.T.dF[g], dB = A.T.dB[g];
        const double2* __restrict__ ND = A.nd_D + noff;
        const double* __restrict__ NA = A.nd_a + noff;

        for (int n0 = 0; n0 < ne; n0 += 32) {
            const bool act = n0 + lane < ne;
            const int n = act ? n0 + lane : ne - 1;
            const double zr0 = A.E.zr[n], zi0 = A.E.zi[n];
            const double wn = act ? A.E.w[n] : 0.0;
            const int nb = A.E.partner[n];

            // ---------------- pass 1: gamma-tilde from u_out down to u_in; record T and gamma-tilde ----------
            double2 Dhi = ND[nn - 1]; double ahi = NA[nn - 1];
            cplx gt;
            if (A.bc_mode == 1) {
                gt = scm::gamma_hom(-Dhi.x, Dhi.y, zr0 + ahi, zi0);
            } else if (A.ga_n[dB]) {
                const cplx s = gather_start(A, dB, nb);            // gamma of the mirrored trajectory at its entry
                gt = mk(s.re, -s.im);
            } else {
                const cplx s = scm::gamma_hom(A.fb_D[dB].x, A.fb_D[dB].y, A.E.zr[nb] + A.fb_a[dB], A.E.zi[nb]);
                gt = mk(s.re, -s.im);
            }
            {
                // piece nn: [u_jl, u_out], coefficients of node nn-1 (nearest-neighbour extrapolation, :1003)
                const double zr = zr0 + ahi;
                const cplx T = scm::coef_T(fma(Dhi.x, Dhi.x, Dhi.y * Dhi.y), zr, zi0, l1);
                gt = scm::step_T(gt, -Dhi.x, Dhi.y, zr, zi0, T);
                sT[(size_t)nn * 32 + lane] = make_double2(T.re, T.im);
                sG[(size_t)(nn - 1) * 32 + lane] = make_double2(gt.re, gt.im);
            }
            double2 Dnx = nn >= 2 ? ND[nn - 2] : Dhi; double anx = nn >= 2 ? NA[nn - 2] : ahi;
            for (int m = nn - 1; m >= 1; --m) {
                // piece m: [u_{m-1}, u_m], half-step coefficients by linear interpolation (:1003)
                const double2 Dlo = Dnx; const double alo = anx;
                if (m >= 2) { Dnx = ND[m - 2]; anx = NA[m - 2]; }          // prefetch for the next iteration
                const double Dr = 0.5 * (Dlo.x + Dhi.x), Di = 0.5 * (Dlo.y + Dhi.y);
                const double zr = zr0 + 0.5 * (alo + ahi);
                const cplx T = scm::coef_T(fma(Dr, Dr, Di * Di), zr, zi0, A.h);
                gt = scm::step_T(gt, -Dr, Di, zr, zi0, T);
                sT[(size_t)m * 32 + lane] = make_double2(T.re, T.im);
                sG[(size_t)(m - 1) * 32 + lane] = make_double2(gt.re, gt.im);
                Dhi = Dlo; ahi = alo;
            }
            {
                // piece 0: [u_in, u_jf], coefficients of node 0
                const double zr = zr0 + ahi;
                const cplx T = scm::coef_T(fma(Dhi.x, Dhi.x, Dhi.y * Dhi.y), zr, zi0, l0);
                gt = scm::step_T(gt, -Dhi.x, Dhi.y, zr, zi0, T);
                sT[lane] = make_double2(T.re, T.im);
                if (act) A.store_new[(size_t)dB * ne + nb] = make_double2(gt.re, -gt.im);
            }

            // ---------------- pass 2: gamma from u_in up to u_out; products and energy reduction ------------
            cplx gm;
            double2 Dlo = Dhi; double alo = ahi;        // node 0
            if (A.bc_mode == 1) gm = scm::gamma_hom(Dlo.x, Dlo.y, zr0 + alo, zi0);
            else if (A.ga_n[dF]) gm = gather_start(A, dF, n);
            else gm = scm::gamma_hom(A.fb_D[dF].x, A.fb_D[dF].y, zr0 + A.fb_a[dF], zi0);
            {
                const double2 t = sT[lane];
                gm = scm::step_T(gm, Dlo.x, Dlo.y, zr0 + alo, zi0, mk(t.x, t.y));
            }
            double2 Tn = sT[(size_t)1 * 32 + lane];
            double2 Gn = sG[lane];
            double2 Dn2 = nn >= 2 ? ND[1] : Dlo; double an2 = nn >= 2 ? NA[1] : alo;
            for (int m = 0; m < nn; ++m) {
                // node m: gm = gamma(u_m), Gn = gamma-tilde(u_m), (Dlo, alo) = node coefficients
                const double2 Tc = Tn; const double2 Gc = Gn;
                if (m + 1 < nn) { Tn = sT[(size_t)(m + 2) * 32 + lane]; Gn = sG[(size_t)(m + 1) * 32 + lane]; }
                if (MODE != 2) {
                    const double Pr = fma(gm.re, Gc.x, -gm.im * Gc.y), Pi = fma(gm.re, Gc.y, gm.im * Gc.x);
                    const double qr = 1.0 + Pr;
                    const double rq = scm::rcp_nr(fma(qr, qr, Pi * Pi));
                    const double ir = qr * rq, ii = -Pi * rq;               // 1/(1+P)
                    if (STATS) max2 = fmax(max2, fmax(fma(gm.re, gm.re, gm.im * gm.im), fma(Gc.x, Gc.x, Gc.y * Gc.y)));
                    if (MODE == 0) {
                        const double wr = wn * ir, wi = wn * ii;
                        const int r = (m & (RED_NODES - 1)) * RED_VALS;
                        stage[r + 0][lane] = fma(gm.re, wr, -gm.im * wi);    // SF  = w gamma/(1+P)
                        stage[r + 1][lane] = fma(gm.re, wi, gm.im * wr);
                        stage[r + 2][lane] = fma(Gc.x, wr, -Gc.y * wi);      // X2  = w gamma~/(1+P)  (SF of k+N/2 = conj)
                        stage[r + 3][lane] = fma(Gc.x, wi, Gc.y * wr);
                        stage[r + 4][lane] = 2.0 * wi;                       // SG  = w Im g = 2 w Im 1/(1+P)
                        stage[r + 5][lane] = wn * fma(Dlo.x, gm.im - Gc.y, -Dlo.y * (gm.re + Gc.x));   // SI
                        if ((m & (RED_NODES - 1)) == RED_NODES - 1 || m == nn - 1) {
                            __syncwarp();
                            const int cnt = ((m & (RED_NODES - 1)) + 1) * RED_VALS;
                            if (lane < cnt) {
                                double s = 0.0;
#pragma unroll 8
                                for (int i = 0; i < 32; ++i) s += stage[lane][(i + lane) & 31];
                                double* dst = A.part + (size_t)(noff + (m & ~(RED_NODES - 1))) * RED_VALS + lane;
                                if (n0) s += *dst;
                                *dst = s;
                            }
                            __syncwarp();
                        }
                    } else if (act) {
                        A.ldos[(size_t)(noff + m) * ne + n] = fma(2.0, ir, -1.0);   // Re g = 2 Re 1/(1+P) - 1
                    }
                }
                // step to node m+1 (or to u_out)
                if (m + 1 < nn) {
                    const double2 Dhi2 = Dn2; const double ahi2 = an2;
                    if (m + 2 < nn) { Dn2 = ND[m + 2]; an2 = NA[m + 2]; }
                    const double Dr = 0.5 * (Dlo.x + Dhi2.x), Di = 0.5 * (Dlo.y + Dhi2.y);
                    gm = scm::step_T(gm, Dr, Di, zr0 + 0.5 * (alo + ahi2), zi0, mk(Tc.x, Tc.y));
                    Dlo = Dhi2; alo = ahi2;
                } else {
                    gm = scm::step_T(gm, Dlo.x, Dlo.y, zr0 + alo, zi0, mk(Tc.x, Tc.y));
                }
            }
            if (act) A.store_new[(size_t)dF * ne + n] = make_double2(gm.re, gm.im);
        }
    }
    if (STATS) {
#pragma unroll
        for (int o = 16; o; o >>= 1) max2 = fmax(max2, __shfl_xor_sync(0xffffffffu, max2, o));
        if (lane == 0) A.stat_max2[slot] = max2;
    }
}

// ------------------------------------------------------------------------------------------------
// a6 + a7: rotate back, sum over angles, finalise
// ------------------------------------------------------------------------------------------------
struct BackArgs {
    GridDev G;
    int nphi, nrot; double c;
    const double* vx; const double* vy; const double* eta; const double* W;
    const int* line_g;           // [pair][t] -> physical trajectory or -1
    TrajDev T;
    const double* part;          // [node][6]
    double t, D; int sigma;
    double2* delta_new; double* jx; double* jy; double* feI;
    int* n_bad;
};

// weights of the (up to 4) valid lattice nodes around a grid point for pair p; returns count
__device__ __forceinline__ int back_weights(const BackArgs& B, int p, double x, double y, long long node[4], double w[4]) {
    const double cx = B.vx[p], cy = B.vy[p];
    const double uu = (x * cx + y * cy) / B.G.h + B.c, ww = (-x * cy + y * cx) / B.G.h + B.c;
    const int j0 = (int)floor(uu), t0 = (int)floor(ww);
    const double fu = uu - j0, fw = ww - t0;
    const int* lg = B.line_g + (size_t)p * B.nrot;
    int n = 0; double sw = 0.0;
#pragma unroll
    for (int b = 0; b < 2; ++b) {
        const int tt = t0 + b;
        if (tt < 0 || tt >= B.nrot) continue;
        const int g = lg[tt];
        if (g < 0) continue;
        const int jf = B.T.jf[g], nn = B.T.nn[g];
#pragma unroll
        for (int a = 0; a < 2; ++a) {
            const int jj = j0 + a;
            if (jj < jf || jj >= jf + nn) continue;
            const double wt = (a ? fu : 1.0 - fu) * (b ? fw : 1.0 - fw);
            node[n] = B.T.noff[g] + (jj - jf); w[n] = wt; sw += wt; ++n;
        }
    }
    if (sw > 1e-12) { const double r = 1.0 / sw; for (int i = 0; i < n; ++i) w[i] *= r; return n; }
    double bd = 1e300; long long best = -1;
    for (int tt = t0 - 2; tt <= t0 + 3; ++tt) {
        if (tt < 0 || tt >= B.nrot) continue;
        const int g = lg[tt];
        if (g < 0) continue;
        const int jf = B.T.jf[g], nn = B.T.nn[g];
        for (int jj = j0 - 2; jj <= j0 + 3; ++jj) {
            if (jj < jf || jj >= jf + nn) continue;
            const double d = (uu - jj) * (uu - jj) + (ww - tt) * (ww - tt);
            if (d < bd) { bd = d; best = B.T.noff[g] + (jj - jf); }
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
    // Delta_new = -2 i t Num / D (Eq. 22 with f = -2 pi i gamma/(1+P)); j = 2 sigma t J (Eq. 8); I = t I (Eq. 19)
    const double s = 2.0 * B.t / B.D;
    if (B.delta_new) B.delta_new[q] = make_double2(s * ni, -s * nr);
    if (B.jx) B.jx[q] = 2.0 * B.sigma * B.t * sjx;
    if (B.jy) B.jy[q] = 2.0 * B.sigma * B.t * sjy;
    if (B.feI) B.feI[q] = B.t * sI;
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
__global__ void debug_traj_kernel(MarchArgs A, int g, int n, double2* outG, double2* outGT) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const int nn = A.T.nn[g]; const long long noff = A.T.noff[g];
    const double2* ND = A.nd_D + noff; const double* NA = A.nd_a + noff;
    const int nb = A.E.partner[n];
    const double zr0 = A.E.zr[n], zi0 = A.E.zi[n];
    const int dF = A.T.dF[g], dB = A.T.dB[g];
    cplx gt;
    if (A.bc_mode == 1) gt = scm::gamma_hom(-ND[nn - 1].x, ND[nn - 1].y, zr0 + NA[nn - 1], zi0);
    else if (A.ga_n[dB]) { cplx s = gather_start(A, dB, nb); gt = mk(s.re, -s.im); }
    else { cplx s = scm::gamma_hom(A.fb_D[dB].x, A.fb_D[dB].y, A.E.zr[nb] + A.fb_a[dB], A.E.zi[nb]); gt = mk(s.re, -s.im); }
    for (int m = nn; m >= 1; --m) {
        double Dr, Di, a, len;
        if (m == nn) { Dr = ND[nn - 1].x; Di = ND[nn - 1].y; a = NA[nn - 1]; len = A.T.l1[g]; }
        else { Dr = 0.5 * (ND[m - 1].x + ND[m].x); Di = 0.5 * (ND[m - 1].y + ND[m].y); a = 0.5 * (NA[m - 1] + NA[m]); len = A.h; }
        const cplx T = scm::coef_T(Dr * Dr + Di * Di, zr0 + a, zi0, len);
        gt = scm::step_T(gt, -Dr, Di, zr0 + a, zi0, T);
        outGT[m - 1] = make_double2(gt.re, gt.im);
    }
    cplx gm;
    if (A.bc_mode == 1) gm = scm::gamma_hom(ND[0].x, ND[0].y, zr0 + NA[0], zi0);
    else if (A.ga_n[dF]) gm = gather_start(A, dF, n);
    else gm = scm::gamma_hom(A.fb_D[dF].x, A.fb_D[dF].y, zr0 + A.fb_a[dF], zi0);
    for (int m = 0; m < nn; ++m) {
        double Dr, Di, a, len;
        if (m == 0) { Dr = ND[0].x; Di = ND[0].y; a = NA[0]; len = A.T.l0[g]; }
        else { Dr = 0.5 * (ND[m - 1].x + ND[m].x); Di = 0.5 * (ND[m - 1].y + ND[m].y); a = 0.5 * (NA[m - 1] + NA[m]); len = A.h; }
        const cplx T = scm::coef_T(Dr * Dr + Di * Di, zr0 + a, zi0, len);
        gm = scm::step_T(gm, Dr, Di, zr0 + a, zi0, T);
        outG[m] = make_double2(gm.re, gm.im);
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
