// sc_field_kernels.cuh — grid-field kernels around the sweep: vector-potential solve (a8) and the
// self-consistency mixing (a9).  All reductions are two-stage with a fixed block count and a fixed
// summation order (deterministic, no atomics).
//
// a8: A_ind = -(1/kappa^2) G (*) (j - <j>_mask)  (PAPER.md D1 :1009, :1040), G_{m,n} from the closed form
// D3-D6 (:1014-1021).  The paper truncates an eigen-decomposition of G "to increase performance" (:1033);
// here the cross-correlation is done exactly as a zero-padded (2nx x 2ny) FFT convolution (cuFFT D2Z/Z2D —
// a library FFT, off the roofline-judged path): O(N^2 log N) instead of O(N^4).
// a9: x = (Re D, Im D, kappa^2 A_x, kappa^2 A_y) (E3 :1053), d = g(x) - x (E4), Picard (E5), Barzilai-Borwein
// (E8-E11), Polyak (E6-E7) or CongAcc (E12-E17), with step sizes, weights and the bisection of E17 kept on the device.
#pragma once
#include <cuda_runtime.h>
#include <cufft.h>

#include <cmath>
#include <string>
#include <vector>

namespace scf {

constexpr int RED_BLOCKS = 296;
constexpr int RED_THREADS = 256;
constexpr int NX_MAX = 10;          // slices of the iterate x: (Re, Im) of up to 4 order-parameter components + kappa^2 A_x, A_y
constexpr int RED_MAXOUT = 3 * NX_MAX;   // outputs of one reduction (CongAcc: 3 dot products per slice)
constexpr int ST_ALPHA = 8, ST_W = 24;   // offsets of alpha_c and w_c in the device state array
constexpr int RED_RES = RED_BLOCKS * RED_MAXOUT;   // offset of the results behind the partials

// parameters of the accelerators (PAPER.md Listings 14-16 :1093, :1121, :1157)
struct AccelParams { double drag = 0.5, kfac = 1.234, smin = 0.7, amin = 1e-3, amax = 100.0; };

struct FieldState {
    // vector potential
    int nx = 0, ny = 0; double h = 0;
    cufftHandle plan_f = 0, plan_b = 0; bool plans = false;
    cufftDoubleComplex* Ghat = nullptr; double* pad = nullptr; cufftDoubleComplex* spec = nullptr;
    double* red = nullptr;          // RED_BLOCKS * RED_MAXOUT partials + 32 results
    double vp_eps = 0.0;            // > 0: the paper's truncated eigen-decomposition of G (D7-D9) instead of the exact FFT correlation
    struct LowRank* lr = nullptr;
    // driver
    size_t ng = 0; int nc = 1;      // grid points, order-parameter components (x has 2 nc + 2 slices of ng)
    double *Atot_x = nullptr, *Atot_y = nullptr, *jx = nullptr, *jy = nullptr, *feI = nullptr, *gAx = nullptr, *gAy = nullptr;
    double2* dnew = nullptr;
    double* d_prev = nullptr;       // (2 nc + 2) * ng
    double* d_cur = nullptr;        // (2 nc + 2) * ng
    double *prev_jx = nullptr, *prev_jy = nullptr, *prev_fe = nullptr;
    double* upd = nullptr;          // (2 nc + 2) * ng: x_{i+1} - x_i
    double* aux = nullptr;          // same size: Polyak velocity v / CongAcc moving average m (allocated on first use)
    double* state = nullptr;        // [0] alpha, [1] iteration index, [2..5] residuals (delta, A, j, fe), [ST_ALPHA..] alpha_c, [ST_W..] w_c
    AccelParams par;
    bool driver = false, first = true; int last_kind = -1;
};

// driver buffers only (the number of order-parameter components changed); keeps the FFT plans and the G table
inline void release_driver(FieldState& F) {
    void** ptrs[] = {(void**)&F.Atot_x, (void**)&F.Atot_y, (void**)&F.jx, (void**)&F.jy, (void**)&F.feI, (void**)&F.gAx, (void**)&F.gAy,
                     (void**)&F.dnew, (void**)&F.d_prev, (void**)&F.d_cur, (void**)&F.prev_jx, (void**)&F.prev_jy, (void**)&F.prev_fe,
                     (void**)&F.state, (void**)&F.upd, (void**)&F.aux};
    for (void** p : ptrs) { if (*p) cudaFree(*p); *p = nullptr; }
    F.driver = false; F.first = true; F.last_kind = -1;
}
inline void release_lowrank(FieldState& F);
inline void release(FieldState& F) {
    release_lowrank(F);
    if (F.plans) { cufftDestroy(F.plan_f); cufftDestroy(F.plan_b); }
    void* ptrs[] = {F.Ghat, F.pad, F.spec, F.red, F.Atot_x, F.Atot_y, F.jx, F.jy, F.feI, F.gAx, F.gAy, F.dnew,
                    F.d_prev, F.d_cur, F.prev_jx, F.prev_jy, F.prev_fe, F.state, F.upd, F.aux};
    for (void* p : ptrs) if (p) cudaFree(p);
    F = FieldState();
}

// ---- deterministic reductions --------------------------------------------------------------------
// MAXR: maximum of non-negative terms instead of their sum (max-norm residuals)
template <typename Op, bool MAXR = false>
__global__ void reduce_stage1(size_t n, Op op, double* partial, int nout) {
    __shared__ double sh[RED_THREADS];
    for (int c = 0; c < nout; ++c) {
        double s = 0.0;
        for (size_t i = (size_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (size_t)RED_BLOCKS * RED_THREADS) {
            if (MAXR) s = fmax(s, op(i, c)); else s += op(i, c);
        }
        sh[threadIdx.x] = s;
        __syncthreads();
        for (int o = RED_THREADS / 2; o; o >>= 1) {
            if (threadIdx.x < o) sh[threadIdx.x] = MAXR ? fmax(sh[threadIdx.x], sh[threadIdx.x + o]) : sh[threadIdx.x] + sh[threadIdx.x + o];
            __syncthreads();
        }
        if (threadIdx.x == 0) partial[(size_t)c * RED_BLOCKS + blockIdx.x] = sh[0];
        __syncthreads();
    }
}
template <bool MAXR = false>
__global__ void reduce_stage2(const double* partial, int nout, double* out) {
    const int c = threadIdx.x;
    if (c >= nout) return;
    double s = 0.0;
    for (int b = 0; b < RED_BLOCKS; ++b) s = MAXR ? fmax(s, partial[(size_t)c * RED_BLOCKS + b]) : s + partial[(size_t)c * RED_BLOCKS + b];
    out[c] = s;
}

// ---- vector potential -------------------------------------------------------------------------------
inline double G_closed(int m, int n, double h) {
    // PAPER.md D3-D6 (:1014-1021), lengths in xi0
    double acc = 0.0;
    for (int sa = 1; sa >= -1; sa -= 2)
        for (int sb = 1; sb >= -1; sb -= 2) {
            const double p = 1.0 + 2.0 * sa * m, q = 1.0 + 2.0 * sb * n;      // (1+2m), (1+2n) with signed indices
            const double mm = sa * (double)m, nn = sb * (double)n;
            const double alpha = p * q * std::log(0.5 * p * p + 0.5 * q * q);
            const double beta1 = (-2.0 * mm * mm + 2.0 * nn * nn + 4.0 * nn + 1.0) * std::atan(p / q);
            const double beta2 = (-2.0 * nn * nn + 2.0 * mm * mm + 4.0 * mm + 1.0) * std::atan(q / p);
            acc += alpha + beta1 + beta2;
        }
    const double PI_ = 3.14159265358979323846;
    return h * h / (4.0 * PI_) * (2.0 * std::log(h) - std::log(2.0) - 3.0 + 0.25 * acc);
}

}  // namespace scf
#include "sc_lowrank.cuh"
namespace scf {
inline void release_lowrank(FieldState& F) { if (F.lr) { release(*F.lr); delete F.lr; F.lr = nullptr; } }

__global__ void pad_current_kernel(int nx, int ny, const unsigned char* mask, const double* j, const double* mean, int comp, double* pad) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, jj = blockIdx.y;
    const int px = 2 * nx;
    if (i >= px) return;
    double v = 0.0;
    if (i < nx && jj < ny) { const size_t q = (size_t)jj * nx + i; if (mask[q]) v = j[q] - mean[comp]; }
    pad[(size_t)jj * px + i] = v;
}
__global__ void spec_mul_kernel(size_t n, cufftDoubleComplex* s, const cufftDoubleComplex* g) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const cufftDoubleComplex a = s[i], b = g[i];
    s[i] = make_cuDoubleComplex(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__global__ void crop_kernel(int nx, int ny, const double* pad, double scale, double* out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= nx) return;
    out[(size_t)j * nx + i] = scale * pad[(size_t)j * 2 * nx + i];
}

struct MeanOp {
    const unsigned char* mask; const double* jx; const double* jy;
    __device__ double operator()(size_t i, int c) const { return mask[i] ? (c == 0 ? jx[i] : c == 1 ? jy[i] : 1.0) : 0.0; }
};
__global__ void mean_finish_kernel(double* r) { const double cnt = r[2] > 0 ? r[2] : 1.0; r[0] /= cnt; r[1] /= cnt; }
struct FemagOp {
    const unsigned char* mask; const double *jx, *jy, *ax, *ay;
    __device__ double operator()(size_t i, int) const { return mask[i] ? jx[i] * ax[i] + jy[i] * ay[i] : 0.0; }
};

#define SCF_CU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { err = std::string(#call) + ": " + cudaGetErrorString(e_); return e_ == cudaErrorMemoryAllocation ? 2 : 1; } } while (0)
#define SCF_FFT(call) do { cufftResult r_ = (call); if (r_ != CUFFT_SUCCESS) { err = std::string(#call) + ": cufft error " + std::to_string((int)r_); return 1; } } while (0)

inline int ensure_vp(FieldState& F, int nx, int ny, double h, cudaStream_t s, std::string& err) {
    if (F.plans) return 0;
    F.nx = nx; F.ny = ny; F.h = h;
    const int px = 2 * nx, py = 2 * ny; const size_t nspec = (size_t)py * (px / 2 + 1);
    SCF_CU(cudaMalloc((void**)&F.pad, (size_t)px * py * sizeof(double)));
    SCF_CU(cudaMalloc((void**)&F.spec, nspec * sizeof(cufftDoubleComplex)));
    SCF_CU(cudaMalloc((void**)&F.Ghat, nspec * sizeof(cufftDoubleComplex)));
    if (!F.red) SCF_CU(cudaMalloc((void**)&F.red, (RED_RES + 64) * sizeof(double)));
    SCF_FFT(cufftPlan2d(&F.plan_f, py, px, CUFFT_D2Z));
    SCF_FFT(cufftPlan2d(&F.plan_b, py, px, CUFFT_Z2D));
    SCF_FFT(cufftSetStream(F.plan_f, s)); SCF_FFT(cufftSetStream(F.plan_b, s));
    F.plans = true;
    // kernel table on the circular (2ny x 2nx) grid: K[dy][dx] = G_{|dx|,|dy|}; host evaluation of the closed form
    std::vector<double> tab((size_t)nx * ny), K((size_t)px * py, 0.0);
    for (int n = 0; n < ny; ++n) for (int m = 0; m < nx; ++m) tab[(size_t)n * nx + m] = G_closed(m, n, h);
    for (int dy = -(ny - 1); dy <= ny - 1; ++dy)
        for (int dx = -(nx - 1); dx <= nx - 1; ++dx)
            K[(size_t)((dy + py) % py) * px + ((dx + px) % px)] = tab[(size_t)std::abs(dy) * nx + std::abs(dx)];
    SCF_CU(cudaMemcpyAsync(F.pad, K.data(), K.size() * sizeof(double), cudaMemcpyHostToDevice, s));
    SCF_FFT(cufftExecD2Z(F.plan_f, F.pad, F.Ghat));
    SCF_CU(cudaStreamSynchronize(s));
    return 0;
}

inline int vector_potential(FieldState& F, int nx, int ny, double h, const unsigned char* mask, double kappa,
                            const double* jx, const double* jy, double* Ax, double* Ay, double* fe_mag,
                            cudaStream_t s, std::string& err) {
    const size_t ng = (size_t)nx * ny;
    if (!(kappa > 0)) {       // infinite penetration depth: A_ind = 0 (:890)
        SCF_CU(cudaMemsetAsync(Ax, 0, ng * sizeof(double), s)); SCF_CU(cudaMemsetAsync(Ay, 0, ng * sizeof(double), s));
        if (fe_mag) *fe_mag = 0.0;
        return 0;
    }
    if (int rc = ensure_vp(F, nx, ny, h, s, err)) return rc;
    const int px = 2 * nx, py = 2 * ny; const size_t nspec = (size_t)py * (px / 2 + 1);
    double* res = F.red + RED_RES;
    ++sck::g_launches, reduce_stage1<<<RED_BLOCKS, RED_THREADS, 0, s>>>(ng, MeanOp{mask, jx, jy}, F.red, 3);
    ++sck::g_launches, reduce_stage2<false><<<1, 32, 0, s>>>(F.red, 3, res);
    ++sck::g_launches, mean_finish_kernel<<<1, 1, 0, s>>>(res);
    if (F.vp_eps > 0.0) {      // the paper's truncated eigen-decomposition (D7-D9) instead of the exact correlation
        if (!F.lr) F.lr = new LowRank();
        if (int rc = ensure_lowrank(*F.lr, nx, ny, h, F.vp_eps, s, err)) return rc;
        for (int comp = 0; comp < 2; ++comp) {
            ++sck::g_launches, masked_current_kernel<<<(unsigned)((ng + 255) / 256), 256, 0, s>>>(ng, mask, comp ? jy : jx, res, comp, F.lr->J);
            if (int rc = lowrank_apply(*F.lr, -1.0 / (kappa * kappa), comp ? Ay : Ax, s, err)) return rc;
        }
    }
    const double scale = -1.0 / (kappa * kappa) / ((double)px * py);
    for (int comp = 0; comp < 2 && !(F.vp_eps > 0.0); ++comp) {
        dim3 g1((px + 127) / 128, py);
        ++sck::g_launches, pad_current_kernel<<<g1, 128, 0, s>>>(nx, ny, mask, comp ? jy : jx, res, comp, F.pad);
        SCF_FFT(cufftExecD2Z(F.plan_f, F.pad, F.spec));
        ++sck::g_launches, spec_mul_kernel<<<(unsigned)((nspec + 255) / 256), 256, 0, s>>>(nspec, F.spec, F.Ghat);
        SCF_FFT(cufftExecZ2D(F.plan_b, F.spec, F.pad));
        dim3 g2((nx + 127) / 128, ny);
        ++sck::g_launches, crop_kernel<<<g2, 128, 0, s>>>(nx, ny, F.pad, scale, comp ? Ay : Ax);
    }
    SCF_CU(cudaGetLastError());
    if (fe_mag) {
        ++sck::g_launches, reduce_stage1<<<RED_BLOCKS, RED_THREADS, 0, s>>>(ng, FemagOp{mask, jx, jy, Ax, Ay}, F.red, 1);
        ++sck::g_launches, reduce_stage2<false><<<1, 32, 0, s>>>(F.red, 1, res + 4);
        double v = 0; SCF_CU(cudaMemcpyAsync(&v, res + 4, sizeof(double), cudaMemcpyDeviceToHost, s));
        SCF_CU(cudaStreamSynchronize(s));
        *fe_mag = 0.5 * h * h * v;
    }
    return 0;
}

// ---- driver ---------------------------------------------------------------------------------------
inline int ensure_driver(FieldState& F, size_t ng, int nc, std::string& err) {
    if (F.driver) return 0;
    F.ng = ng; F.nc = nc;
    const size_t nx = (size_t)(2 * nc + 2) * ng;
    double** bufs[] = {&F.Atot_x, &F.Atot_y, &F.jx, &F.jy, &F.feI, &F.gAx, &F.gAy, &F.prev_jx, &F.prev_jy, &F.prev_fe};
    for (double** b : bufs) { SCF_CU(cudaMalloc((void**)b, ng * sizeof(double))); SCF_CU(cudaMemset(*b, 0, ng * sizeof(double))); }
    SCF_CU(cudaMalloc((void**)&F.dnew, nc * ng * sizeof(double2)));
    SCF_CU(cudaMalloc((void**)&F.d_prev, nx * sizeof(double))); SCF_CU(cudaMalloc((void**)&F.d_cur, nx * sizeof(double)));
    SCF_CU(cudaMalloc((void**)&F.upd, nx * sizeof(double)));
    SCF_CU(cudaMalloc((void**)&F.state, 64 * sizeof(double))); SCF_CU(cudaMemset(F.state, 0, 64 * sizeof(double)));
    if (!F.red) SCF_CU(cudaMalloc((void**)&F.red, (RED_RES + 64) * sizeof(double)));
    F.driver = true; F.first = true;
    return 0;
}

__global__ void add_fields_kernel(size_t n, double* ox, double* oy, const double* ax, const double* ay, const double* bx, const double* by) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    ox[i] = (ax ? ax[i] : 0.0) + (bx ? bx[i] : 0.0);
    oy[i] = (ay ? ay[i] : 0.0) + (by ? by[i] : 0.0);
}
inline void add_fields(double* ox, double* oy, const double* ax, const double* ay, const double* bx, const double* by, size_t n, cudaStream_t s) {
    ++sck::g_launches, add_fields_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(n, ox, oy, ax, ay, bx, by);
}

// d = g(x) - x for the concatenated iterate x = (Re D_0, Im D_0, ..., Re D_{nc-1}, Im D_{nc-1}, kappa^2 A_x, kappa^2 A_y) (E3 :1053)
__global__ void diff_kernel(size_t ng, int nc, const double2* delta, const double2* dnew, const double* aix, const double* aiy,
                            const double* gax, const double* gay, double k2, int withA, double* d) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ng) return;
    for (int c = 0; c < nc; ++c) {
        d[(2 * c) * ng + i] = dnew[c * ng + i].x - delta[c * ng + i].x;
        d[(2 * c + 1) * ng + i] = dnew[c * ng + i].y - delta[c * ng + i].y;
    }
    d[(2 * nc) * ng + i] = withA ? k2 * (gax[i] - aix[i]) : 0.0;
    d[(2 * nc + 1) * ng + i] = withA ? k2 * (gay[i] - aiy[i]) : 0.0;
}
struct DotOp {     // c = 0: dp.dd, 1: dp.dp, 2: dd.dd, with dd = d - dp
    const double* d; const double* dp;
    __device__ double operator()(size_t i, int c) const {
        const double a = dp[i], b = d[i] - dp[i];
        return c == 0 ? a * b : c == 1 ? a * a : b * b;
    }
};
// state[0] = alpha, state[1] = iteration index i (reading R-BB: i starts at 0, first update uses alpha = step)
__global__ void alpha_kernel(double* state, const double* dots, int accelerator, double step, int first, AccelParams P) {
    if (first) { state[0] = step; state[1] = 0.0; for (int c = 0; c < NX_MAX; ++c) { state[ST_ALPHA + c] = step; state[ST_W + c] = 0.0; } }
    const int i = (int)state[1];
    if (accelerator == 1 && i >= 1) {
        const double dot = fabs(dots[0]);
        double s = 1.0;
        if (i & 1) { if (dot > 0) s = dots[1] / dot; } else { if (dots[2] > 0) s = dot / dots[2]; }
        state[0] = fmin(fmax(state[0] * s, P.amin), P.amax);
    } else if (accelerator != 1) state[0] = step;
    state[1] = i + 1;
}
// CongAcc (E12-E17 :1134-1151): dots of slice c = {m.m, m.d, d.d}[c]; one thread per slice
struct CongDotOp {   // output c = 3 * slice + {0: m.m, 1: m.d, 2: d.d}; i runs over one slice (ng values)
    size_t ng; const double* m; const double* d;
    __device__ double operator()(size_t i, int c) const {
        const size_t q = (size_t)(c / 3) * ng + i;
        const int w = c % 3;
        return w == 0 ? m[q] * m[q] : w == 1 ? m[q] * d[q] : d[q] * d[q];
    }
};
__device__ inline double cong_cos_mix(double w, double mm, double md, double dd) {
    const double num = w * md + (1.0 - w) * dd;
    const double n2 = w * w * mm + 2.0 * w * (1.0 - w) * md + (1.0 - w) * (1.0 - w) * dd;
    return (n2 > 0 && dd > 0) ? num / sqrt(n2 * dd) : 1.0;
}
// runs after alpha_kernel (state[1] already holds i + 1); one thread per slice of x
__global__ void congacc_kernel(double* state, const double* dots, int nslice, AccelParams P) {
    const int c = threadIdx.x;
    if (c >= nslice) return;
    const int i = (int)state[1] - 1;
    const double mm = dots[3 * c], md = dots[3 * c + 1], dd = dots[3 * c + 2];
    const double s = (mm > 0 && dd > 0) ? md / sqrt(mm * dd) : 0.0;            // E12
    state[ST_ALPHA + c] = fmin(fmax(state[ST_ALPHA + c] * pow(P.kfac, s), P.amin), P.amax);   // E13
    if (i == 0) state[ST_W + c] = 0.0;                                          // w_0 = 0 (:1151)
    else if (s < P.smin) {                                                      // E14, E17 by bisection
        double lo = 0.0, hi = 1.0;
        for (int it = 0; it < 60; ++it) {
            const double mid = 0.5 * (lo + hi);
            if (cong_cos_mix(mid, mm, md, dd) >= P.smin) lo = mid; else hi = mid;
        }
        state[ST_W + c] = 0.5 * (lo + hi);
    }
}
// the increment x_{i+1} - x_i: alpha d (Picard E5, BB E11); v <- (1 - drag) v + alpha d (Polyak E6-E7);
// m_c <- w_c m_c + (1 - w_c) d_c, alpha_c m_c (CongAcc E15-E16)
__global__ void step_kernel(size_t ng, int nslice, int accelerator, const double* d, double* aux, const double* state, double drag, double* upd) {
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= nslice * ng) return;
    if (accelerator == 2) { const double v = (1.0 - drag) * aux[q] + state[0] * d[q]; aux[q] = v; upd[q] = v; }
    else if (accelerator == 3) {
        const int c = (int)(q / ng);
        const double w = state[ST_W + c];
        const double m = w * aux[q] + (1.0 - w) * d[q];
        aux[q] = m; upd[q] = state[ST_ALPHA + c] * m;
    } else upd[q] = state[0] * d[q];
}
// Terms of the norms of Eq. 27 (:201; p in {1, 2, infinity}, :960).  One element of a field is one complex number
// (Delta_G at a grid point) or one 2-vector (A, j at a grid point) or one real number (I); P2 = true gives |element|^2
// (summed, root taken at the end), false |element| (summed for p = 1, maximised for p = infinity).
template <bool P2> __device__ __forceinline__ double norm_term(double a, double b) { return P2 ? a * a + b * b : sqrt(a * a + b * b); }
template <bool P2, bool MAXR> __device__ __forceinline__ double norm_join(double s, double v) { return MAXR ? fmax(s, v) : s + v; }
template <bool P2, bool MAXR>
struct NormOp {    // c: 0 dx_delta, 1 x_delta, 2 dx_A, 3 x_A (before the update); delta = all components
    size_t ng; int nc; const double2* delta; const double* aix; const double* aiy; const double* u; double k2; int withA;
    __device__ double operator()(size_t i, int c) const {
        if (c == 0) { double s = 0.0; for (int g = 0; g < nc; ++g) s = norm_join<P2, MAXR>(s, norm_term<P2>(u[(2 * g) * ng + i], u[(2 * g + 1) * ng + i])); return s; }
        if (c == 1) { double s = 0.0; for (int g = 0; g < nc; ++g) s = norm_join<P2, MAXR>(s, norm_term<P2>(delta[g * ng + i].x, delta[g * ng + i].y)); return s; }
        if (!withA) return 0.0;
        if (c == 2) return norm_term<P2>(u[(2 * nc) * ng + i] / k2, u[(2 * nc + 1) * ng + i] / k2);
        return norm_term<P2>(aix[i], aiy[i]);
    }
};
template <bool P2>
struct ObsNormOp {  // c: 0 j - j_prev, 1 j_prev, 2 fe - fe_prev, 3 fe_prev
    const double *jx, *jy, *fe, *pjx, *pjy, *pfe;
    __device__ double operator()(size_t i, int c) const {
        if (c == 0) return norm_term<P2>(jx[i] - pjx[i], jy[i] - pjy[i]);
        if (c == 1) return norm_term<P2>(pjx[i], pjy[i]);
        if (c == 2) return norm_term<P2>(fe[i] - pfe[i], 0.0);
        return norm_term<P2>(pfe[i], 0.0);
    }
};
__global__ void residual_kernel(double* state, const double* n1, const double* n2, int p2) {
    for (int q = 0; q < 4; ++q) {
        const double* n = q < 2 ? n1 + 2 * q : n2 + 2 * (q - 2);
        const double r = n[1] > 0 ? n[0] / n[1] : n[0];
        state[2 + q] = p2 ? sqrt(r) : r;
    }
}
template <bool P2, bool MAXR>
inline void residual_norms(FieldState& F, size_t ng, int nc, const double2* delta, const double* aix, const double* aiy, double k2, bool withA, cudaStream_t s) {
    double* res = F.red + RED_RES;
    ++sck::g_launches, reduce_stage1<NormOp<P2, MAXR>, MAXR><<<RED_BLOCKS, RED_THREADS, 0, s>>>(ng, NormOp<P2, MAXR>{ng, nc, delta, aix, aiy, F.upd, k2 > 0 ? k2 : 1.0, withA ? 1 : 0}, F.red, 4);
    ++sck::g_launches, reduce_stage2<MAXR><<<1, 32, 0, s>>>(F.red, 4, res + 4);
    ++sck::g_launches, reduce_stage1<ObsNormOp<P2>, MAXR><<<RED_BLOCKS, RED_THREADS, 0, s>>>(ng, ObsNormOp<P2>{F.jx, F.jy, F.feI, F.prev_jx, F.prev_jy, F.prev_fe}, F.red, 4);
    ++sck::g_launches, reduce_stage2<MAXR><<<1, 32, 0, s>>>(F.red, 4, res + 8);
    ++sck::g_launches, residual_kernel<<<1, 1, 0, s>>>(F.state, res + 4, res + 8, P2 ? 1 : 0);
}
__global__ void update_kernel(size_t ng, int nc, double2* delta, double* aix, double* aiy, const double* u,
                              const unsigned char* mask, double k2, int withA) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ng) return;
    const double m = mask[i] ? 1.0 : 0.0;
    for (int c = 0; c < nc; ++c)
        delta[c * ng + i] = make_double2(m * (delta[c * ng + i].x + u[(2 * c) * ng + i]), m * (delta[c * ng + i].y + u[(2 * c + 1) * ng + i]));
    if (withA) { aix[i] += u[(2 * nc) * ng + i] / k2; aiy[i] += u[(2 * nc + 1) * ng + i] / k2; }
}

// norm_p: the p of Eq. 27's residual norms: 2 (default), 1, or -1 for the maximum norm
inline int mix(FieldState& F, int accelerator, double step, double kappa, bool withA, double2* delta, double* aix, double* aiy,
               const unsigned char* mask, size_t ng, int norm_p, cudaStream_t s, std::string& err) {
    const double k2 = withA ? kappa * kappa : 0.0;
    const int nc = F.nc, nslice = 2 * nc + 2;
    const size_t nxl = (size_t)nslice * ng;
    const unsigned nb = (unsigned)((ng + 255) / 256), nbx = (unsigned)((nxl + 255) / 256);
    double* res = F.red + RED_RES;
    if (accelerator != F.last_kind) F.first = true;         // a change of method restarts it (v_0 = 0, w_0 = 0, m_0 = 0)
    if (accelerator >= 2) {
        if (!F.aux) SCF_CU(cudaMalloc((void**)&F.aux, nxl * sizeof(double)));
        if (F.first) SCF_CU(cudaMemsetAsync(F.aux, 0, nxl * sizeof(double), s));
    }
    ++sck::g_launches, diff_kernel<<<nb, 256, 0, s>>>(ng, nc, delta, F.dnew, aix, aiy, F.gAx, F.gAy, k2, withA ? 1 : 0, F.d_cur);
    if (!F.first && accelerator == 1) {
        ++sck::g_launches, reduce_stage1<<<RED_BLOCKS, RED_THREADS, 0, s>>>(nxl, DotOp{F.d_cur, F.d_prev}, F.red, 3);
        ++sck::g_launches, reduce_stage2<false><<<1, 32, 0, s>>>(F.red, 3, res);
    }
    ++sck::g_launches, alpha_kernel<<<1, 1, 0, s>>>(F.state, res, accelerator, step, F.first ? 1 : 0, F.par);
    if (accelerator == 3) {
        ++sck::g_launches, reduce_stage1<<<RED_BLOCKS, RED_THREADS, 0, s>>>(ng, CongDotOp{ng, F.aux, F.d_cur}, F.red, 3 * nslice);
        ++sck::g_launches, reduce_stage2<false><<<1, 32, 0, s>>>(F.red, 3 * nslice, res + 16);
        ++sck::g_launches, congacc_kernel<<<1, 32, 0, s>>>(F.state, res + 16, nslice, F.par);
    }
    ++sck::g_launches, step_kernel<<<nbx, 256, 0, s>>>(ng, nslice, accelerator, F.d_cur, F.aux, F.state, F.par.drag, F.upd);
    if (norm_p == 1) residual_norms<false, false>(F, ng, nc, delta, aix, aiy, k2, withA, s);
    else if (norm_p < 0) residual_norms<false, true>(F, ng, nc, delta, aix, aiy, k2, withA, s);
    else residual_norms<true, false>(F, ng, nc, delta, aix, aiy, k2, withA, s);
    ++sck::g_launches, update_kernel<<<nb, 256, 0, s>>>(ng, nc, delta, aix, aiy, F.upd, mask, k2 > 0 ? k2 : 1.0, withA ? 1 : 0);
    SCF_CU(cudaMemcpyAsync(F.prev_jx, F.jx, ng * sizeof(double), cudaMemcpyDeviceToDevice, s));
    SCF_CU(cudaMemcpyAsync(F.prev_jy, F.jy, ng * sizeof(double), cudaMemcpyDeviceToDevice, s));
    SCF_CU(cudaMemcpyAsync(F.prev_fe, F.feI, ng * sizeof(double), cudaMemcpyDeviceToDevice, s));
    std::swap(F.d_cur, F.d_prev);
    F.first = false; F.last_kind = accelerator;
    SCF_CU(cudaGetLastError());
    return 0;
}

inline int read_residuals(FieldState& F, double r[4], cudaStream_t s, std::string& err) {
    double st[6];
    SCF_CU(cudaMemcpyAsync(st, F.state, 6 * sizeof(double), cudaMemcpyDeviceToHost, s));
    SCF_CU(cudaStreamSynchronize(s));
    r[0] = st[2]; r[1] = st[3]; r[2] = st[4]; r[3] = st[5];
    return 0;
}

}  // namespace scf
