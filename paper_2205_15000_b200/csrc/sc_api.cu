// sc_api.cu — C ABI of libsc_riccati.so (include/sc_riccati.h): context, tables, launches.
// Product code: no CPU fallback; every numerical step runs in the kernels of sc_kernels.cuh.
#include <cuda_runtime.h>
#include <cufft.h>

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdio>
#include <cstring>
#include <numeric>
#include <set>
#include <string>
#include <vector>

#include "../../include/sc_riccati.h"
#include "sc_geometry.hpp"
#include "sc_kernels.cuh"
#include "sc_probe_kernels.cuh"
#include "sc_field_kernels.cuh"

#define SC_VERSION_STR "sc_riccati 0.1 (sm_100a)"

namespace {

template <typename T>
struct DevBuf {
    T* p = nullptr; size_t n = 0;
    cudaError_t alloc(size_t count) {
        release(); n = count;
        if (!count) return cudaSuccess;
        return cudaMalloc((void**)&p, count * sizeof(T));
    }
    cudaError_t upload(const std::vector<T>& v, cudaStream_t s) {
        cudaError_t e = alloc(v.size());
        if (e != cudaSuccess || v.empty()) return e;
        return cudaMemcpyAsync(p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, s);
    }
    void release() { if (p) cudaFree(p); p = nullptr; n = 0; }
    ~DevBuf() { release(); }
};

struct EnergySet {
    std::vector<double> zr, zi, w; std::vector<int> partner;
    DevBuf<double> d_zr, d_zi, d_w; DevBuf<int> d_partner;
    std::vector<double> tc; DevBuf<double> d_tc; int tmode = 1;     // Taylor table of T; 1: real coefficients, 2: complex
    std::vector<double> tcp; DevBuf<double> d_tcp;                  // tmode 1: pole-subtracted table
    bool unit_weights = false;                                      // all w == 1 and ne % 32 == 0
    int ne = 0;
    sck::EnergyDev dev() const { return sck::EnergyDev{ne, d_zr.p, d_zi.p, d_w.p, d_partner.p, d_tc.p, d_tcp.p, tmode}; }
};

// T(w) = tanh(h sqrt w)/sqrt w for complex w (even in sqrt w: no branch issue); series near w = 0
std::complex<double> T_of_w(std::complex<double> w, double h) {
    const std::complex<double> u = h * h * w;
    if (std::abs(u) < 1e-4) return h * (1.0 - u / 3.0 + 2.0 * u * u / 15.0 - 17.0 * u * u * u / 315.0);
    const std::complex<double> x = std::sqrt(w);
    return std::tanh(h * x) / x;
}

// Table behind sc_math.cuh taylor_real / taylor_cplx: for every energy z0, the Taylor coefficients
// c_k = T^(k)(w0)/k! of T(w) about w0 = -z0^2, k = 0..TC_KMAX.  T(w) = sum_j (2/h)/(w + (2j+1)^2 wp), wp = (pi/2h)^2,
// is analytic inside the circle through the nearest pole; the c_k come from the trapezoid rule on a circle of
// half that radius (geometric convergence).  On the imaginary axis w0 is real and so are the c_k.
// Row = Re c_0..c_8, Im c_0..c_8, (distance to the nearest pole)^2.
void taylor_table(EnergySet& E, double h) {
    const double PI = 3.14159265358979323846, wp = (PI / (2.0 * h)) * (PI / (2.0 * h));
    const int M = 128, K = sck::TC_KMAX;
    E.tmode = 1;
    for (double v : E.zr) if (v != 0.0) E.tmode = 2;
    E.tc.assign((size_t)E.zr.size() * sck::TC_LD, 0.0);
    std::vector<std::complex<double>> f(M);
    for (size_t n = 0; n < E.zi.size(); ++n) {
        const std::complex<double> z0(E.zr[n], E.zi[n]), w0 = -z0 * z0;
        double rad = 1e300;
        for (int j = 0; j < 64; ++j) rad = std::min(rad, std::abs(w0 + (2.0 * j + 1.0) * (2.0 * j + 1.0) * wp));
        const double rho = 0.5 * rad;
        for (int j = 0; j < M; ++j) f[j] = T_of_w(w0 + std::polar(rho, 2.0 * PI * j / M), h);
        double rk = 1.0;
        for (int k = 0; k <= K; ++k) {
            std::complex<double> acc = 0.0;
            for (int j = 0; j < M; ++j) acc += f[j] * std::polar(1.0, -2.0 * PI * ((j * k) % M) / M);
            E.tc[n * sck::TC_LD + k] = acc.real() / M / rk;
            E.tc[n * sck::TC_LD + K + 1 + k] = E.tmode == 2 ? acc.imag() / M / rk : 0.0;
            rk *= rho;
        }
        E.tc[n * sck::TC_LD + 2 * (K + 1)] = rad * rad;
    }
    // Imaginary axis: second table with the nearest pole removed, R(w) = T(w) - (2/h)/(w + wp), analytic out to the
    // second pole: |w - w0| < w0 + 9 wp.  Row = r_0..r_8, (w0 + 9 wp)^2, w0 + wp, 2/h.
    E.tcp.clear();
    if (E.tmode != 1) return;
    E.tcp.assign((size_t)E.zr.size() * sck::TCP_LD, 0.0);
    for (size_t n = 0; n < E.zi.size(); ++n) {
        const double w0 = E.zi[n] * E.zi[n], rad = w0 + 9.0 * wp, rho = 0.5 * rad;
        for (int j = 0; j < M; ++j) {
            const std::complex<double> w = w0 + std::polar(rho, 2.0 * PI * j / M);
            f[j] = T_of_w(w, h) - (2.0 / h) / (w + wp);
        }
        double rk = 1.0;
        for (int k = 0; k <= 8; ++k) {
            std::complex<double> acc = 0.0;
            for (int j = 0; j < M; ++j) acc += f[j] * std::polar(1.0, -2.0 * PI * ((j * k) % M) / M);
            E.tcp[n * sck::TCP_LD + k] = acc.real() / M / rk;
            rk *= rho;
        }
        E.tcp[n * sck::TCP_LD + 9] = rad * rad;
        E.tcp[n * sck::TCP_LD + 10] = w0 + wp;
        E.tcp[n * sck::TCP_LD + 11] = 2.0 / h;
    }
}

}  // namespace

struct sc_ctx {
    std::string err;
    sc_opts opt{};
    sc_grid grid{};
    double t = 0, kappa = -1; int sym = 0;
    int ncomp = 1; int syms[sck::MAX_COMP] = {0, 0, 0, 0}; double tc_ratio[sck::MAX_COMP] = {1, 1, 1, 1};   // Eq. 1 :37 components
    cudaStream_t stream = nullptr;
    bool on_device = false;                       // sc_create reached the device part (false: tables only, every compute call fails)
    int n_sm = 148;
    scgeo::Geometry geo;
    // physical trajectories (k < N/2)
    int G = 0; int smax = 0; long long n_nodes = 0; long long n_pieces_logical = 0;
    std::vector<int> h_k, h_t, h_jf, h_nn, h_dF, h_dB, h_order, h_line_g, h_line_n;
    std::vector<long long> h_noff;
    DevBuf<int> d_k, d_t, d_jf, d_nn, d_dF, d_dB, d_order, d_line_g, d_line_n;
    DevBuf<double> d_l0, d_l1;
    DevBuf<long long> d_noff;
    DevBuf<double> d_vx, d_vy, d_eta, d_W;
    DevBuf<unsigned char> d_mask, d_ga_n;
    DevBuf<int> d_ga_idx; DevBuf<double> d_ga_w;
    // fallback rows
    std::vector<int> fb_rows; std::vector<double> fb_phi;      // mirrored direction of every fallback row
    DevBuf<int> d_fb_rows; DevBuf<double> d_fb_px, d_fb_py, d_fb_dx, d_fb_dy, d_fb_eta;
    DevBuf<double2> d_fb_D; DevBuf<double> d_fb_a;
    // fields
    DevBuf<double2> d_delta; DevBuf<double> d_Ax, d_Ay; bool have_A = false, have_fields = false;
    DevBuf<double> d_Aext_x, d_Aext_y; bool have_Aext = false;
    DevBuf<double2> d_ndD; DevBuf<double> d_nda; DevBuf<float2> d_ndDr; DevBuf<char> d_pc; DevBuf<float2> d_pmax; bool nodes_fresh = false;
    bool f32 = false;            // opts.precision == 32: pc, stores, scratch hold float; ABI buffers stay fp64
    size_t rsz() const { return f32 ? sizeof(float) : sizeof(double); }
    // energies and stores
    EnergySet mats;
    DevBuf<char> d_store[2]; int cur = 0; bool stores_valid = false;      // V2 of R [directed trajectory][energy]
    // scratch
    DevBuf<char> d_scr; long long scr_stride = 0; int n_slots = 0;       // scr_stride in bytes
    DevBuf<double> d_part; DevBuf<int> d_counter; DevBuf<int> d_nbad; DevBuf<int> d_nonfinite; DevBuf<double> d_statmax; DevBuf<unsigned long long> d_nstored;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    static constexpr int MEV = 64;                 // ring of event pairs around the march launches (sc_debug_march_time)
    cudaEvent_t mev[MEV][2] = {}; int mev_n = 0;
    long long march_units = 0;                    // (piece, energy) units of the march launches since the last sc_debug_march_units
    std::string last_variant;                     // template arguments of the most recent march launch (sc_debug_last_march_variant)
    std::set<const void*> smem_opted;             // march instantiations whose dynamic shared memory was opted in on THIS context's device
    // Eq. 22 denominator sum (sum_n w_n t / eps_n over the WHOLE job's energy table) and the energy-shard hook
    double denom_sum = 0.0;
    double* hook_acc = nullptr; sc_allreduce_fn hook_fn = nullptr; void* hook_user = nullptr;
    // sc_ldos: energy table, boundary stores, per-node Re g window and work lists stay alive after the call returns
    // (the call only enqueues); they are re-used by the next sc_ldos and freed by sc_destroy
    EnergySet ldos_E; DevBuf<char> ldos_st[2]; DevBuf<double> ldos_ldn; DevBuf<int> ldos_items, ldos_out_idx;
    // vector potential / driver state
    scf::FieldState fs;
};

namespace {

sc_status fail(sc_ctx* c, sc_status s, const std::string& m) { if (c) c->err = m; return s; }
#define CU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return fail(ctx, e_ == cudaErrorMemoryAllocation ? SC_ERR_NOMEM : SC_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); } while (0)

// every ABI call that touches the device runs on the context's device, whatever the caller's current device is
#define ON_DEVICE(ctx) do { if (!(ctx)->on_device) return fail(ctx, SC_ERR_CUDA, "context has no CUDA device (sc_create failed)"); CU(cudaSetDevice((ctx)->opt.device)); } while (0)

sck::GridDev grid_dev(const sc_ctx* c) {
    return sck::GridDev{c->grid.nx, c->grid.ny, c->grid.h, c->d_mask.p, c->d_delta.p,
                        c->have_A ? c->d_Ax.p : nullptr, c->have_A ? c->d_Ay.p : nullptr, c->ncomp};
}
sck::TrajDev traj_dev(const sc_ctx* c) {
    return sck::TrajDev{c->G, c->d_k.p, c->d_t.p, c->d_jf.p, c->d_nn.p, c->d_l0.p, c->d_l1.p, c->d_noff.p, c->d_dF.p, c->d_dB.p};
}

sc_status upload_energies(sc_ctx* ctx, EnergySet& E) {
    E.ne = (int)E.zr.size();
    E.unit_weights = E.ne % 32 == 0;
    for (double v : E.w) if (v != 1.0) E.unit_weights = false;
    taylor_table(E, ctx->grid.h);
    CU(E.d_tc.upload(E.tc, ctx->stream)); CU(E.d_tcp.upload(E.tcp, ctx->stream));
    CU(E.d_zr.upload(E.zr, ctx->stream)); CU(E.d_zi.upload(E.zi, ctx->stream));
    CU(E.d_w.upload(E.w, ctx->stream)); CU(E.d_partner.upload(E.partner, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return SC_OK;
}

sc_status ensure_nodes(sc_ctx* ctx) {
    if (ctx->nodes_fresh) return SC_OK;
    if (!ctx->have_fields) return fail(ctx, SC_ERR_STATE, "sc_set_fields has not been called");
    const int wpb = 8;
    // n_bad[0]: interpolation points without a valid neighbour found by rotate-in (cleared here, where it is produced);
    // n_bad[1]: by the rotate-back of the current call (cleared by that call)
    CU(cudaMemsetAsync(ctx->d_nbad.p, 0, sizeof(int), ctx->stream));
    if (ctx->f32)
        ++sck::g_launches, sck::rotate_in_kernel<float><<<(ctx->G + wpb - 1) / wpb, wpb * 32, 0, ctx->stream>>>(
            grid_dev(ctx), traj_dev(ctx), ctx->d_vx.p, ctx->d_vy.p, ctx->d_eta.p, ctx->geo.nphi, ctx->geo.c, ctx->opt.charge_sign,
            ctx->d_ndD.p, ctx->d_nda.p, ctx->d_ndDr.p, (float4*)ctx->d_pc.p, ctx->d_pmax.p, ctx->d_nbad.p);
    else
        ++sck::g_launches, sck::rotate_in_kernel<double><<<(ctx->G + wpb - 1) / wpb, wpb * 32, 0, ctx->stream>>>(
            grid_dev(ctx), traj_dev(ctx), ctx->d_vx.p, ctx->d_vy.p, ctx->d_eta.p, ctx->geo.nphi, ctx->geo.c, ctx->opt.charge_sign,
            ctx->d_ndD.p, ctx->d_nda.p, nullptr, (double4*)ctx->d_pc.p, ctx->d_pmax.p, ctx->d_nbad.p);
    if (!ctx->fb_rows.empty()) {
        const int n = (int)ctx->fb_rows.size();
        ++sck::g_launches, sck::fallback_kernel<<<(n + 127) / 128, 128, 0, ctx->stream>>>(grid_dev(ctx), n, ctx->d_fb_rows.p, ctx->d_fb_px.p,
            ctx->d_fb_py.p, ctx->d_fb_dx.p, ctx->d_fb_dy.p, ctx->d_fb_eta.p, ctx->opt.charge_sign, ctx->d_fb_D.p, ctx->d_fb_a.p);
    }
    CU(cudaGetLastError());
    ctx->nodes_fresh = true;
    return SC_OK;
}

template <typename R> const typename sck::VT<R>::V2* node_D(const sc_ctx* ctx);
template <> const double2* node_D<double>(const sc_ctx* ctx) { return ctx->d_ndD.p; }
template <> const float2* node_D<float>(const sc_ctx* ctx) { return ctx->d_ndDr.p; }

template <typename R>
sck::MarchArgsT<R> march_args(sc_ctx* ctx, const EnergySet& E, const char* store_old_raw, char* store_new_raw) {
    using V2 = typename sck::VT<R>::V2; using V4 = typename sck::VT<R>::V4;
    const V2* store_old = (const V2*)store_old_raw; V2* store_new = (V2*)store_new_raw;
    sck::MarchArgsT<R> A{};
    A.T = traj_dev(ctx); A.E = E.dev(); A.order = ctx->d_order.p; A.n_items = ctx->G;
    A.nd_D = node_D<R>(ctx); A.pc = (const V4*)ctx->d_pc.p; A.pmax = ctx->d_pmax.p; A.h = ctx->grid.h; A.bc_mode = ctx->opt.bc_mode;
    A.ga_idx = ctx->d_ga_idx.p; A.ga_w = ctx->d_ga_w.p; A.ga_n = ctx->d_ga_n.p;
    A.fb_D = ctx->d_fb_D.p; A.fb_a = ctx->d_fb_a.p;
    A.store_old = store_old; A.store_new = store_new;
    A.scr = ctx->d_scr.p; A.scr_stride = ctx->scr_stride;
    A.part = ctx->d_part.p; A.ldos = nullptr; A.counter = ctx->d_counter.p; A.stat_max2 = ctx->d_statmax.p; A.n_stored = ctx->d_nstored.p;
    return A;
}

template <int MODE, bool STATS, int STEP, typename R, int TM, bool UW = false>
sc_status launch_march_t(sc_ctx* ctx, const sck::MarchArgsT<R>& A) {
    // persistent grid: one CTA per resident slot of this instantiation (n_slots is sized for the largest, MARCH_MIN_CTAS)
    const int blocks = ctx->n_sm * sck::kMarchCtasPerSm<MODE, STATS, STEP, TM, UW>;
    const int smem = sck::march_smem<R>();
    // the opt-in to > 48 KB of dynamic shared memory is a per-device attribute of the function: remember it per context
    const void* fn = (const void*)sck::march_kernel<MODE, STATS, STEP, R, TM, UW>;
    if (!ctx->smem_opted.count(fn)) {
        CU(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        ctx->smem_opted.insert(fn);
    }
    char name[96];
    std::snprintf(name, sizeof(name), "march_kernel<%d,%s,%d,%s,%d,%s>", MODE, STATS ? "true" : "false", STEP,
                  sizeof(R) == 8 ? "double" : "float", TM, UW ? "true" : "false");
    ctx->last_variant = name;
    cudaEvent_t* ev = ctx->mev[ctx->mev_n % sc_ctx::MEV];
    CU(cudaEventRecord(ev[0], ctx->stream));
    ++sck::g_launches, sck::march_kernel<MODE, STATS, STEP, R, TM, UW><<<blocks, sck::MARCH_WARPS * 32, smem, ctx->stream>>>(A);
    CU(cudaEventRecord(ev[1], ctx->stream));
    ++ctx->mev_n;
    CU(cudaGetLastError());
    return SC_OK;
}

template <int MODE, typename R>
sc_status launch_march_r(sc_ctx* ctx, const EnergySet& E, const char* so, char* sn, bool stats,
                         const int* items, int n_items, double* ldos) {
    sck::MarchArgsT<R> A = march_args<R>(ctx, E, so, sn);
    if (items) { A.order = items; A.n_items = n_items; }
    else ctx->march_units += ctx->n_pieces_logical * E.ne;
    A.ldos = ldos;
    const bool st = stats && MODE == 0;
    // the common case — plain Matsubara sums, unit weights, whole warps of energies — has the weights compiled out
    if (MODE == 0 && !st && ctx->opt.stepper == 0 && E.tmode == 1 && E.unit_weights) return launch_march_t<MODE, false, 0, R, 1, MODE == 0>(ctx, A);
    if (ctx->opt.stepper == 1) return st ? launch_march_t<MODE, MODE == 0, 1, R, 1>(ctx, A) : launch_march_t<MODE, false, 1, R, 1>(ctx, A);
    if (E.tmode == 2) return st ? launch_march_t<MODE, MODE == 0, 0, R, 2>(ctx, A) : launch_march_t<MODE, false, 0, R, 2>(ctx, A);
    return st ? launch_march_t<MODE, MODE == 0, 0, R, 1>(ctx, A) : launch_march_t<MODE, false, 0, R, 1>(ctx, A);
}

// one march launch over the work list (default: all physical trajectories, longest first)
template <int MODE>
sc_status launch_march(sc_ctx* ctx, const EnergySet& E, const char* so, char* sn, bool stats,
                       const int* items = nullptr, int n_items = 0, double* ldos = nullptr) {
    CU(cudaMemsetAsync(ctx->d_counter.p, 0, sizeof(int), ctx->stream));
    return ctx->f32 ? launch_march_r<MODE, float>(ctx, E, so, sn, stats, items, n_items, ldos)
                    : launch_march_r<MODE, double>(ctx, E, so, sn, stats, items, n_items, ldos);
}

sc_status reset_stores(sc_ctx* ctx, const EnergySet& E, char* store) {
    const long long total = (long long)ctx->G * E.ne;
    const unsigned nb = (unsigned)((total + 255) / 256);
    if (ctx->f32) ++sck::g_launches, sck::reset_store_kernel<float><<<nb, 256, 0, ctx->stream>>>(traj_dev(ctx), E.dev(), (const float4*)ctx->d_pc.p, (float2*)store);
    else ++sck::g_launches, sck::reset_store_kernel<double><<<nb, 256, 0, ctx->stream>>>(traj_dev(ctx), E.dev(), (const double4*)ctx->d_pc.p, (double2*)store);
    CU(cudaGetLastError());
    return SC_OK;
}

sck::BackArgs back_args(sc_ctx* ctx, void* delta_new, double* jx, double* jy, double* feI) {
    sck::BackArgs B{};
    B.G = grid_dev(ctx); B.nphi = ctx->geo.nphi; B.nrot = ctx->geo.nrot; B.c = ctx->geo.c;
    B.vx = ctx->d_vx.p; B.vy = ctx->d_vy.p; B.eta = ctx->d_eta.p; B.W = ctx->d_W.p;
    B.line_g = ctx->d_line_g.p; B.line_n = ctx->d_line_n.p; B.T = traj_dev(ctx); B.part = ctx->d_part.p;
    B.t = ctx->t; B.sigma = ctx->opt.charge_sign;
    for (int c = 0; c < sck::MAX_COMP; ++c) B.D[c] = std::log(ctx->t / ctx->tc_ratio[c]) + ctx->denom_sum;
    B.delta_new = (double2*)delta_new; B.jx = jx; B.jy = jy; B.feI = feI; B.n_bad = ctx->d_nbad.p + 1;
    return B;
}

sc_status fill_stats(sc_ctx* ctx, sc_sweep_stats* st, int ne, bool had_stats) {
    if (!st) return SC_OK;
    CU(cudaEventRecord(ctx->ev1, ctx->stream));
    CU(cudaEventSynchronize(ctx->ev1));
    float ms = 0; CU(cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1));
    st->ms = ms;
    int nb[2] = {0, 0}; CU(cudaMemcpy(nb, ctx->d_nbad.p, 2 * sizeof(int), cudaMemcpyDeviceToHost));
    st->n_bad = nb[0] + nb[1];
    st->n_updates = 2LL * 2LL * ctx->n_pieces_logical * ne;     // gamma and gamma-tilde, both angles of every pair
    st->n_updates_executed = 2LL * ctx->n_pieces_logical * ne;
    if (had_stats) {
        std::vector<double> m(ctx->n_slots);
        CU(cudaMemcpy(m.data(), ctx->d_statmax.p, m.size() * sizeof(double), cudaMemcpyDeviceToHost));
        double mx = 0; for (double v : m) mx = std::max(mx, v);
        st->min_one_minus_abs_gamma = 1.0 - std::sqrt(mx);
    }
    return SC_OK;
}

}  // namespace

extern "C" {

const char* sc_version(void) { return SC_VERSION_STR; }
const char* sc_last_error(const sc_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

sc_status sc_create(const sc_grid* grid, const unsigned char* mask, const sc_shape* shapes, int nshapes,
                    double T_over_Tc, double kappa, sc_symmetry symmetry, const sc_opts* opts, sc_ctx** out) {
    if (!out) return SC_ERR_ARG;
    *out = nullptr;
    sc_ctx* ctx = new sc_ctx();
    *out = ctx;     // returned even on failure so that sc_last_error works; the caller still destroys it
    if (!grid || !mask || !shapes || nshapes <= 0 || !opts) return fail(ctx, SC_ERR_ARG, "null argument");
    if (grid->nx < 2 || grid->ny < 2 || !(grid->h > 0)) return fail(ctx, SC_ERR_ARG, "bad grid");
    if (!(T_over_Tc > 0)) return fail(ctx, SC_ERR_ARG, "T/Tc must be positive");
    if (opts->n_matsubara < 1) return fail(ctx, SC_ERR_ARG, "n_matsubara < 1");
    if (opts->precision != 64 && opts->precision != 32 && opts->precision != 0) return fail(ctx, SC_ERR_ARG, "precision must be 64 or 32");
    if (opts->stepper != 0 && opts->stepper != 1) return fail(ctx, SC_ERR_ARG, "stepper must be 0 (closed form) or 1 (implicit mid-point)");
    if (opts->residual_norm != 0 && opts->residual_norm != 2 && opts->residual_norm != 1 && opts->residual_norm != -1)
        return fail(ctx, SC_ERR_ARG, "residual_norm must be 2 (or 0), 1, or -1 (maximum norm)");
    ctx->opt = *opts; ctx->grid = *grid; ctx->t = T_over_Tc; ctx->kappa = kappa; ctx->sym = (int)symmetry;
    ctx->ncomp = 1; ctx->syms[0] = (int)symmetry; ctx->tc_ratio[0] = 1.0;
    ctx->f32 = opts->precision == 32;
    if (ctx->opt.charge_sign == 0) ctx->opt.charge_sign = -1;
    // ---- geometry (host) ----
    scgeo::Geometry& Gm = ctx->geo;
    Gm.nx = grid->nx; Gm.ny = grid->ny; Gm.h = grid->h; Gm.nphi = opts->n_angles;
    for (int s = 0; s < nshapes; ++s) {
        scgeo::ShapeH S{shapes[s].kind, shapes[s].add, shapes[s].cx, shapes[s].cy, shapes[s].r, {}, {}};
        if (S.kind == 1) {
            if (shapes[s].nvert < 3 || !shapes[s].vx || !shapes[s].vy) return fail(ctx, SC_ERR_ARG, "polygon needs >= 3 vertices");
            S.vx.assign(shapes[s].vx, shapes[s].vx + shapes[s].nvert); S.vy.assign(shapes[s].vy, shapes[s].vy + shapes[s].nvert);
        } else if (S.kind != 0) return fail(ctx, SC_ERR_ARG, "unknown shape kind");
        Gm.shapes.push_back(S);
    }
    for (int j = 0; j < grid->ny; ++j)
        for (int i = 0; i < grid->nx; ++i) {
            const double x = (i - 0.5 * (grid->nx - 1)) * grid->h, y = (j - 0.5 * (grid->ny - 1)) * grid->h;
            if ((mask[(size_t)j * grid->nx + i] != 0) != scgeo::in_grain(Gm.shapes, x, y))
                return fail(ctx, SC_ERR_GEOMETRY, "mask disagrees with the shape list");
        }
    if (scgeo::build(Gm, ctx->sym, opts->crystal_rotation, opts->quadrature)) return fail(ctx, SC_ERR_GEOMETRY, Gm.err);
    const int N = Gm.nphi, H = N / 2, NR = Gm.nrot;

    // ---- physical trajectories = directed trajectories of the first half of the angles ----
    ctx->G = Gm.aoff[H];
    if (ctx->G == 0) return fail(ctx, SC_ERR_GEOMETRY, "grain contains no lattice node");
    const int G = ctx->G;
    ctx->h_k.resize(G); ctx->h_t.resize(G); ctx->h_jf.resize(G); ctx->h_nn.resize(G); ctx->h_dF.resize(G); ctx->h_dB.resize(G);
    ctx->h_noff.resize(G); ctx->h_line_g.assign((size_t)H * NR, -1); ctx->h_line_n.assign((size_t)H * NR, 0);
    std::vector<double> l0(G), l1(G);
    long long nodes = 0, pieces = 0; int smax = 0;
    for (int g = 0; g < G; ++g) {
        const scgeo::DTraj& d = Gm.dt[g];
        ctx->h_k[g] = d.k; ctx->h_t[g] = d.t; ctx->h_jf[g] = d.jf; ctx->h_nn[g] = d.jl - d.jf + 1;
        l0[g] = (d.jf - Gm.c) * Gm.h - d.u_in; l1[g] = d.u_out - (d.jl - Gm.c) * Gm.h;
        ctx->h_noff[g] = nodes; nodes += ctx->h_nn[g]; pieces += ctx->h_nn[g] + 1; smax = std::max(smax, ctx->h_nn[g]);
        ctx->h_dF[g] = g;
        // mirror image on angle k+H: line N_rot-1-t, and (holes, concave unions) the intervals of a line in reverse order
        const size_t li = (size_t)d.k * NR + d.t, lm = (size_t)(d.k + H) * NR + (NR - 1 - d.t);
        const int c = g - Gm.line_first[li], cnt = Gm.line_count[li];
        if (Gm.line_first[lm] < 0 || Gm.line_count[lm] != cnt) return fail(ctx, SC_ERR_GEOMETRY, "internal: mirror trajectory missing");
        ctx->h_dB[g] = Gm.line_first[lm] + (cnt - 1 - c);
        if (c == 0) ctx->h_line_g[li] = g;
        ctx->h_line_n[li] = cnt;
    }
    ctx->n_nodes = nodes; ctx->n_pieces_logical = pieces; ctx->smax = smax;
    ctx->h_order.resize(G);
    std::iota(ctx->h_order.begin(), ctx->h_order.end(), 0);
    std::stable_sort(ctx->h_order.begin(), ctx->h_order.end(), [&](int a, int b) { return ctx->h_nn[a] > ctx->h_nn[b]; });

    const int ND = (int)Gm.dt.size();
    std::vector<int> ga_idx((size_t)ND * 4, 0); std::vector<double> ga_w((size_t)ND * 4, 0.0); std::vector<unsigned char> ga_n(ND, 0);
    std::vector<double> fpx, fpy, fdx, fdy, feta;
    for (int d = 0; d < ND; ++d) {
        const scgeo::DTraj& D = Gm.dt[d];
        ga_n[d] = (unsigned char)D.gn;
        for (int i = 0; i < D.gn; ++i) { ga_idx[4 * d + i] = D.gidx[i]; ga_w[4 * d + i] = D.gw[i]; }
        if (D.gn == 0) {
            const double w = (D.t - Gm.c) * Gm.h;
            ctx->fb_rows.push_back(d);
            fpx.push_back(D.u_in * Gm.vx[D.k] - w * Gm.vy[D.k]); fpy.push_back(D.u_in * Gm.vy[D.k] + w * Gm.vx[D.k]);
            fdx.push_back(D.mdir[0]); fdy.push_back(D.mdir[1]);
            ctx->fb_phi.push_back(std::atan2(D.mdir[1], D.mdir[0]));
            feta.push_back(scgeo::eta_of(ctx->sym, ctx->fb_phi.back(), opts->crystal_rotation));
        }
    }

    // ---- device ---- (the host tables above stay inspectable through sc_debug_tables even when this fails)
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(ctx, SC_ERR_CUDA, "no CUDA device: this library has no CPU path");
    CU(cudaSetDevice(opts->device));
    ctx->on_device = true;
    cudaDeviceProp prop; CU(cudaGetDeviceProperties(&prop, opts->device));
    ctx->n_sm = prop.multiProcessorCount;
    ctx->stream = (cudaStream_t)opts->cuda_stream;
    CU(cudaEventCreate(&ctx->ev0)); CU(cudaEventCreate(&ctx->ev1));
    for (auto& e : ctx->mev) { CU(cudaEventCreate(&e[0])); CU(cudaEventCreate(&e[1])); }

    // ---- upload ----
    cudaStream_t s = ctx->stream;
    std::vector<unsigned char> hm(mask, mask + (size_t)grid->nx * grid->ny);
    CU(ctx->d_mask.upload(hm, s));
    CU(ctx->d_k.upload(ctx->h_k, s)); CU(ctx->d_t.upload(ctx->h_t, s)); CU(ctx->d_jf.upload(ctx->h_jf, s)); CU(ctx->d_nn.upload(ctx->h_nn, s));
    CU(ctx->d_dF.upload(ctx->h_dF, s)); CU(ctx->d_dB.upload(ctx->h_dB, s)); CU(ctx->d_order.upload(ctx->h_order, s));
    CU(ctx->d_line_g.upload(ctx->h_line_g, s)); CU(ctx->d_line_n.upload(ctx->h_line_n, s)); CU(ctx->d_l0.upload(l0, s)); CU(ctx->d_l1.upload(l1, s)); CU(ctx->d_noff.upload(ctx->h_noff, s));
    CU(ctx->d_vx.upload(Gm.vx, s)); CU(ctx->d_vy.upload(Gm.vy, s)); CU(ctx->d_eta.upload(Gm.eta, s)); CU(ctx->d_W.upload(Gm.W, s));
    CU(ctx->d_ga_idx.upload(ga_idx, s)); CU(ctx->d_ga_w.upload(ga_w, s)); CU(ctx->d_ga_n.upload(ga_n, s));
    CU(ctx->d_fb_rows.upload(ctx->fb_rows, s)); CU(ctx->d_fb_px.upload(fpx, s)); CU(ctx->d_fb_py.upload(fpy, s));
    CU(ctx->d_fb_dx.upload(fdx, s)); CU(ctx->d_fb_dy.upload(fdy, s)); CU(ctx->d_fb_eta.upload(feta, s));
    CU(ctx->d_fb_D.alloc(ND)); CU(ctx->d_fb_a.alloc(ND));
    CU(cudaMemsetAsync(ctx->d_fb_D.p, 0, ND * sizeof(double2), s)); CU(cudaMemsetAsync(ctx->d_fb_a.p, 0, ND * sizeof(double), s));

    const size_t ng = (size_t)grid->nx * grid->ny;
    CU(ctx->d_delta.alloc(ng)); CU(ctx->d_Ax.alloc(ng)); CU(ctx->d_Ay.alloc(ng));
    CU(ctx->d_ndD.alloc(nodes)); CU(ctx->d_nda.alloc(nodes)); CU(ctx->d_pc.alloc((size_t)(nodes + G) * 4 * ctx->rsz())); CU(ctx->d_pmax.alloc(G));
    if (ctx->f32) CU(ctx->d_ndDr.alloc(nodes));
    CU(ctx->d_part.alloc((size_t)nodes * sck::RED_VALS));
    CU(ctx->d_counter.alloc(1)); CU(ctx->d_nbad.alloc(2)); CU(ctx->d_nonfinite.alloc(1)); CU(ctx->d_nstored.alloc(2));
    CU(cudaMemsetAsync(ctx->d_nbad.p, 0, 2 * sizeof(int), s)); CU(cudaMemsetAsync(ctx->d_nstored.p, 0, 2 * sizeof(unsigned long long), s));

    // Matsubara energies eps_n = t(n+1/2) (:98), unit weights, self-partnered (z = i eps -> -conj z = z)
    EnergySet& E = ctx->mats;
    for (int n = 0; n < opts->n_matsubara; ++n) { E.zr.push_back(0.0); E.zi.push_back(T_over_Tc * (n + 0.5)); E.w.push_back(1.0); E.partner.push_back(n); }
    if (sc_status st = upload_energies(ctx, E)) return st;
    for (int n = 0; n < opts->n_matsubara; ++n) ctx->denom_sum += 1.0 / (n + 0.5);
    CU(ctx->d_store[0].alloc((size_t)ND * E.ne * 2 * ctx->rsz())); CU(ctx->d_store[1].alloc((size_t)ND * E.ne * 2 * ctx->rsz()));

    // persistent march grid: MARCH_MIN_CTAS CTAs of 8 warps per SM; per-warp scratch of smax + 1 (+2 spare) entries x 32 lanes
    // x {T, gamma~} (rounds that recompute T in pass 2 use half of each row's bytes)
    ctx->n_slots = ctx->n_sm * sck::MARCH_MIN_CTAS * sck::MARCH_WARPS;
    ctx->scr_stride = (long long)(smax + 3) * 32 * 4 * (long long)ctx->rsz();
    CU(ctx->d_scr.alloc((size_t)ctx->n_slots * ctx->scr_stride + 16384));   // + 16 KB: the L2 prefetch of the last slot may run past its end
    CU(ctx->d_statmax.alloc(ctx->n_slots));
    CU(cudaMemsetAsync(ctx->d_statmax.p, 0, ctx->n_slots * sizeof(double), s));
    CU(cudaStreamSynchronize(s));
    return SC_OK;
}

sc_status sc_destroy(sc_ctx* ctx) {
    if (!ctx) return SC_ERR_ARG;
    if (ctx->ev0) cudaEventDestroy(ctx->ev0);
    if (ctx->ev1) cudaEventDestroy(ctx->ev1);
    for (auto& e : ctx->mev) { if (e[0]) cudaEventDestroy(e[0]); if (e[1]) cudaEventDestroy(e[1]); }
    scf::release(ctx->fs);
    delete ctx;
    return SC_OK;
}

sc_status sc_set_fields(sc_ctx* ctx, const void* delta, const double* Ax, const double* Ay) {
    if (!ctx || !delta) return fail(ctx, SC_ERR_ARG, "null argument");
    ON_DEVICE(ctx);
    const size_t ng = (size_t)ctx->grid.nx * ctx->grid.ny;
    CU(cudaMemcpyAsync(ctx->d_delta.p, delta, ctx->ncomp * ng * sizeof(double2), cudaMemcpyDeviceToDevice, ctx->stream));
    ctx->have_A = Ax && Ay;
    if (ctx->have_A) {
        CU(cudaMemcpyAsync(ctx->d_Ax.p, Ax, ng * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
        CU(cudaMemcpyAsync(ctx->d_Ay.p, Ay, ng * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    }
    ctx->have_fields = true; ctx->nodes_fresh = false;
    return SC_OK;
}

sc_status sc_set_components(sc_ctx* ctx, int n, const sc_symmetry* symmetries, const double* tc_ratio) {
    if (!ctx || !symmetries || !tc_ratio) return fail(ctx, SC_ERR_ARG, "null argument");
    if (n < 1 || n > sck::MAX_COMP) return fail(ctx, SC_ERR_ARG, "1 <= n_components <= 4");
    ON_DEVICE(ctx);
    const int N = ctx->geo.nphi; const size_t ng = (size_t)ctx->grid.nx * ctx->grid.ny, nfb = ctx->fb_rows.size();
    std::vector<double> eta((size_t)n * N), feta((size_t)n * nfb);
    for (int c = 0; c < n; ++c) {
        if ((int)symmetries[c] < 0 || (int)symmetries[c] > 3) return fail(ctx, SC_ERR_ARG, "unknown symmetry");
        if (!(tc_ratio[c] > 0) || tc_ratio[c] > 1.0) return fail(ctx, SC_ERR_ARG, "tc_ratio must lie in (0, 1]: T_c is the largest T_c^G");
        for (int k = 0; k < N; ++k) eta[(size_t)c * N + k] = scgeo::eta_of((int)symmetries[c], 2.0 * scgeo::kPi * k / N, ctx->opt.crystal_rotation);
        for (size_t i = 0; i < nfb; ++i) feta[c * nfb + i] = scgeo::eta_of((int)symmetries[c], ctx->fb_phi[i], ctx->opt.crystal_rotation);
    }
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->ncomp = n;
    for (int c = 0; c < sck::MAX_COMP; ++c) { ctx->syms[c] = c < n ? (int)symmetries[c] : 0; ctx->tc_ratio[c] = c < n ? tc_ratio[c] : 1.0; }
    ctx->sym = ctx->syms[0];
    CU(ctx->d_eta.upload(eta, ctx->stream)); CU(ctx->d_fb_eta.upload(feta, ctx->stream));
    CU(ctx->d_delta.alloc(n * ng));
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->have_fields = false; ctx->nodes_fresh = false; ctx->stores_valid = false;
    scf::release_driver(ctx->fs);                      // the iterate's length changes with the number of components
    return SC_OK;
}

sc_status sc_set_energies(sc_ctx* ctx, const double* z_re, const double* z_im, const double* w, int n, double denominator_sum) {
    if (!ctx || !z_re || !z_im || !w || n < 1) return fail(ctx, SC_ERR_ARG, "bad argument");
    ON_DEVICE(ctx);
    // validate into locals: on SC_ERR_ARG the context keeps its previous table, untouched
    std::vector<int> partner(n, -1);
    double ds = 0.0;
    for (int m = 0; m < n; ++m) {
        if (!(z_im[m] > 0)) return fail(ctx, SC_ERR_ARG, "energies must lie in the upper half plane");
        ds += w[m] * ctx->t / z_im[m];
        // partner: -conj(z) (Eq. 13 :95); Matsubara / Ozaki energies on the imaginary axis are their own partner
        for (int q = 0; q < n; ++q)
            if (std::fabs(z_re[q] + z_re[m]) <= 1e-12 * (1.0 + std::fabs(z_re[m])) && std::fabs(z_im[q] - z_im[m]) <= 1e-12 * z_im[m]) { partner[m] = q; break; }
        if (partner[m] < 0) return fail(ctx, SC_ERR_ARG, "energy table is not closed under z -> -conj(z)");
        // the sums of angle k + N/2 are taken from the partner energies of angle k (Eq. 13): partners must weigh the same
        if (std::fabs(w[partner[m]] - w[m]) > 1e-12 * std::fabs(w[m])) return fail(ctx, SC_ERR_ARG, "partner energies z and -conj(z) must have equal weights");
    }
    for (int m = 0; m < n; ++m)
        if (partner[partner[m]] != m) return fail(ctx, SC_ERR_ARG, "duplicate energies: z -> -conj(z) is not an involution on the table");
    EnergySet& E = ctx->mats;
    E.zr.assign(z_re, z_re + n); E.zi.assign(z_im, z_im + n); E.w.assign(w, w + n); E.partner = partner;
    ctx->denom_sum = std::isnan(denominator_sum) ? ds : denominator_sum;
    if (sc_status st = upload_energies(ctx, E)) return st;
    const size_t ND = ctx->geo.dt.size();
    CU(ctx->d_store[0].alloc(ND * E.ne * 2 * ctx->rsz())); CU(ctx->d_store[1].alloc(ND * E.ne * 2 * ctx->rsz()));
    ctx->stores_valid = false; ctx->cur = 0;
    return SC_OK;
}

sc_status sc_set_allreduce_hook(sc_ctx* ctx, double* acc, sc_allreduce_fn fn, void* user) {
    if (!ctx || ((fn != nullptr) != (acc != nullptr))) return fail(ctx, SC_ERR_ARG, "hook and accumulator buffer must be given together");
    ctx->hook_acc = acc; ctx->hook_fn = fn; ctx->hook_user = user;
    return SC_OK;
}

sc_status sc_reset_boundary(sc_ctx* ctx) {
    if (!ctx) return SC_ERR_ARG;
    ON_DEVICE(ctx);
    if (sc_status st = ensure_nodes(ctx)) return st;
    if (sc_status st = reset_stores(ctx, ctx->mats, ctx->d_store[ctx->cur].p)) return st;
    ctx->stores_valid = true;
    return SC_OK;
}

sc_status sc_riccati_sweep(sc_ctx* ctx, void* delta_new, double* jx, double* jy, double* fe_I, sc_sweep_stats* stats) {
    if (!ctx) return SC_ERR_ARG;
    if (!ctx->have_fields) return fail(ctx, SC_ERR_STATE, "sc_riccati_sweep before sc_set_fields");
    ON_DEVICE(ctx);
    if (stats) CU(cudaEventRecord(ctx->ev0, ctx->stream));
    CU(cudaMemsetAsync(ctx->d_nbad.p + 1, 0, sizeof(int), ctx->stream));
    if (sc_status st = ensure_nodes(ctx)) return st;
    if (!ctx->stores_valid) { if (sc_status st = sc_reset_boundary(ctx)) return st; }
    if (sc_status st = launch_march<0>(ctx, ctx->mats, ctx->d_store[ctx->cur].p, ctx->d_store[ctx->cur ^ 1].p, stats != nullptr)) return st;
    ctx->cur ^= 1;
    sck::BackArgs B = back_args(ctx, delta_new, jx, jy, fe_I);
    B.raw = ctx->hook_fn ? ctx->hook_acc : nullptr;
    dim3 grd((ctx->grid.nx + sck::BACK_TX - 1) / sck::BACK_TX, (ctx->grid.ny + sck::BACK_TY - 1) / sck::BACK_TY);
    ++sck::g_launches, sck::rotate_back_kernel<<<grd, dim3(sck::BACK_TX, sck::BACK_TY), 0, ctx->stream>>>(B);
    CU(cudaGetLastError());
    if (ctx->hook_fn) {
        // energy-sharded sweep: the caller sums the raw accumulators of all shards on this stream, then a7 runs
        ctx->hook_fn(ctx->hook_user);
        const size_t ng = (size_t)ctx->grid.nx * ctx->grid.ny;
        sck::FinArgs FA; for (int c = 0; c < sck::MAX_COMP; ++c) FA.D[c] = B.D[c];
        ++sck::g_launches, sck::finalise_kernel<<<(unsigned)((ng + 255) / 256), 256, 0, ctx->stream>>>(ng, ctx->ncomp, ctx->hook_acc, ctx->t, FA, ctx->opt.charge_sign,
                                                                                  (double2*)delta_new, jx, jy, fe_I);
        CU(cudaGetLastError());
    }
    if (stats) {          // SC_ERR_NUMERIC: a reduced field is not finite (checked only where the call synchronises anyway)
        const size_t ng = (size_t)ctx->grid.nx * ctx->grid.ny;
        CU(cudaMemsetAsync(ctx->d_nonfinite.p, 0, sizeof(int), ctx->stream));
        const double* fields[4] = {(const double*)delta_new, jx, jy, fe_I};
        const size_t counts[4] = {2 * ng * ctx->ncomp, ng, ng, ng};
        for (int f = 0; f < 4; ++f)
            if (fields[f]) ++sck::g_launches, sck::nonfinite_kernel<<<(unsigned)((counts[f] + 255) / 256), 256, 0, ctx->stream>>>(counts[f], fields[f], ctx->d_nonfinite.p);
        CU(cudaGetLastError());
        if (sc_status st = fill_stats(ctx, stats, ctx->mats.ne, true)) return st;
        int bad = 0; CU(cudaMemcpy(&bad, ctx->d_nonfinite.p, sizeof(int), cudaMemcpyDeviceToHost));
        if (bad) return fail(ctx, SC_ERR_NUMERIC, std::to_string(bad) + " non-finite values in the sweep's output fields");
        return SC_OK;
    }
    return SC_OK;
}

sc_status sc_ldos(sc_ctx* ctx, const double* energies, int n_e, double broadening, int n_boundary_iters,
                  double* ldos, sc_sweep_stats* stats) {
    if (!ctx || !energies || n_e < 1 || !ldos) return fail(ctx, SC_ERR_ARG, "bad argument");
    if (!(broadening > 0)) return fail(ctx, SC_ERR_ARG, "broadening must be positive");
    if (n_boundary_iters < 1) return fail(ctx, SC_ERR_ARG, "n_boundary_iters < 1");
    if (!ctx->have_fields) return fail(ctx, SC_ERR_STATE, "sc_ldos before sc_set_fields");
    ON_DEVICE(ctx);
    if (stats) CU(cudaEventRecord(ctx->ev0, ctx->stream));
    CU(cudaMemsetAsync(ctx->d_nbad.p + 1, 0, sizeof(int), ctx->stream));
    if (sc_status st = ensure_nodes(ctx)) return st;
    // internal energy list closed under eps -> -eps (gamma-tilde_k(eps) = conj gamma_{k+N/2}(-eps), Eq. 13 :95)
    CU(cudaStreamSynchronize(ctx->stream));       // an earlier sc_ldos may still be reading the tables replaced below
    EnergySet& E = ctx->ldos_E;
    E.zr.clear(); E.zi.clear(); E.w.clear();
    std::vector<int> out_idx(n_e);
    for (int m = 0; m < n_e; ++m) { E.zr.push_back(energies[m]); E.zi.push_back(broadening); E.w.push_back(1.0); out_idx[m] = m; }
    E.partner.assign(n_e, -1);
    for (int m = 0; m < n_e; ++m) {
        if (E.partner[m] >= 0) continue;
        // the first still unpaired energy equal to -eps_m (eps = 0 pairs with itself; repeated energies pair off one by one)
        int best = -1; const double bd = 1e-12 * (1.0 + std::fabs(energies[m]));
        for (int q = 0; q < (int)E.zr.size(); ++q) if (E.partner[q] < 0 && std::fabs(E.zr[q] + energies[m]) <= bd && (q != m || energies[m] == 0.0)) { best = q; break; }
        if (best < 0 && std::fabs(energies[m]) <= bd) best = m;
        if (best < 0) { best = (int)E.zr.size(); E.zr.push_back(-energies[m]); E.zi.push_back(broadening); E.w.push_back(0.0); E.partner.push_back(m); }
        E.partner[m] = best; E.partner[best] = m;
    }
    if (sc_status st = upload_energies(ctx, E)) return st;
    const int ND = (int)ctx->geo.dt.size();
    const size_t store_bytes = (size_t)ND * E.ne * 2 * ctx->rsz();
    for (auto& b : ctx->ldos_st) if (b.n < store_bytes) CU(b.alloc(store_bytes));
    if (sc_status st = reset_stores(ctx, E, ctx->ldos_st[0].p)) return st;
    char* so = ctx->ldos_st[0].p; char* sn = ctx->ldos_st[1].p;
    for (int it = 0; it + 1 < n_boundary_iters; ++it) {
        if (sc_status st = launch_march<2>(ctx, E, so, sn, false)) return st;
        std::swap(so, sn);
    }
    // last sweep: per-energy Re g at every node, in batches of angle pairs sized to the free memory.  Node offsets are
    // pair-major, so the nodes of a batch are one contiguous window; all batches share one window buffer and run back to
    // back on the stream (stream order keeps a batch's march behind the previous batch's rotate-back: no host sync).
    const int H = ctx->geo.nphi / 2;
    std::vector<long long> pair_nodes(H + 1, 0);
    for (int g = 0; g < ctx->G; ++g) pair_nodes[ctx->h_k[g] + 1] += ctx->h_nn[g];
    for (int p = 0; p < H; ++p) pair_nodes[p + 1] += pair_nodes[p];
    size_t freeb = 0, totalb = 0; CU(cudaMemGetInfo(&freeb, &totalb));
    const size_t budget = std::max(ctx->ldos_ldn.n * sizeof(double), std::min<size_t>(freeb / 2, (size_t)48 << 30));
    std::vector<int> bounds{0};
    long long win_max = 0;
    for (int p0 = 0; p0 < H;) {
        int p1 = p0 + 1;
        while (p1 < H && (size_t)(pair_nodes[p1 + 1] - pair_nodes[p0]) * E.ne * sizeof(double) <= budget) ++p1;
        win_max = std::max(win_max, pair_nodes[p1] - pair_nodes[p0]);
        bounds.push_back(p1); p0 = p1;
    }
    if (ctx->ldos_ldn.n < (size_t)win_max * E.ne) CU(ctx->ldos_ldn.alloc((size_t)win_max * E.ne));
    // work lists of all batches, each longest-first, concatenated
    std::vector<int> items; std::vector<int> item_off{0};
    for (size_t b = 0; b + 1 < bounds.size(); ++b) {
        for (int g : ctx->h_order) if (ctx->h_k[g] >= bounds[b] && ctx->h_k[g] < bounds[b + 1]) items.push_back(g);
        item_off.push_back((int)items.size());
    }
    CU(ctx->ldos_items.upload(items, ctx->stream)); CU(ctx->ldos_out_idx.upload(out_idx, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));       // `items` / `out_idx` are stack-owned host vectors
    for (size_t b = 0; b + 1 < bounds.size(); ++b) {
        const int p0 = bounds[b], p1 = bounds[b + 1];
        double* const ldn = ctx->ldos_ldn.p - (size_t)pair_nodes[p0] * E.ne;       // node offsets are global
        if (sc_status st = launch_march<1>(ctx, E, so, sn, false, ctx->ldos_items.p + item_off[b], item_off[b + 1] - item_off[b], ldn)) return st;
        sck::BackLdosArgs L{};
        L.B = back_args(ctx, nullptr, nullptr, nullptr, nullptr);
        L.ne_out = n_e; L.out_idx = ctx->ldos_out_idx.p; L.partner = E.d_partner.p; L.ne = E.ne;
        L.ldos_nodes = ldn; L.out = ldos; L.p0 = p0; L.p1 = p1; L.accumulate = b ? 1 : 0;
        dim3 grd((n_e + 63) / 64, ctx->grid.nx, ctx->grid.ny);
        ++sck::g_launches, sck::rotate_back_ldos_kernel<<<grd, 64, 0, ctx->stream>>>(L);
        CU(cudaGetLastError());
    }
    sc_status r = fill_stats(ctx, stats, E.ne, false);
    if (stats) { stats->n_updates *= n_boundary_iters; stats->n_updates_executed *= n_boundary_iters; }
    return r;
}

sc_status sc_set_external_field(sc_ctx* ctx, const double* Ax, const double* Ay) {
    if (!ctx) return SC_ERR_ARG;
    ON_DEVICE(ctx);
    const size_t ng = (size_t)ctx->grid.nx * ctx->grid.ny;
    ctx->have_Aext = Ax && Ay;
    if (ctx->have_Aext) {
        CU(ctx->d_Aext_x.alloc(ng)); CU(ctx->d_Aext_y.alloc(ng));
        CU(cudaMemcpyAsync(ctx->d_Aext_x.p, Ax, ng * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
        CU(cudaMemcpyAsync(ctx->d_Aext_y.p, Ay, ng * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    }
    return SC_OK;
}

sc_status sc_update_vector_potential(sc_ctx* ctx, const double* jx, const double* jy, double* Ax, double* Ay, double* fe_mag) {
    if (!ctx || !jx || !jy || !Ax || !Ay) return fail(ctx, SC_ERR_ARG, "null argument");
    ON_DEVICE(ctx);
    std::string e;
    int rc = scf::vector_potential(ctx->fs, ctx->grid.nx, ctx->grid.ny, ctx->grid.h, ctx->d_mask.p, ctx->kappa, jx, jy, Ax, Ay, fe_mag, ctx->stream, e);
    if (rc) return fail(ctx, rc == 2 ? SC_ERR_NOMEM : SC_ERR_CUDA, e);
    return SC_OK;
}

sc_status sc_iterate(sc_ctx* ctx, int accelerator, double step, int burnin, void* delta_inout, double* Aix, double* Aiy, sc_sweep_stats* stats) {
    if (!ctx || !delta_inout) return fail(ctx, SC_ERR_ARG, "null argument");
    if (accelerator < 0 || accelerator > 3) return fail(ctx, SC_ERR_ARG, "accelerator must be 0 (Picard), 1 (Barzilai-Borwein), 2 (Polyak) or 3 (CongAcc)");
    ON_DEVICE(ctx);
    const int nx = ctx->grid.nx, ny = ctx->grid.ny; const size_t ng = (size_t)nx * ny;
    const bool withA = ctx->kappa > 0 && Aix && Aiy;
    std::string e;
    if (int rc = scf::ensure_driver(ctx->fs, ng, ctx->ncomp, e)) return fail(ctx, rc == 2 ? SC_ERR_NOMEM : SC_ERR_CUDA, e);
    if (stats) CU(cudaEventRecord(ctx->ev0, ctx->stream));
    // total A = A_ext + A_ind
    scf::FieldState& F = ctx->fs;
    const double* Atx = nullptr; const double* Aty = nullptr;
    if (ctx->have_Aext || (Aix && Aiy)) {
        scf::add_fields(F.Atot_x, F.Atot_y, ctx->have_Aext ? ctx->d_Aext_x.p : nullptr, ctx->have_Aext ? ctx->d_Aext_y.p : nullptr, Aix, Aiy, ng, ctx->stream);
        Atx = F.Atot_x; Aty = F.Atot_y;
    }
    if (sc_status st = sc_set_fields(ctx, delta_inout, Atx, Aty)) return st;
    if (sc_status st = sc_riccati_sweep(ctx, F.dnew, F.jx, F.jy, F.feI, nullptr)) return st;
    if (!burnin) {
        if (withA) {
            if (int rc = scf::vector_potential(F, nx, ny, ctx->grid.h, ctx->d_mask.p, ctx->kappa, F.jx, F.jy, F.gAx, F.gAy, nullptr, ctx->stream, e))
                return fail(ctx, rc == 2 ? SC_ERR_NOMEM : SC_ERR_CUDA, e);
        }
        if (int rc = scf::mix(F, accelerator, step, ctx->kappa, withA, (double2*)delta_inout, Aix, Aiy, ctx->d_mask.p, ng, ctx->opt.residual_norm, ctx->stream, e))
            return fail(ctx, SC_ERR_CUDA, e);
    }
    if (stats) {
        if (sc_status st = fill_stats(ctx, stats, ctx->mats.ne, false)) return st;
        double r[4] = {0, 0, 0, 0};
        if (!burnin) { if (int rc = scf::read_residuals(F, r, ctx->stream, e)) return fail(ctx, SC_ERR_CUDA, e); }
        stats->res_delta = r[0]; stats->res_A = r[1]; stats->res_j = r[2]; stats->res_fe = r[3];
        stats->min_one_minus_abs_gamma = 0.0;
        if (!std::isfinite(r[0]) || !std::isfinite(r[1]) || !std::isfinite(r[2]) || !std::isfinite(r[3]))
            return fail(ctx, SC_ERR_NUMERIC, "non-finite residual: the iterate has diverged or an input field is not finite");
    }
    return SC_OK;
}

sc_status sc_set_vector_potential_error(sc_ctx* ctx, double eps, int* n_kept) {
    if (!ctx || !(eps >= 0.0) || eps >= 1.0) return fail(ctx, SC_ERR_ARG, "vector_potential_error must lie in [0, 1)");
    ctx->fs.vp_eps = eps;
    if (n_kept) {
        *n_kept = 0;
        if (eps > 0.0) {
            ON_DEVICE(ctx);
            std::string e;
            if (!ctx->fs.lr) ctx->fs.lr = new scf::LowRank();
            if (int rc = scf::ensure_lowrank(*ctx->fs.lr, ctx->grid.nx, ctx->grid.ny, ctx->grid.h, eps, ctx->stream, e))
                return fail(ctx, rc == 2 ? SC_ERR_NOMEM : SC_ERR_CUDA, e);
            *n_kept = ctx->fs.lr->nstar;
        }
    }
    return SC_OK;
}

sc_status sc_set_accelerator_params(sc_ctx* ctx, double drag, double step_factor, double cos_similarity_min,
                                    double step_min, double step_max) {
    if (!ctx) return SC_ERR_ARG;
    scf::AccelParams P = ctx->fs.par;
    if (drag > 0) { if (drag > 1) return fail(ctx, SC_ERR_ARG, "drag must lie in (0, 1]"); P.drag = drag; }
    if (step_factor > 0) { if (step_factor < 1) return fail(ctx, SC_ERR_ARG, "step_factor must be >= 1"); P.kfac = step_factor; }
    if (cos_similarity_min > 0) { if (cos_similarity_min >= 1) return fail(ctx, SC_ERR_ARG, "cos_similarity_min must be < 1"); P.smin = cos_similarity_min; }
    if (step_min > 0) P.amin = step_min;
    if (step_max > 0) P.amax = step_max;
    if (!(P.amin <= P.amax)) return fail(ctx, SC_ERR_ARG, "step_min > step_max");
    ctx->fs.par = P;
    return SC_OK;
}

// ---------------------------------------------------------------------------------------------- debug
sc_status sc_debug_geometry(sc_ctx* ctx, int* n_rot, int* n_traj_total, long long* n_pieces_total) {
    if (!ctx) return SC_ERR_ARG;
    if (n_rot) *n_rot = ctx->geo.nrot;
    if (n_traj_total) *n_traj_total = (int)ctx->geo.dt.size();
    if (n_pieces_total) *n_pieces_total = 2 * ctx->n_pieces_logical;
    return SC_OK;
}

sc_status sc_debug_tables(sc_ctx* ctx, int k, int* n, int* it, double* dt, int* gidx, double* gw) {
    if (!ctx || k < 0 || k >= ctx->geo.nphi || !n) return fail(ctx, SC_ERR_ARG, "bad argument");
    const int a = ctx->geo.aoff[k], b = ctx->geo.aoff[k + 1];
    *n = b - a;
    if (!it) return SC_OK;
    for (int d = a; d < b; ++d) {
        const scgeo::DTraj& D = ctx->geo.dt[d]; const int i = d - a;
        it[6 * i + 0] = D.t; it[6 * i + 1] = D.jf; it[6 * i + 2] = D.jl; it[6 * i + 3] = D.elem_in; it[6 * i + 4] = D.elem_out; it[6 * i + 5] = 0;
        dt[2 * i + 0] = D.u_in; dt[2 * i + 1] = D.u_out;
        for (int q = 0; q < 4; ++q) { gidx[4 * i + q] = q < D.gn ? D.gidx[q] : -1; gw[4 * i + q] = q < D.gn ? D.gw[q] : 0.0; }
    }
    return SC_OK;
}

sc_status sc_debug_trajectory(sc_ctx* ctx, int k, int local, int n_energy, int* n_nodes, void* gamma, void* gamma_tilde) {
    if (!ctx || k < 0 || k >= ctx->geo.nphi / 2) return fail(ctx, SC_ERR_ARG, "k must be < n_angles/2");
    ON_DEVICE(ctx);
    const int g = ctx->geo.aoff[k] + local;
    if (local < 0 || g >= ctx->geo.aoff[k + 1] || n_energy < 0 || n_energy >= ctx->mats.ne) return fail(ctx, SC_ERR_ARG, "bad index");
    if (!ctx->stores_valid) return fail(ctx, SC_ERR_STATE, "no sweep has been run");
    const int nn = ctx->h_nn[g];
    DevBuf<double2> dG, dGT; CU(dG.alloc(nn)); CU(dGT.alloc(nn));
    // the last sweep read store[cur^1] (now the "new" side) and wrote store[cur]
    if (ctx->f32) ++sck::g_launches, sck::debug_traj_kernel<float><<<1, 32, 0, ctx->stream>>>(march_args<float>(ctx, ctx->mats, ctx->d_store[ctx->cur ^ 1].p, nullptr), ctx->opt.stepper, g, n_energy, dG.p, dGT.p);
    else ++sck::g_launches, sck::debug_traj_kernel<double><<<1, 32, 0, ctx->stream>>>(march_args<double>(ctx, ctx->mats, ctx->d_store[ctx->cur ^ 1].p, nullptr), ctx->opt.stepper, g, n_energy, dG.p, dGT.p);
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(gamma, dG.p, nn * sizeof(double2), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaMemcpyAsync(gamma_tilde, dGT.p, nn * sizeof(double2), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    if (n_nodes) *n_nodes = nn;
    return SC_OK;
}

sc_status sc_debug_partial(sc_ctx* ctx, int k, void* SF, double* SG, double* SI) {
    if (!ctx || k < 0 || k >= ctx->geo.nphi || !SF || !SG || !SI) return fail(ctx, SC_ERR_ARG, "bad argument");
    ON_DEVICE(ctx);
    const int H = ctx->geo.nphi / 2, NR = ctx->geo.nrot, p = k % H;
    const int g0 = ctx->geo.aoff[p], g1 = ctx->geo.aoff[p + 1];
    if (g1 == g0) return SC_OK;
    const long long n0 = ctx->h_noff[g0], n1 = ctx->h_noff[g1 - 1] + ctx->h_nn[g1 - 1];
    std::vector<double> buf((size_t)(n1 - n0) * sck::RED_VALS);
    CU(cudaStreamSynchronize(ctx->stream));
    CU(cudaMemcpy(buf.data(), ctx->d_part.p + (size_t)n0 * sck::RED_VALS, buf.size() * sizeof(double), cudaMemcpyDeviceToHost));
    double* sf = (double*)SF;
    std::fill(sf, sf + 2 * (size_t)NR * NR, 0.0); std::fill(SG, SG + (size_t)NR * NR, 0.0); std::fill(SI, SI + (size_t)NR * NR, 0.0);
    for (int g = g0; g < g1; ++g)
        for (int m = 0; m < ctx->h_nn[g]; ++m) {
            const double* v = &buf[(size_t)(ctx->h_noff[g] - n0 + m) * sck::RED_VALS];
            int t = ctx->h_t[g], j = ctx->h_jf[g] + m;
            if (k < H) { const size_t q = (size_t)t * NR + j; sf[2 * q] = v[0]; sf[2 * q + 1] = v[1]; SG[q] = 2.0 * v[4]; SI[q] = v[5]; }
            else { const size_t q = (size_t)(NR - 1 - t) * NR + (NR - 1 - j); sf[2 * q] = v[2]; sf[2 * q + 1] = -v[3]; SG[q] = -2.0 * v[4]; SI[q] = v[5]; }
        }
    return SC_OK;
}

sc_status sc_debug_stores(sc_ctx* ctx, int k, void* gamma_end, void* gamma_tilde_end) {
    if (!ctx || k < 0 || k >= ctx->geo.nphi || !gamma_end || !gamma_tilde_end) return fail(ctx, SC_ERR_ARG, "bad argument");
    ON_DEVICE(ctx);
    if (!ctx->stores_valid) return fail(ctx, SC_ERR_STATE, "no sweep has been run");
    const int H = ctx->geo.nphi / 2, ne = ctx->mats.ne, km = (k + H) % ctx->geo.nphi;
    const int a0 = ctx->geo.aoff[k], a1 = ctx->geo.aoff[k + 1], m0 = ctx->geo.aoff[km], m1 = ctx->geo.aoff[km + 1];
    if (a1 - a0 != m1 - m0) return fail(ctx, SC_ERR_GEOMETRY, "internal: mirror angle has a different trajectory count");
    const size_t rowb = (size_t)ne * 2 * ctx->rsz();
    std::vector<char> own((size_t)(a1 - a0) * rowb), mir((size_t)(m1 - m0) * rowb);
    CU(cudaStreamSynchronize(ctx->stream));
    CU(cudaMemcpy(own.data(), ctx->d_store[ctx->cur].p + (size_t)a0 * rowb, own.size(), cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(mir.data(), ctx->d_store[ctx->cur].p + (size_t)m0 * rowb, mir.size(), cudaMemcpyDeviceToHost));
    auto at = [&](const std::vector<char>& b, size_t row, int n, double& re, double& im) {
        if (ctx->f32) { const float* v = (const float*)(b.data() + row * rowb) + 2 * n; re = v[0]; im = v[1]; }
        else { const double* v = (const double*)(b.data() + row * rowb) + 2 * n; re = v[0]; im = v[1]; }
    };
    // mirror of directed trajectory d: h_dB for the first half of the angles, its inverse for the second half
    std::vector<int> mirror(a1 - a0);
    if (k < H) for (int d = a0; d < a1; ++d) mirror[d - a0] = ctx->h_dB[d];
    else for (int g = m0; g < m1; ++g) mirror[ctx->h_dB[g] - a0] = g;
    double* G = (double*)gamma_end; double* GT = (double*)gamma_tilde_end;
    for (int d = a0; d < a1; ++d)
        for (int n = 0; n < ne; ++n) {
            const size_t o = 2 * ((size_t)(d - a0) * ne + n);
            at(own, d - a0, n, G[o], G[o + 1]);
            double re, im; at(mir, mirror[d - a0] - m0, ctx->mats.partner[n], re, im);
            GT[o] = re; GT[o + 1] = -im;                        // Eq. 13 (:95): gamma-tilde_k(eps) = conj gamma_{k+N/2}(-conj eps)
        }
    return SC_OK;
}

sc_status sc_debug_math(sc_ctx* ctx, int n, double* max_rel_err) {
    if (!ctx || !max_rel_err) return SC_ERR_ARG;
    ON_DEVICE(ctx);
    DevBuf<double> d; CU(d.alloc(6)); CU(cudaMemsetAsync(d.p, 0, 6 * sizeof(double), ctx->stream));
    ++sck::g_launches, sck::math_test_kernel<<<64, 128, 0, ctx->stream>>>(n, d.p);
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(max_rel_err, d.p, 6 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return SC_OK;
}

sc_status sc_debug_last_march_ms(sc_ctx* ctx, float* ms) {
    if (!ctx || !ms) return SC_ERR_ARG;
    ON_DEVICE(ctx);
    if (ctx->mev_n == 0) return fail(ctx, SC_ERR_STATE, "no march kernel has been launched");
    cudaEvent_t* ev = ctx->mev[(ctx->mev_n - 1) % sc_ctx::MEV];
    CU(cudaEventSynchronize(ev[1]));
    CU(cudaEventElapsedTime(ms, ev[0], ev[1]));
    return SC_OK;
}

sc_status sc_debug_march_time(sc_ctx* ctx, float* total_ms, int* n_launches) {
    if (!ctx) return SC_ERR_ARG;
    ON_DEVICE(ctx);
    const int n = std::min(ctx->mev_n, (int)sc_ctx::MEV);
    float tot = 0.f;
    for (int i = 0; i < n; ++i) {
        cudaEvent_t* ev = ctx->mev[(ctx->mev_n - 1 - i) % sc_ctx::MEV];
        CU(cudaEventSynchronize(ev[1]));
        float ms = 0.f; CU(cudaEventElapsedTime(&ms, ev[0], ev[1]));
        tot += ms;
    }
    if (total_ms) *total_ms = tot;
    if (n_launches) *n_launches = n;
    ctx->mev_n = 0;
    return SC_OK;
}

sc_status sc_debug_march_units(sc_ctx* ctx, long long* units_total, long long* units_stored_T, long long* units_pole_table) {
    if (!ctx) return SC_ERR_ARG;
    ON_DEVICE(ctx);
    CU(cudaStreamSynchronize(ctx->stream));
    unsigned long long ns[2] = {0, 0}; CU(cudaMemcpy(ns, ctx->d_nstored.p, sizeof(ns), cudaMemcpyDeviceToHost));
    CU(cudaMemset(ctx->d_nstored.p, 0, sizeof(ns)));
    if (units_stored_T) *units_stored_T = (long long)ns[0];
    if (units_pole_table) *units_pole_table = (long long)ns[1];
    if (units_total) *units_total = ctx->march_units;
    ctx->march_units = 0;
    return SC_OK;
}

sc_status sc_debug_last_march_variant(sc_ctx* ctx, char* name, int len) {
    if (!ctx || !name || len < 1) return SC_ERR_ARG;
    if (ctx->last_variant.empty()) return fail(ctx, SC_ERR_STATE, "no march kernel has been launched");
    std::snprintf(name, (size_t)len, "%s", ctx->last_variant.c_str());
    return SC_OK;
}

sc_status sc_debug_launch_count(sc_ctx* ctx, long long* n_kernels) {
    if (!ctx) return SC_ERR_ARG;
    if (n_kernels) *n_kernels = sck::g_launches;
    sck::g_launches = 0;
    return SC_OK;
}

sc_status sc_debug_fp64_peak(sc_ctx* ctx, double* dfma_per_s, double* sm_clock_mhz) {
    if (!ctx || !dfma_per_s) return SC_ERR_ARG;
    ON_DEVICE(ctx);
    DevBuf<double> d; CU(d.alloc(1));
    const int iters = 20000, blocks = ctx->n_sm * 4, threads = 256;
    ++sck::g_launches, sck::fp64_peak_kernel<<<blocks, threads, 0, ctx->stream>>>(iters / 10, d.p);    // warm-up
    double best = 0;
    for (int rep = 0; rep < 3; ++rep) {
        CU(cudaEventRecord(ctx->ev0, ctx->stream));
        ++sck::g_launches, sck::fp64_peak_kernel<<<blocks, threads, 0, ctx->stream>>>(iters, d.p);
        CU(cudaEventRecord(ctx->ev1, ctx->stream));
        CU(cudaEventSynchronize(ctx->ev1));
        float ms = 0; CU(cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1));
        best = std::max(best, (double)blocks * threads * (double)iters * 64.0 / (ms * 1e-3));
    }
    *dfma_per_s = best;
    if (sm_clock_mhz) { int khz = 0; cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, ctx->opt.device); *sm_clock_mhz = khz / 1000.0; }
    return SC_OK;
}

sc_status sc_debug_fp64_peak_sustained(sc_ctx* ctx, double seconds, double* dfma_per_s) {
    if (!ctx || !dfma_per_s || !(seconds > 0) || seconds > 30) return fail(ctx, SC_ERR_ARG, "bad argument");
    ON_DEVICE(ctx);
    DevBuf<double> d; CU(d.alloc(1));
    const int iters = 20000, blocks = ctx->n_sm * 4, threads = 256;
    // back-to-back launches for `seconds`: the rate the part holds once it sits at its power limit
    ++sck::g_launches, sck::fp64_peak_kernel<<<blocks, threads, 0, ctx->stream>>>(iters, d.p);
    CU(cudaEventRecord(ctx->ev0, ctx->stream));
    ++sck::g_launches, sck::fp64_peak_kernel<<<blocks, threads, 0, ctx->stream>>>(iters, d.p);
    CU(cudaEventRecord(ctx->ev1, ctx->stream));
    CU(cudaEventSynchronize(ctx->ev1));
    float one = 0; CU(cudaEventElapsedTime(&one, ctx->ev0, ctx->ev1));
    const int n = std::max(4, (int)(seconds * 1e3 / std::max(one, 1e-3f)));
    for (int i = 0; i < n / 2; ++i) ++sck::g_launches, sck::fp64_peak_kernel<<<blocks, threads, 0, ctx->stream>>>(iters, d.p);   // reach the steady clock
    CU(cudaEventRecord(ctx->ev0, ctx->stream));
    for (int i = 0; i < n - n / 2; ++i) ++sck::g_launches, sck::fp64_peak_kernel<<<blocks, threads, 0, ctx->stream>>>(iters, d.p);
    CU(cudaEventRecord(ctx->ev1, ctx->stream));
    CU(cudaEventSynchronize(ctx->ev1));
    float ms = 0; CU(cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1));
    *dfma_per_s = (double)(n - n / 2) * blocks * threads * (double)iters * 64.0 / (ms * 1e-3);
    return SC_OK;
}

sc_status sc_debug_pipe_peak(sc_ctx* ctx, int pipe, double seconds, double* ops_per_s) {
    if (!ctx || !ops_per_s || pipe < 1 || (pipe > 3 && pipe < 10) || pipe > 15 || !(seconds > 0) || seconds > 30) return fail(ctx, SC_ERR_ARG, "bad argument");
    ON_DEVICE(ctx);
    DevBuf<float> d; CU(d.alloc(2));
    const int blocks = ctx->n_sm * 4, threads = 256;
    const int iters = pipe == 1 ? 20000 : (pipe >= 10 ? 4000 : 2000);
    const double per_thread = (double)iters * 64.0;       // 8 chains x 8 per loop body, in both kernels
    auto launch = [&]() {
        ++sck::g_launches;
        if (pipe == 1) sck::fp32_peak_kernel<<<blocks, threads, 0, ctx->stream>>>(iters, d.p);
        else if (pipe == 2) sck::mufu_peak_kernel<false><<<blocks, threads, 0, ctx->stream>>>(iters, d.p);
        else if (pipe == 3) sck::mufu_peak_kernel<true><<<blocks, threads, 0, ctx->stream>>>(iters, d.p);
        else if (pipe == 10) sck::fp64_mix_kernel<0, 0><<<blocks, threads, 0, ctx->stream>>>(iters, (double*)d.p);
        else if (pipe == 11) sck::fp64_mix_kernel<4, 0><<<blocks, threads, 0, ctx->stream>>>(iters, (double*)d.p);
        else if (pipe == 12) sck::fp64_mix_kernel<8, 0><<<blocks, threads, 0, ctx->stream>>>(iters, (double*)d.p);
        else if (pipe == 13) sck::fp64_mix_kernel<0, 1><<<blocks, threads, 0, ctx->stream>>>(iters, (double*)d.p);
        else if (pipe == 14) sck::fp64_mix_kernel<3, 1><<<blocks, threads, 0, ctx->stream>>>(iters, (double*)d.p);
        else sck::fp64_operand_kernel<<<blocks, threads, 0, ctx->stream>>>(iters, (double*)d.p);
    };
    launch();
    CU(cudaEventRecord(ctx->ev0, ctx->stream));
    launch();
    CU(cudaEventRecord(ctx->ev1, ctx->stream));
    CU(cudaEventSynchronize(ctx->ev1));
    float one = 0; CU(cudaEventElapsedTime(&one, ctx->ev0, ctx->ev1));
    const int n = std::max(4, (int)(seconds * 1e3 / std::max(one, 1e-3f)));
    for (int i = 0; i < n / 2; ++i) launch();                                    // reach the steady clock
    CU(cudaEventRecord(ctx->ev0, ctx->stream));
    for (int i = 0; i < n - n / 2; ++i) launch();
    CU(cudaEventRecord(ctx->ev1, ctx->stream));
    CU(cudaEventSynchronize(ctx->ev1));
    CU(cudaGetLastError());
    float ms = 0; CU(cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1));
    *ops_per_s = (double)(n - n / 2) * blocks * threads * per_thread / (ms * 1e-3);
    return SC_OK;
}

}  // extern "C"
