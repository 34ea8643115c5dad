/* sc_riccati.h — C ABI of the B200-native Riccati-parametrised Eilenberger sweep.
 *
 * What it computes (all citations are PAPER.md:<line> = arXiv 2205.15000 "SuperConga"):
 *   for every Fermi angle phi_k (:189) and every energy (Matsubara i*eps_n, or eps + i*delta, :98) the
 *   coherence functions gamma, gamma-tilde are marched along straight trajectories R(s) = R_min + s v_F
 *   (Eq. 23 :153) through a 2-D grain with specular walls (:155, :161), solving the Riccati equations
 *   (Eq. 25-26 :169-172) with the closed-form step for piecewise-constant Delta, A (the "stepping
 *   method", :982).  From g = (1 - gamma gamma~)/(1 + gamma gamma~) (Eq. 24 :165) it accumulates the
 *   gap-equation right-hand side (Eq. 22 :144), the current density (Eq. 8 :69), the Eilenberger
 *   free-energy term I(R) (Eq. 19 :128) and the LDOS (Eq. 14 :100); the induced vector potential is
 *   Eq. D1 (:1009) and the self-consistency update is Algorithm 1 (:203-205) with the Picard or
 *   Barzilai-Borwein accelerator (App. E :1066-1127).  Readings of silent passages: DESIGN.md §3.
 *
 * Units (:104-112, Table II :1204-1230): energies in 2 pi kB Tc, lengths in xi0 (v_F = 1), t = T/Tc,
 * A in Phi0/(pi xi0), j in j0, free-energy density in (2 pi kB Tc)^2 N_F.
 *
 * Conventions
 *   Pointers marked "dev" are CUDA device pointers on opts.device, "host" are host pointers.  The
 *   caller owns every field buffer; the context owns tables, boundary stores and scratch.  Nothing
 *   returned has to be freed except the context (sc_destroy).  Every call enqueues on opts.cuda_stream
 *   and returns without a host synchronisation, except sc_create, sc_ldos's table upload, the
 *   sc_debug_* taps, and any call given a non-NULL stats pointer (one small D2H copy).
 *   Grid layout: row-major [j][i], x_i = (i - (nx-1)/2) h, y_j = (j - (ny-1)/2) h.  Complex fields are
 *   interleaved (re, im) fp64.  Outputs are exactly 0 outside the mask.
 *   Errors: a status code is returned (never an exception or abort across the ABI); the message is
 *   available from sc_last_error().  All kernels are sm_100a; there is no CPU fallback: without a CUDA
 *   device sc_create returns SC_ERR_CUDA.
 *   One context per host thread.
 */
#ifndef SC_RICCATI_H
#define SC_RICCATI_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sc_ctx sc_ctx;

typedef enum { SC_OK = 0, SC_ERR_ARG = 1, SC_ERR_GEOMETRY = 2, SC_ERR_STATE = 3,
               SC_ERR_CUDA = 4, SC_ERR_NOMEM = 5, SC_ERR_NUMERIC = 6 } sc_status;
/* SC_ERR_NUMERIC: a reduced output field (sc_riccati_sweep) or a residual (sc_iterate) is not finite.  It is only
 * detected by calls given a stats pointer — the calls that synchronise anyway; the outputs are still written. */

/* Order-parameter basis functions eta(phi) on a circular Fermi surface, Table III (:1238-1246):
 * s: 1;  d_{x2-y2}: sqrt2 cos 2phi;  d_xy: sqrt2 sin 2phi;  g: sqrt2 sin 4phi. */
typedef enum { SC_SYM_S = 0, SC_SYM_DX2Y2 = 1, SC_SYM_DXY = 2, SC_SYM_G = 3 } sc_symmetry;

typedef struct { int nx, ny; double h; } sc_grid;

/* One CSG component of the grain (:411-448, :928-958), applied in list order: kind 0 = disc
 * (cx, cy, r), kind 1 = convex polygon with nvert vertices in counter-clockwise order (host pointers,
 * copied by sc_create).  add = 1 adds the area, add = 0 removes it. */
typedef struct { int kind; int add; double cx, cy, r; int nvert; const double *vx, *vy; } sc_shape;

typedef struct {
    int n_angles;        /* N_phi, even; phi_k = 2 pi k / N_phi (:189) */
    int n_matsubara;     /* N_eps; eps_n = t (n + 1/2), n = 0..N_eps-1 (:98) */
    int precision;       /* 64 (default) or 32: arithmetic of the march; ABI buffers stay fp64 */
    int stepper;         /* 0 = closed-form step (:982); 1 = implicit mid-point C4-C9 (:984-1001) */
    int quadrature;      /* 0 = paper's rule: Boole / Simpson 3/8 / Simpson 1/3 / trapezoid by N_phi mod 4,3,2 (:189); 1 = trapezoid */
    int charge_sign;     /* sigma_e = -1 for electrons (:43, :890) */
    int bc_mode;         /* 0 = specular (:155); 1 = bulk: every start value is the local homogeneous solution */
    double crystal_rotation; /* rotation of the crystal axes in full turns (:890) */
    int device;          /* CUDA device ordinal */
    void* cuda_stream;   /* cudaStream_t; NULL = default stream */
    int residual_norm;   /* p of the residual norms of Eq. 27 (:201; "norm" in :960): 2 (0 = default), 1, or -1 = maximum norm.
                          * One element is one complex Delta_G(R), one vector A(R) or j(R), or one real I(R). */
} sc_opts;

typedef struct {
    double res_delta, res_j, res_A, res_fe;   /* Eq. 27 (:201) in the norm opts.residual_norm; filled by sc_iterate */
    double min_one_minus_abs_gamma;           /* min over nodes of 1 - max(|gamma|,|gamma~|) (invariant |gamma| < 1) */
    long long n_updates;                      /* logical trajectory-step updates of the sweep: 2 * N_phi * N_eps * sum_t pieces */
    long long n_updates_executed;             /* steps actually marched (Eq. 13 symmetry halves them) */
    float ms;                                 /* device time of the call (CUDA events on the stream) */
    int n_bad;                                /* interpolation points with no valid neighbour (must be 0) */
} sc_sweep_stats;

/* Build the trajectory tables for a grain (:153, :189, Fig. 2 :195).  mask: host, nx*ny bytes, 1 iff the
 * grid point is strictly inside the CSG of `shapes` (checked: SC_ERR_GEOMETRY on disagreement).
 * T_over_Tc = t.  kappa <= 0 means infinite penetration depth (A_ind = 0, :890). */
sc_status sc_create(const sc_grid* grid, const unsigned char* mask, const sc_shape* shapes, int nshapes,
                    double T_over_Tc, double kappa, sc_symmetry symmetry, const sc_opts* opts, sc_ctx** out);
sc_status sc_destroy(sc_ctx* ctx);

/* Set Delta(R) (dev, complex fp64 [ny][nx]; [n][ny][nx] after sc_set_components) and the TOTAL vector potential A = A_ext + A_ind (dev fp64
 * [ny][nx] each; NULL = 0).  Copies into context-owned buffers; does not touch the boundary stores. */
sc_status sc_set_fields(sc_ctx* ctx, const void* delta, const double* Ax, const double* Ay);

/* Several order-parameter components (Eq. 1 :37, Listing 11 :909-926): Delta(p_F,R) = sum_G Delta_G(R) eta_G(p_F)
 * with basis functions symmetries[0..n-1] (Table III :1238) and critical temperatures T_c^G = tc_ratio[G] * T_c
 * (host arrays; T_c, the energy unit, is the largest: 0 < tc_ratio <= 1), 1 <= n <= 4.  Each component obeys its own gap
 * equation (Eq. 22 :144 with ln(T/T_c^G)).  Afterwards EVERY order-parameter buffer of the ABI (sc_set_fields' delta,
 * sc_riccati_sweep's delta_new, sc_iterate's delta_inout) is complex fp64 [n][ny][nx], and sc_iterate mixes
 * x = (Re D_0, Im D_0, ..., kappa^2 A_x, kappa^2 A_y) (E3 :1053; 2n + 2 CongAcc components).  Call it after sc_create
 * and before sc_set_fields: it invalidates the fields, the boundary stores and the driver state.  sc_create's single
 * symmetry is the n = 1 case.  SC_ERR_ARG if n, a symmetry or a ratio is out of range. */
sc_status sc_set_components(sc_ctx* ctx, int n, const sc_symmetry* symmetries, const double* tc_ratio);

/* Replace the Matsubara table by any energies z_n = z_re + i z_im (Im z > 0) with weights w_n (host, n values):
 * Ozaki poles (:207, reading R-A4), or ONE SHARD of the Matsubara energies when the sweep is split by energy across
 * GPUs.  The table must be closed under z -> -conj(z) with equal weights for the two partners (Eq. 13 :95:
 * the sums of angle k + N/2 are taken from the partner energies of angle k; energies on the imaginary axis are their own
 * partners).  denominator_sum = sum over the WHOLE job's table of w_n t / Im z_n, the second term of the denominator of
 * Eq. 22 (:144); NaN = compute it from this table.  Re-sizes and invalidates the boundary stores. */
sc_status sc_set_energies(sc_ctx* ctx, const double* z_re, const double* z_im, const double* w, int n,
                          double denominator_sum);

/* Energy-sharded sweeps: with a hook set, sc_riccati_sweep (and sc_iterate) write the five un-finalised
 * accumulators sum_k W_k {Re, Im conj(eta_k) SF_k, v_kx SG_k, v_ky SG_k, SI_k} of this context's energies into
 * acc (dev fp64 [5][ny][nx], caller-owned; with n order-parameter components [2n+3][ny][nx]: Re, Im per component,
 * then the current and I terms), call fn(user) on the host — which must enqueue, on the context's
 * stream, the sum of acc over all shards (one all-reduce) — and then apply Eq. 22 / Eq. 8 / Eq. 19 to the summed
 * accumulators.  fn = NULL, acc = NULL removes the hook. */
typedef void (*sc_allreduce_fn)(void* user);
sc_status sc_set_allreduce_hook(sc_ctx* ctx, double* acc, sc_allreduce_fn fn, void* user);

/* Boundary stores := local homogeneous solution at each trajectory end (Algorithm 1 "Initialize
 * gamma_dD", :205; reading R8).  Needs fields.  Called implicitly by the first sweep. */
sc_status sc_reset_boundary(sc_ctx* ctx);

/* One Jacobi sweep at the Matsubara energies (:187 "update of the boundary values can be done in
 * parallel"): reads boundary store A, writes B, swaps.  Outputs (dev, any may be NULL):
 *   delta_new  complex [ny][nx]   Eq. 22 (:144), n >= 0 only and doubled
 *   jx, jy     fp64   [ny][nx]    Eq. 8 (:69) in units of j0
 *   fe_I       fp64   [ny][nx]    I(R) of Eq. 19 (:128)
 * Repeated calls with unchanged fields are the paper's burn-in (:962). */
sc_status sc_riccati_sweep(sc_ctx* ctx, void* delta_new, double* jx, double* jy, double* fe_I,
                           sc_sweep_stats* stats);

/* LDOS N(eps_m, R)/N_F = <Re g_n> (Eq. 14 :100) at eps_m + i*broadening for the current fields, after
 * n_boundary_iters Jacobi sweeps from freshly reset stores (:366 burn-in).  energies: host, n_e values.
 * ldos: dev fp64 [n_e][ny][nx].  The Matsubara boundary stores are not touched. */
sc_status sc_ldos(sc_ctx* ctx, const double* energies, int n_e, double broadening, int n_boundary_iters,
                  double* ldos, sc_sweep_stats* stats);

/* A_ind = -(1/kappa^2) sum G_{|m'-m|,|n'-n|} (j - <j>_mask) (Eq. D1-D6 :1009-1021, :1040) on the whole
 * grid (dev in, dev out); fe_magnetic (host, may be NULL) = (h^2/2) sum_mask j.A_ind (reading R18). */
sc_status sc_update_vector_potential(sc_ctx* ctx, const double* jx, const double* jy,
                                     double* Aind_x, double* Aind_y, double* fe_magnetic);

/* Choose how sc_update_vector_potential / sc_iterate evaluate D1: eps = 0 (default) the exact cross-correlation with the
 * full G table (zero-padded FFT); eps > 0 the paper's truncated eigen-decomposition G = sum_k lambda_k V^(k) V^(k)T
 * (D7 :1027) keeping the N* eigenpairs of largest |lambda| with sqrt(1 - sum_{n<N*} lambda_n^2 / sum_n lambda_n^2) < eps
 * (D9 :1036, the config key vector_potential_error) and N* pairs of separable 1-D cross-correlations (D8 :1031).
 * n_kept (host, may be NULL): receives N* (0 for eps = 0); asking for it runs the eigen-decomposition now (synchronises).
 * SC_ERR_ARG unless 0 <= eps < 1. */
sc_status sc_set_vector_potential_error(sc_ctx* ctx, double eps, int* n_kept);

/* Set the external vector potential used by sc_iterate (dev fp64 [ny][nx]; NULL = 0). */
sc_status sc_set_external_field(sc_ctx* ctx, const double* Aext_x, const double* Aext_y);

/* One self-consistency iteration (Algorithm 1 :203-205): fields := (delta, A_ext + A_ind); sweep; A-solve;
 * x = (Re D, Im D, kappa^2 A_ind) (E3 :1053), d = g(x) - x (E4), then by accelerator
 *   0 Picard           x += step d                                                        (E5 :1070)
 *   1 Barzilai-Borwein x += alpha d, alpha_0 = step, alternating BB1/BB2 scaling, clipped   (E8-E11 :1107-1115)
 *   2 Polyak           v <- (1 - drag) v + step d, x += v, v_0 = 0                          (E6-E7 :1087-1089)
 *   3 CongAcc          per component of x: cosine-similarity-adapted step and moving average (E12-E17 :1134-1151)
 * Changing the accelerator between calls restarts it.  burnin != 0 keeps delta, A_ind fixed (:962).
 * delta_inout / Aind_*_inout: dev, updated in place. */
sc_status sc_iterate(sc_ctx* ctx, int accelerator, double step, int burnin, void* delta_inout,
                     double* Aind_x_inout, double* Aind_y_inout, sc_sweep_stats* stats);

/* Parameters of the accelerators (PAPER.md Listings 14-16 :1093, :1121, :1157); an argument <= 0 keeps its
 * current value.  Defaults: drag 0.5 (Polyak beta in (0,1]); step_factor k = 1.234 and cos_similarity_min
 * s_min = 0.7 (CongAcc E13-E14); step sizes of Barzilai-Borwein and CongAcc clipped to [step_min, step_max] =
 * [1e-3, 100].  SC_ERR_ARG if a value is out of range. */
sc_status sc_set_accelerator_params(sc_ctx* ctx, double drag, double step_factor, double cos_similarity_min,
                                    double step_min, double step_max);

/* The residual of Eq. 27 (:201), ||x_new - x_old||_p / ||x_old||_p over n complex fp64 elements (the res_delta of
 * sc_iterate for x = Delta), for callers that may not allocate: code under CUDA graph capture, tight serving loops.
 * It needs no context and calls no cudaMalloc / cudaFree or allocating library routine: the partial sums of its
 * reduction live in a static device array of the library (64.25 KiB, held by every GPU that loads the library until
 * exit), which bounds the size: n <= SC_RESIDUAL_STATIC_MAX_ELEMENTS, beyond that SC_ERR_ARG.
 *   x_new, x_old  dev, complex fp64 [n] (caller-owned, read only)
 *   norm_p        2 (0 = default), 1, or -1 = maximum norm, as opts.residual_norm
 *   out           dev fp64 [3] (caller-owned): ||x_new - x_old||_p, ||x_old||_p, their ratio (the numerator if x_old = 0)
 *   device        CUDA device ordinal, made current; < 0 = the calling thread's current device
 *   cuda_stream   cudaStream_t the work (one 8-byte memset + one kernel) is enqueued on; no host synchronisation
 *   err, err_len  host buffer for the message of a non-zero status (may be NULL)
 * The first call on a device looks the array's address up (cudaGetSymbolAddress): make it outside graph capture.
 * All calls on a device share the array: calls that overlap on the GPU (two streams, two host threads) race. */
#define SC_RESIDUAL_STATIC_MAX_ELEMENTS 8388608LL
sc_status sc_residual_norm_static(const void* x_new, const void* x_old, long long n, int norm_p, double* out,
                                  int device, void* cuda_stream, char* err, int err_len);

/* ---- parity / debug taps (synchronise) -------------------------------------------------------- */
/* Geometry: lattice size N_rot, number of trajectories of angle k (all N_phi angles are addressable). */
sc_status sc_debug_geometry(sc_ctx* ctx, int* n_rot, int* n_traj_total, long long* n_pieces_total);
/* Tables of angle k (host out, caller-sized from sc_debug_geometry): per trajectory
 *   it[6] = {t, jf, jl, elem_in, elem_out, 0}, dt[2] = {u_in, u_out}, gidx[4] (entry gather: global
 *   directed-trajectory ids (angle-major, line order), -1 unused), gw[4] weights.  Returns count in *n. */
sc_status sc_debug_tables(sc_ctx* ctx, int k, int* n, int* it, double* dt, int* gidx, double* gw);
/* gamma (and gamma-tilde) at the nodes of trajectory `local` of angle k (k < N_phi/2) for Matsubara index
 * n_energy, as marched by the LAST sweep's inputs (re-marches that one trajectory). host out, complex. */
sc_status sc_debug_trajectory(sc_ctx* ctx, int k, int local, int n_energy, int* n_nodes, void* gamma, void* gamma_tilde);
/* Per-angle energy-summed node sums of the last sweep for angle k on the rotated lattice [t][j] (host out,
 * N_rot*N_rot each; SF complex): SF = sum gamma/(1+P), SG = sum Im g, SI (Eq. 19 numerator). */
sc_status sc_debug_partial(sc_ctx* ctx, int k, void* SF, double* SG, double* SI);
/* The boundary values the LAST sweep's march launch wrote (the production launch itself, not a re-march): for every
 * trajectory of angle k (all N_phi angles are addressable, in the order of sc_debug_tables) and every energy of the
 * table, gamma at the exit point and gamma-tilde at the entry point (host out, complex fp64 [n_traj(k)][n_energies] each).
 * The library stores gamma_end for all directed trajectories only; gamma-tilde_end of (k, t) is returned as the conjugate
 * of gamma_end of the mirror trajectory on angle k + N/2 at the partner energy (Eq. 13 :95). */
sc_status sc_debug_stores(sc_ctx* ctx, int k, void* gamma_end, void* gamma_tilde_end);
/* Device-math self test: max relative error of the fp64 reciprocal / rsqrt / exp / sincos building blocks
 * against the CUDA math library on n random arguments (host out, 6 values). */
sc_status sc_debug_math(sc_ctx* ctx, int n, double* max_rel_err);
/* Register-resident DFMA microbenchmark: measured fp64 FMA instructions per second of the device (the
 * roofline denominator of the march kernel). */
sc_status sc_debug_fp64_peak(sc_ctx* ctx, double* dfma_per_s, double* sm_clock_mhz);
/* The same microbenchmark launched back to back for `seconds` (<= 30), rate of the second half: what the FP64 pipe
 * sustains once the part sits at its power limit (the march runs for seconds at a time). */
sc_status sc_debug_fp64_peak_sustained(sc_ctx* ctx, double seconds, double* dfma_per_s);
/* The same kind of register-resident loop for the other pipes the march uses, held for `seconds` (<= 30): pipe 1 = fp32
 * FMA (FFMA; roofline denominator of opts.precision = 32), 2 = MUFU.RCP (fp32 reciprocal seed), 3 = MUFU.RCP64H (fp64
 * reciprocal seed) — the special-function issue rate north_star asks about.  ops_per_s counts thread-level
 * instructions per second over the whole device.  Pipes 10-14 run the DFMA loop with other instructions mixed in and
 * return DFMA per second: 10 = DFMA only, 11 = + 0.5 integer instruction per DFMA, 12 = + 1 integer, 13 = + 0.125
 * shared-memory load (and its DADD), 14 = + 0.375 integer + 0.125 shared-memory load — what the non-FP64 instructions of
 * the march cost next to half-rate DFMA; 15 = DFMA only, but with three different, changing register operands per instruction
 * (DESIGN.md §6). */
sc_status sc_debug_pipe_peak(sc_ctx* ctx, int pipe, double seconds, double* ops_per_s);

/* Device time of the most recent march kernel launch (CUDA events recorded on the stream around that launch
 * alone); synchronises.  Used by bench.py for the roofline of the dominant kernel. */
sc_status sc_debug_last_march_ms(sc_ctx* ctx, float* ms);
/* Sum of the device times of the march launches since the previous call of this function (at most the last 64),
 * each bracketed by its own CUDA events on the stream, and their count; synchronises, then resets the count.
 * bench.py calls it around the timed region: the roofline of the dominant kernel comes from the launches that
 * the timed steps themselves made.  Either output may be NULL (reset only). */
sc_status sc_debug_march_time(sc_ctx* ctx, float* total_ms, int* n_launches);
/* (piece, energy, angle pair) units marched by the full-work-list march launches since the previous call of this
 * function, and how many of them belonged to rounds that (i) spilled the step coefficient T between the passes
 * (some piece outside the radii of the per-energy tables: 64 B of scratch traffic per unit), (ii) re-evaluated it in
 * pass 2 from the pole-subtracted table; the rest re-evaluated it from the pole-free table (both 32 B per unit;
 * DESIGN.md 4-6); synchronises, then resets.  Any output may be NULL. */
sc_status sc_debug_march_units(sc_ctx* ctx, long long* units_total, long long* units_stored_T, long long* units_pole_table);

/* Template arguments of the most recent march launch, e.g. "march_kernel<0,false,0,double,1,true>" =
 * <MODE 0 sums / 1 LDOS / 2 boundary only, STATS, STEPPER, working precision, T-table layout 1 imaginary axis / 2 general,
 * unit weights compiled out> (name: host out, len bytes).  The parity tests assert with it that the instantiation
 * bench.py times is the one they compared with the oracle.  SC_ERR_STATE before the first sweep. */
sc_status sc_debug_last_march_variant(sc_ctx* ctx, char* name, int len);
/* Kernels of this library launched by the calling host thread since the previous call of this function (counted at the
 * launch sites; cuFFT / cuBLAS / cuSOLVER launches, memsets and copies are not included); resets.  n_kernels may be NULL. */
sc_status sc_debug_launch_count(sc_ctx* ctx, long long* n_kernels);

const char* sc_last_error(const sc_ctx* ctx);
const char* sc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SC_RICCATI_H */
