// sc_oracle.cpp — CPU ORACLE for the Riccati-parametrised Eilenberger sweep.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load it.  It shares no code with the CUDA path under
// paper_2205_15000_b200/ (no headers, helpers, tables or constants) and never imports it.
//
// It is a plain, slow, step-by-step implementation of what PAPER.md (arXiv 2205.15000, "SuperConga")
// states, in the paper's order and notation, fp64 (std::complex<double>), straightforward loops
//     angles -> trajectories -> energies -> steps,
// marching BOTH gamma and gamma-tilde for ALL angles and using NO symmetry shortcut.  Where the paper
// is silent the reading of DESIGN.md §3 (R1..R22, taken from SURVEY.md §8c) is followed and cited.
//
// Units (Table II :1204-1230): energies in 2 pi kB Tc, lengths in xi0 (v_F = 1),
// t = T/Tc, Matsubara eps_n = t (n + 1/2), A in A0 = Phi0/(pi xi0) so that (e/c) v_F.A -> sigma_e v.A.
//
// Pins (tests/test_oracle_pins*.py, listed with the sabotages they catch in DESIGN.md §7): closed-form step vs adaptive
// ODE solve, bulk fixed point, uniform gap closed form, BCS gap 1.764 / 2.14, Doppler-shift current, bulk free energy
// Eq. 38, ABS kink, Eq. 13 symmetry, global-phase covariance, G_{m,n} vs quadrature of D2, brute-force ray tracing on and
// off the lattice (ODE reference), gather weights against prescribed linear stores and analytic normals (square, disc,
// annulus), rotate-in / rotate-back against a library bilinear interpolant, charge conservation at self-consistency,
// rotation covariance P11, and the paper's annulus benchmarks Eq. 43 and Eq. 48-53.
// Parity unpinned (fixed only by DESIGN.md readings): the interpolation FALLBACKS at corners / grazing incidence — the
// nearest-mask-point search of R5, the "no valid candidate" branch of R6/R7 and the renormalisation of the gather
// weights when a candidate ends on another wall.
//
// Build: g++ -O2 -fopenmp -shared -fPIC -std=c++17 sc_oracle.cpp -o libsc_oracle.so

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

typedef std::complex<double> cd;
static const cd I_(0.0, 1.0);
static const double PI = 3.14159265358979323846;

// ---------------------------------------------------------------------------------------------------
// Geometry: discs and convex CCW polygons, added / removed in list order.
// ---------------------------------------------------------------------------------------------------
struct Shape {
    int kind;  // 0 disc, 1 convex polygon
    int add;
    double cx, cy, r;
    std::vector<double> vx, vy;
};
struct End {        // one crossing of a line with the grain boundary
    double u;       // trajectory coordinate of the crossing
    int elem;       // wall element id = shape index * 65536 + edge index (disc: edge 0)
    double nx, ny;  // outward unit normal of the GRAIN at the crossing
};
struct Interval { End in, out; };

struct Gather {     // R6/R7: up to 4 (trajectory, weight) pairs; n == 0 -> homogeneous fallback
    int n;
    int idx[4];
    double w[4];
    double dirx, diry;   // mirrored direction v_in / v_out (used by the fallback only)
};
struct Traj {
    int k, t;            // angle index, lattice line index
    double u_in, u_out;  // exact boundary crossings ("exact location ... of boundaries")
    int jf, jl;          // first / last lattice node strictly inside (R3)
    End e_in, e_out;
    Gather g_in, g_out;  // start value of gamma at u_in, of gamma-tilde at u_out
};

struct Ctx {
    int nx, ny; double h;
    std::vector<Shape> shapes;
    std::vector<unsigned char> mask;
    int nphi, sym; double rot; int quad, sigma, bc_mode, stepper; double t;
    int nrot; double c;
    std::vector<double> vx, vy, W;   // v_k = (vx,vy); n_k = (-vy, vx); quadrature weight
    std::vector<double> eta;         // eta_k (real for all Table III functions)
    // several order-parameter components (Eq. 1 :37): Delta(p_F,R) = sum_G Delta_G(R) eta_G(p_F); syms.size() >= 1,
    // syms[0] == sym.  The fields handed to the sweep are then [ncomp][ny][nx].
    std::vector<int> syms;
    std::vector<std::vector<Traj>> traj;               // [k][local]
    std::vector<int> off;                              // global trajectory id offset per angle
    std::vector<std::vector<std::vector<int>>> line;   // [k][t] -> local trajectory indices
    int ntraj;
    int n_gather_fallback;
    std::string err;
};

// eta(phi) for a circular Fermi surface, Table III (:1238-1246); crystal axes rotated by
// `rot` full turns.
static double basis(int sym, double phi, double rot) {
    double p = phi - 2.0 * PI * rot;
    switch (sym) {
        case 0: return 1.0;
        case 1: return std::sqrt(2.0) * std::cos(2.0 * p);
        case 2: return std::sqrt(2.0) * std::sin(2.0 * p);
        case 3: return std::sqrt(2.0) * std::sin(4.0 * p);
    }
    return 0.0;
}

// Fermi-surface quadrature: Boole / Simpson 3/8 / Simpson 1/3 / trapezoid by N mod 4,3,2
// on the periodic interval, normalised so that sum_k W_k = 1 (Eq. 5 :55).  quad = 1 forces trapezoid.
static std::vector<double> quadrature(int n, int quad) {
    std::vector<double> W(n);
    for (int k = 0; k < n; ++k) {
        if (quad == 1) W[k] = 1.0 / n;
        else if (n % 4 == 0) { static const double b[4] = {28, 64, 24, 64}; W[k] = b[k % 4] / (45.0 * n); }
        else if (n % 3 == 0) { static const double s[3] = {6, 9, 9}; W[k] = s[k % 3] / (8.0 * n); }
        else if (n % 2 == 0) { static const double s[2] = {2, 4}; W[k] = s[k % 2] / (3.0 * n); }
        else W[k] = 1.0 / n;
    }
    return W;
}

// Clip the line R(u) = u v + w n against one shape: at most one interval (convex shapes).
static bool clip_shape(const Shape& s, int sid, double vx, double vy, double w, Interval& out) {
    double nx = -vy, ny = vx;
    if (s.kind == 0) {
        double uc = s.cx * vx + s.cy * vy;          // centre along the line
        double q = w - (s.cx * nx + s.cy * ny);     // perpendicular offset of the line from the centre
        double d2 = s.r * s.r - q * q;
        if (!(d2 > 0.0)) return false;
        double half = std::sqrt(d2);
        out.in.u = uc - half; out.out.u = uc + half;
        out.in.elem = out.out.elem = sid * 65536;
        double px = out.in.u * vx + w * nx - s.cx, py = out.in.u * vy + w * ny - s.cy;
        out.in.nx = px / s.r; out.in.ny = py / s.r;
        px = out.out.u * vx + w * nx - s.cx; py = out.out.u * vy + w * ny - s.cy;
        out.out.nx = px / s.r; out.out.ny = py / s.r;
        return true;
    }
    // convex polygon: half-plane clipping, edge e from V_e to V_{e+1}, outward normal (dy,-dx)/len
    int nv = (int)s.vx.size();
    double lo = -1e300, hi = 1e300; int elo = -1, ehi = -1;
    double lnx = 0, lny = 0, hnx = 0, hny = 0;
    for (int e = 0; e < nv; ++e) {
        double x0 = s.vx[e], y0 = s.vy[e], x1 = s.vx[(e + 1) % nv], y1 = s.vy[(e + 1) % nv];
        double dx = x1 - x0, dy = y1 - y0, len = std::sqrt(dx * dx + dy * dy);
        double ex = dy / len, ey = -dx / len;
        double den = ex * vx + ey * vy;
        double num = ex * (x0 - w * nx) + ey * (y0 - w * ny);   // inside: u*den < num
        if (std::fabs(den) <= 1e-12) { if (!(num > 0.0)) return false; continue; }   // parallel edge
        double ub = num / den;
        if (den > 0.0) { if (ub < hi) { hi = ub; ehi = e; hnx = ex; hny = ey; } }
        else           { if (ub > lo) { lo = ub; elo = e; lnx = ex; lny = ey; } }
    }
    if (elo < 0 || ehi < 0 || !(hi - lo > 0.0)) return false;
    out.in.u = lo; out.in.elem = sid * 65536 + elo; out.in.nx = lnx; out.in.ny = lny;
    out.out.u = hi; out.out.elem = sid * 65536 + ehi; out.out.nx = hnx; out.out.ny = hny;
    return true;
}

// CSG in list order: add = union, remove = subtract.
static std::vector<Interval> clip_line(const std::vector<Shape>& shapes, double vx, double vy, double w) {
    std::vector<Interval> S;
    for (size_t sid = 0; sid < shapes.size(); ++sid) {
        Interval I;
        if (!clip_shape(shapes[sid], (int)sid, vx, vy, w, I)) continue;
        std::vector<Interval> R;
        if (shapes[sid].add) {
            // union: merge I with every interval it overlaps
            for (auto& s : S) {
                if (s.out.u < I.in.u || s.in.u > I.out.u) { R.push_back(s); continue; }
                if (s.in.u < I.in.u) I.in = s.in;
                if (s.out.u > I.out.u) I.out = s.out;
            }
            R.push_back(I);
            std::sort(R.begin(), R.end(), [](const Interval& a, const Interval& b) { return a.in.u < b.in.u; });
        } else {
            // subtract: new ends lie on the removed shape; grain normal = minus the shape's normal
            for (auto& s : S) {
                if (s.out.u <= I.in.u || s.in.u >= I.out.u) { R.push_back(s); continue; }
                if (I.in.u > s.in.u) {
                    Interval a = s; a.out = I.in; a.out.nx = -I.in.nx; a.out.ny = -I.in.ny; R.push_back(a);
                }
                if (I.out.u < s.out.u) {
                    Interval b = s; b.in = I.out; b.in.nx = -I.out.nx; b.in.ny = -I.out.ny; R.push_back(b);
                }
            }
        }
        S.swap(R);
    }
    std::vector<Interval> keep;
    for (auto& s : S) if (s.out.u - s.in.u > 0.0) keep.push_back(s);
    return keep;
}

static bool inside_csg(const std::vector<Shape>& shapes, double x, double y) {
    bool in = false;
    for (auto& s : shapes) {
        bool strict, closed;
        if (s.kind == 0) {
            double d2 = (x - s.cx) * (x - s.cx) + (y - s.cy) * (y - s.cy);
            strict = d2 < s.r * s.r; closed = d2 <= s.r * s.r;
        } else {
            strict = true;
            int nv = (int)s.vx.size();
            for (int e = 0; e < nv; ++e) {
                double x0 = s.vx[e], y0 = s.vy[e], x1 = s.vx[(e + 1) % nv], y1 = s.vy[(e + 1) % nv];
                double dx = x1 - x0, dy = y1 - y0, len = std::sqrt(dx * dx + dy * dy);
                if (!((dy / len) * (x - x0) + (-dx / len) * (y - y0) < 0.0)) strict = false;
            }
            closed = strict;
        }
        if (s.add) in = in || strict; else if (closed) in = false;
    }
    return in;
}

static inline double lattice_u(const Ctx& C, int j) { return (j - C.c) * C.h; }

// R6 / R7: specular start value = interpolation, linear in angle x linear in the
// perpendicular offset, over the incoming trajectories that END (gamma) or BEGIN (gamma-tilde) on the
// same wall element ("gamma(s') = gamma(s)", :191-197).
static Gather build_gather(const Ctx& C, double Rx, double Ry, double nx, double ny, double vx, double vy,
                           int elem, bool want_exit) {
    Gather g; g.n = 0;
    double dot = vx * nx + vy * ny;
    double mx = vx - 2.0 * dot * nx, my = vy - 2.0 * dot * ny;   // mirrored direction
    g.dirx = mx; g.diry = my;
    double dphi = 2.0 * PI / C.nphi;
    double kap = std::atan2(my, mx) / dphi;
    kap = kap - C.nphi * std::floor(kap / C.nphi);
    int k1 = (int)std::floor(kap);
    double om = kap - k1;
    int ka[2]; double wa[2]; int na = 0;
    if (om < 1e-12) { ka[0] = k1 % C.nphi; wa[0] = 1.0; na = 1; }
    else if (om > 1.0 - 1e-12) { ka[0] = (k1 + 1) % C.nphi; wa[0] = 1.0; na = 1; }
    else { ka[0] = k1 % C.nphi; wa[0] = 1.0 - om; ka[1] = (k1 + 1) % C.nphi; wa[1] = om; na = 2; }
    double sw = 0.0;
    for (int ia = 0; ia < na; ++ia) {
        int a = ka[ia];
        double tau = (Rx * (-C.vy[a]) + Ry * C.vx[a]) / C.h + C.c;
        int t1 = (int)std::floor(tau);
        double nu = tau - t1;
        for (int s = 0; s < 2; ++s) {
            int tt = t1 + s;
            double wt = wa[ia] * (s == 0 ? 1.0 - nu : nu);
            if (wt < 1e-9) continue;                       // dropped BEFORE the validity test
            if (tt < 0 || tt >= C.nrot) continue;
            // valid iff that line has a trajectory whose exit (entry) end is on the same wall element;
            // the nearest such end if several
            int best = -1; double bd = 1e300;
            for (int li : C.line[a][tt]) {
                const Traj& T = C.traj[a][li];
                const End& e = want_exit ? T.e_out : T.e_in;
                if (e.elem != elem) continue;
                double ex = e.u * C.vx[a] + lattice_u(C, tt) * (-C.vy[a]);
                double ey = e.u * C.vy[a] + lattice_u(C, tt) * C.vx[a];
                double d = (ex - Rx) * (ex - Rx) + (ey - Ry) * (ey - Ry);
                if (d < bd) { bd = d; best = li; }
            }
            if (best < 0) continue;
            g.idx[g.n] = C.off[a] + best; g.w[g.n] = wt; sw += wt; ++g.n;
        }
    }
    for (int i = 0; i < g.n; ++i) g.w[i] /= sw;
    return g;
}

static int build_tables(Ctx& C) {
    // R1: lattice common to all angles; N_rot = smallest integer >= 2 r_max/h + 2 with N_rot = nx mod 2
    double rmax = 0.0;
    for (auto& s : C.shapes) {
        if (!s.add) continue;
        if (s.kind == 0) rmax = std::max(rmax, std::sqrt(s.cx * s.cx + s.cy * s.cy) + s.r);
        else for (size_t i = 0; i < s.vx.size(); ++i) rmax = std::max(rmax, std::sqrt(s.vx[i] * s.vx[i] + s.vy[i] * s.vy[i]));
    }
    C.nrot = (int)std::ceil(2.0 * rmax / C.h + 2.0 - 1e-9);
    if ((C.nrot - C.nx) % 2 != 0) C.nrot += 1;
    C.c = 0.5 * (C.nrot - 1);
    C.vx.resize(C.nphi); C.vy.resize(C.nphi); C.eta.resize(C.nphi);
    for (int k = 0; k < C.nphi; ++k) {
        double phi = 2.0 * PI * k / C.nphi;              // phi_k = k dphi
        C.vx[k] = std::cos(phi); C.vy[k] = std::sin(phi);
        C.eta[k] = basis(C.sym, phi, C.rot);
    }
    C.W = quadrature(C.nphi, C.quad);
    C.traj.assign(C.nphi, {}); C.line.assign(C.nphi, {}); C.off.assign(C.nphi + 1, 0);
    for (int k = 0; k < C.nphi; ++k) {
        C.line[k].assign(C.nrot, {});
        for (int t = 0; t < C.nrot; ++t) {
            double w = lattice_u(C, t);
            for (auto& iv : clip_line(C.shapes, C.vx[k], C.vy[k], w)) {
                // R3: jf = first j with u_j > u_in, jl = last j with u_j < u_out (strict)
                int jf = (int)std::floor(iv.in.u / C.h + C.c) - 1;
                while (!(lattice_u(C, jf) > iv.in.u)) ++jf;
                int jl = (int)std::floor(iv.out.u / C.h + C.c) + 2;
                while (!(lattice_u(C, jl) < iv.out.u)) --jl;
                if (jf > jl) continue;                     // touches no node: dropped
                if (jf < 0 || jl >= C.nrot) { C.err = "lattice too small"; return 2; }
                Traj T; T.k = k; T.t = t; T.u_in = iv.in.u; T.u_out = iv.out.u; T.jf = jf; T.jl = jl;
                T.e_in = iv.in; T.e_out = iv.out; T.g_in.n = T.g_out.n = 0;
                C.line[k][t].push_back((int)C.traj[k].size());
                C.traj[k].push_back(T);
            }
        }
        C.off[k + 1] = C.off[k] + (int)C.traj[k].size();
    }
    C.ntraj = C.off[C.nphi];
    C.n_gather_fallback = 0;
    for (int k = 0; k < C.nphi; ++k)
        for (auto& T : C.traj[k]) {
            double w = lattice_u(C, T.t), nx = -C.vy[k], ny = C.vx[k];
            double Rx = T.u_in * C.vx[k] + w * nx, Ry = T.u_in * C.vy[k] + w * ny;
            T.g_in = build_gather(C, Rx, Ry, T.e_in.nx, T.e_in.ny, C.vx[k], C.vy[k], T.e_in.elem, true);
            Rx = T.u_out * C.vx[k] + w * nx; Ry = T.u_out * C.vy[k] + w * ny;
            T.g_out = build_gather(C, Rx, Ry, T.e_out.nx, T.e_out.ny, C.vx[k], C.vy[k], T.e_out.elem, false);
            if (T.g_in.n == 0) ++C.n_gather_fallback;
            if (T.g_out.n == 0) ++C.n_gather_fallback;
        }
    return 0;
}

// ---------------------------------------------------------------------------------------------------
// Interpolation ("bilinear interpolation ... from the reference frame to the rotated frame")
// ---------------------------------------------------------------------------------------------------
// R5: Delta = mask-renormalised bilinear over the 4 grid corners (indices clamped); nearest mask point
// within 2 cells if no corner is in the mask.
static cd interp_delta(const Ctx& C, const cd* D, double x, double y, int* bad) {
    double gx = x / C.h + 0.5 * (C.nx - 1), gy = y / C.h + 0.5 * (C.ny - 1);
    int i0 = (int)std::floor(gx), j0 = (int)std::floor(gy);
    double fx = gx - i0, fy = gy - j0;
    double sw = 0.0; cd acc = 0.0;
    for (int b = 0; b < 2; ++b) for (int a = 0; a < 2; ++a) {
        int ii = std::min(std::max(i0 + a, 0), C.nx - 1), jj = std::min(std::max(j0 + b, 0), C.ny - 1);
        double w = (a ? fx : 1.0 - fx) * (b ? fy : 1.0 - fy);
        if (C.mask[(size_t)jj * C.nx + ii]) { sw += w; acc += w * D[(size_t)jj * C.nx + ii]; }
    }
    if (sw > 1e-12) return acc / sw;
    double bd = 1e300; int bi = -1, bj = -1;
    for (int jj = j0 - 2; jj <= j0 + 3; ++jj) for (int ii = i0 - 2; ii <= i0 + 3; ++ii) {
        if (ii < 0 || ii >= C.nx || jj < 0 || jj >= C.ny || !C.mask[(size_t)jj * C.nx + ii]) continue;
        double d = (gx - ii) * (gx - ii) + (gy - jj) * (gy - jj);
        if (d < bd) { bd = d; bi = ii; bj = jj; }
    }
    if (bi < 0) { if (bad) ++*bad; return 0.0; }
    return D[(size_t)bj * C.nx + bi];
}
// A: plain bilinear on the whole grid, indices clamped (A exists outside the grain too).
static double interp_plain(const Ctx& C, const double* F, double x, double y) {
    if (!F) return 0.0;
    double gx = x / C.h + 0.5 * (C.nx - 1), gy = y / C.h + 0.5 * (C.ny - 1);
    int i0 = (int)std::floor(gx), j0 = (int)std::floor(gy);
    double fx = gx - i0, fy = gy - j0, acc = 0.0;
    for (int b = 0; b < 2; ++b) for (int a = 0; a < 2; ++a) {
        int ii = std::min(std::max(i0 + a, 0), C.nx - 1), jj = std::min(std::max(j0 + b, 0), C.ny - 1);
        acc += (a ? fx : 1.0 - fx) * (b ? fy : 1.0 - fy) * F[(size_t)jj * C.nx + ii];
    }
    return acc;
}

// ---------------------------------------------------------------------------------------------------
// Riccati steps (Eq. 25 :169, App. C :968-1003)
//   d gamma / ds = i [ conj(De) gamma^2 + 2 z gamma + De ]            (C1-C2 with v_F = 1)
// ---------------------------------------------------------------------------------------------------
// Delta(p_F, R) of Eq. 1 (:37) for the direction phi at the point (x, y): sum over the components of
// eta_G(phi) times the masked-bilinear interpolant of Delta_G.  `bad` counts the point once.
static cd gap_at(const Ctx& C, const cd* D, double phi, double x, double y, int* bad) {
    const size_t ng = (size_t)C.nx * C.ny;
    cd s = 0.0;
    for (size_t c = 0; c < C.syms.size(); ++c)
        s += basis(C.syms[c], phi, C.rot) * interp_delta(C, D + c * ng, x, y, c == 0 ? bad : nullptr);
    return s;
}

// Homogeneous solution: Omega = sqrt(|De|^2 - z^2) principal branch (Re >= 0),
// gamma_h = -De / (z + i Omega).
// The four functions below are templates on the complex type only so that `orc_opcount` can run the very same
// statements on an operation-counting scalar (bench.py's "textbook" flop count); every caller uses C = cd.
template <class C> static inline C omega_of(C De, C z) { using std::sqrt; using std::norm; return sqrt(C(norm(De), 0.0) - z * z); }
template <class C> static inline C gamma_h(C De, C z) { return -De / (z + C(0.0, 1.0) * omega_of(De, z)); }

// Closed-form ("stepping method") step of length l with constant De, z:
// delta = gamma - gamma_h obeys the Bernoulli equation delta' = -2 Omega delta + i conj(De) delta^2.
template <class C> static inline C step_closed(C g, C De, C z, double l) {
    using std::conj; using std::exp;
    const C I1(0.0, 1.0);
    C Om = omega_of(De, z);
    C gh = -De / (z + I1 * Om);
    C Cc = I1 * conj(De) / (2.0 * Om);
    C e = exp(-2.0 * Om * l);
    C d0 = g - gh;
    return gh + d0 * e / (1.0 + Cc * d0 * (e - 1.0));
}
// Implicit mid-point rule, PAPER.md C4-C9 (:984-1001) verbatim with v_F = 1, h -> l.
template <class C> static inline C step_midpoint(C g, C De, C z, double l) {
    using std::conj; using std::sqrt;
    const C I1(0.0, 1.0);
    C c2 = I1 * (l / 4.0) * conj(De);
    C c1 = 2.0 * c2 * g + I1 * l * z - 1.0;
    C c0 = (c1 - c2 * g + 2.0) * g - 4.0 * conj(c2);
    return 2.0 * c0 / (-c1 + sqrt(c1 * c1 - 4.0 * c2 * c0));
}
static inline cd step(int stepper, cd g, cd De, cd z, double l) {
    return stepper == 1 ? step_midpoint(g, De, z, l) : step_closed(g, De, z, l);
}

// March both coherence functions over a list of pieces (length, De for gamma, Doppler shift a), energy
// z0 (z = z0 + a on each piece).  gamma: pieces in order from g_start, recorded after pieces 0..M-2
// (the nodes).  gamma-tilde: pieces in reverse order from gt_start with De -> -conj(De) (Eq. 26 :172
// integrated along -s), recorded after pieces M-1..1.  Returns the end values.
static void march(int stepper, int M, const double* len, const cd* De, const double* a, cd z0,
                  cd g_start, cd gt_start, cd* G, cd* GT, cd* g_end, cd* gt_end) {
    cd g = g_start;
    for (int m = 0; m < M; ++m) {
        g = step(stepper, g, De[m], z0 + a[m], len[m]);
        if (m < M - 1) G[m] = g;
    }
    *g_end = g;
    cd gt = gt_start;
    for (int m = M - 1; m >= 0; --m) {
        gt = step(stepper, gt, -std::conj(De[m]), z0 + a[m], len[m]);
        if (m >= 1) GT[m - 1] = gt;
    }
    *gt_end = gt;
}

// Node coefficients and pieces of one trajectory (R4, R5; "half-step values by linear
// interpolation; nearest-neighbour extrapolation at the boundary").
struct Pieces {
    int M;                       // number of pieces = nodes + 1
    std::vector<double> len, a;  // per piece
    std::vector<cd> De;          // per piece (Delta eta_k)
    std::vector<cd> Dn;          // per node  (Delta_j eta_k)
    std::vector<double> an;      // per node
};
static void make_pieces(const Ctx& C, const Traj& T, const cd* D, const double* Ax, const double* Ay,
                        Pieces& P, int* bad) {
    int k = T.k, nn = T.jl - T.jf + 1;
    double w = lattice_u(C, T.t), nx = -C.vy[k], ny = C.vx[k];
    P.Dn.resize(nn); P.an.resize(nn);
    for (int m = 0; m < nn; ++m) {
        double u = lattice_u(C, T.jf + m);
        double x = u * C.vx[k] + w * nx, y = u * C.vy[k] + w * ny;
        P.Dn[m] = gap_at(C, D, 2.0 * PI * k / C.nphi, x, y, bad);
        P.an[m] = C.sigma * (C.vx[k] * interp_plain(C, Ax, x, y) + C.vy[k] * interp_plain(C, Ay, x, y));
    }
    P.M = nn + 1; P.len.resize(P.M); P.a.resize(P.M); P.De.resize(P.M);
    P.len[0] = lattice_u(C, T.jf) - T.u_in; P.De[0] = P.Dn[0]; P.a[0] = P.an[0];
    for (int m = 1; m < nn; ++m) {
        P.len[m] = C.h; P.De[m] = 0.5 * (P.Dn[m - 1] + P.Dn[m]); P.a[m] = 0.5 * (P.an[m - 1] + P.an[m]);
    }
    P.len[nn] = T.u_out - lattice_u(C, T.jl); P.De[nn] = P.Dn[nn - 1]; P.a[nn] = P.an[nn - 1];
}

// Start values (R6-R8).  bc_mode 0: specular gather from the previous sweep's end values, fallback =
// homogeneous solution at the boundary point for the mirrored direction; bc_mode 1: homogeneous solution
// of the first (last) piece for the trajectory's own direction.
static cd start_gamma(const Ctx& C, const Traj& T, const Pieces& P, const cd* D, const double* Ax,
                      const double* Ay, const cd* g_old, int ne, int n, cd z0) {
    if (C.bc_mode == 1) return gamma_h(P.De[0], z0 + P.a[0]);
    const Gather& g = T.g_in;
    if (g.n > 0) { cd s = 0.0; for (int i = 0; i < g.n; ++i) s += g.w[i] * g_old[(size_t)g.idx[i] * ne + n]; return s; }
    int k = T.k; double w = lattice_u(C, T.t);
    double x = T.u_in * C.vx[k] - w * C.vy[k], y = T.u_in * C.vy[k] + w * C.vx[k];
    double phi = std::atan2(g.diry, g.dirx);
    cd De = gap_at(C, D, phi, x, y, nullptr);
    double a = C.sigma * (g.dirx * interp_plain(C, Ax, x, y) + g.diry * interp_plain(C, Ay, x, y));
    return gamma_h(De, z0 + a);
}
static cd start_gammat(const Ctx& C, const Traj& T, const Pieces& P, const cd* D, const double* Ax,
                       const double* Ay, const cd* gt_old, int ne, int n, cd z0) {
    // gamma-tilde_h = conj(De)/(z + i Omega) = gamma_h of the tilde equation's De -> -conj(De)
    if (C.bc_mode == 1) return gamma_h(-std::conj(P.De[P.M - 1]), z0 + P.a[P.M - 1]);
    const Gather& g = T.g_out;
    if (g.n > 0) { cd s = 0.0; for (int i = 0; i < g.n; ++i) s += g.w[i] * gt_old[(size_t)g.idx[i] * ne + n]; return s; }
    int k = T.k; double w = lattice_u(C, T.t);
    double x = T.u_out * C.vx[k] - w * C.vy[k], y = T.u_out * C.vy[k] + w * C.vx[k];
    double phi = std::atan2(g.diry, g.dirx);
    cd De = gap_at(C, D, phi, x, y, nullptr);
    double a = C.sigma * (g.dirx * interp_plain(C, Ax, x, y) + g.diry * interp_plain(C, Ay, x, y));
    return gamma_h(-std::conj(De), z0 + a);
}

// ---------------------------------------------------------------------------------------------------
// Operation-counting complex scalar: runs the step templates above and tallies the REAL floating-point operations of
// the textbook complex arithmetic (bench.py reports them as the "textbook" work of one trajectory-step update; the
// tally is derived from the oracle's own statements, nothing is typed in).  Not used by any sweep.
// ---------------------------------------------------------------------------------------------------
namespace opcount {
struct Tally { long mul, add, div, sqrt, exp, sincos; };
static Tally T;
struct CC {
    double re, im;
    CC(double r = 0.0, double i = 0.0) : re(r), im(i) {}
};
static inline CC operator-(CC a) { return CC(-a.re, -a.im); }
static inline CC operator+(CC a, CC b) { T.add += 2; return CC(a.re + b.re, a.im + b.im); }
static inline CC operator-(CC a, CC b) { T.add += 2; return CC(a.re - b.re, a.im - b.im); }
static inline CC operator+(double a, CC b) { T.add += 1; return CC(a + b.re, b.im); }
static inline CC operator-(CC a, double b) { T.add += 1; return CC(a.re - b, a.im); }
static inline CC operator+(CC a, double b) { T.add += 1; return CC(a.re + b, a.im); }
static inline CC operator*(CC a, CC b) { T.mul += 4; T.add += 2; return CC(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re); }
static inline CC operator*(double a, CC b) { T.mul += 2; return CC(a * b.re, a * b.im); }
static inline CC operator*(CC a, double b) { T.mul += 2; return CC(a.re * b, a.im * b); }
static inline CC operator/(CC a, CC b) {             // (a conj b) / |b|^2
    T.mul += 6; T.add += 3; T.div += 2;
    double d = b.re * b.re + b.im * b.im;
    return CC((a.re * b.re + a.im * b.im) / d, (a.im * b.re - a.re * b.im) / d);
}
static inline CC conj(CC a) { return CC(a.re, -a.im); }
static inline double norm(CC a) { T.mul += 2; T.add += 1; return a.re * a.re + a.im * a.im; }
static inline CC sqrt(CC a) {                        // principal branch: |a|, sqrt((|a| + re)/2), im / (2 re')
    T.mul += 4; T.add += 2; T.sqrt += 2; T.div += 1;
    std::complex<double> r = std::sqrt(std::complex<double>(a.re, a.im));
    return CC(r.real(), r.imag());
}
static inline CC exp(CC a) {                         // e^re (cos im + i sin im)
    T.exp += 1; T.sincos += 1; T.mul += 2;
    std::complex<double> r = std::exp(std::complex<double>(a.re, a.im));
    return CC(r.real(), r.imag());
}
}  // namespace opcount

// ---------------------------------------------------------------------------------------------------
// C ABI
// ---------------------------------------------------------------------------------------------------
extern "C" {

struct orc_shape { int kind, add; double cx, cy, r; int nvert; const double *vx, *vy; };

void* orc_create(int nx, int ny, double h, const unsigned char* mask, const orc_shape* shapes, int nshapes,
                 double t, int symmetry, double crystal_rotation, int n_angles, int quadrature_mode,
                 int charge_sign, int bc_mode, int stepper) {
    Ctx* C = new Ctx();
    C->nx = nx; C->ny = ny; C->h = h; C->t = t; C->sym = symmetry; C->rot = crystal_rotation;
    C->nphi = n_angles; C->quad = quadrature_mode; C->sigma = charge_sign; C->bc_mode = bc_mode; C->stepper = stepper;
    for (int s = 0; s < nshapes; ++s) {
        Shape S; S.kind = shapes[s].kind; S.add = shapes[s].add; S.cx = shapes[s].cx; S.cy = shapes[s].cy; S.r = shapes[s].r;
        for (int i = 0; i < shapes[s].nvert; ++i) { S.vx.push_back(shapes[s].vx[i]); S.vy.push_back(shapes[s].vy[i]); }
        C->shapes.push_back(S);
    }
    C->mask.assign(mask, mask + (size_t)nx * ny);
    for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        double x = (i - 0.5 * (nx - 1)) * h, y = (j - 0.5 * (ny - 1)) * h;
        if ((bool)mask[(size_t)j * nx + i] != inside_csg(C->shapes, x, y)) { C->err = "mask disagrees with shapes"; return C; }
    }
    C->syms.assign(1, symmetry);
    build_tables(*C);
    return C;
}
// Several order-parameter components (Eq. 1 :37, Listing 11 :909-926): syms[0..n-1]; afterwards every Delta
// argument is [n][ny][nx] and orc_sweep's num is [n][ny][nx] (num_G = sum_k W_k conj(eta_G,k) SF_k, Eq. 22 :144).
void orc_set_components(void* p, int n, const int* syms) { ((Ctx*)p)->syms.assign(syms, syms + n); }
int orc_ncomp(void* p) { return (int)((Ctx*)p)->syms.size(); }
void orc_destroy(void* p) { delete (Ctx*)p; }
const char* orc_error(void* p) { return ((Ctx*)p)->err.c_str(); }
int orc_nrot(void* p) { return ((Ctx*)p)->nrot; }
int orc_ntraj(void* p) { return ((Ctx*)p)->ntraj; }
int orc_ntraj_angle(void* p, int k) { return (int)((Ctx*)p)->traj[k].size(); }
int orc_traj_offset(void* p, int k) { return ((Ctx*)p)->off[k]; }
int orc_n_gather_fallback(void* p) { return ((Ctx*)p)->n_gather_fallback; }
void orc_angle_info(void* p, int k, double* v, double* eta, double* W) {
    Ctx* C = (Ctx*)p; v[0] = C->vx[k]; v[1] = C->vy[k]; *eta = C->eta[k]; *W = C->W[k];
}
// tables of angle k, for table-level parity: ints [n][6] = t, jf, jl, elem_in, elem_out, (unused);
// doubles [n][6] = u_in, u_out, n_in(x,y), n_out(x,y); gathers: idx [n][2][4] (-1 = unused), w [n][2][4].
void orc_tables(void* p, int k, int* it, double* dt, int* gidx, double* gw) {
    Ctx* C = (Ctx*)p;
    for (size_t i = 0; i < C->traj[k].size(); ++i) {
        const Traj& T = C->traj[k][i];
        it[6 * i + 0] = T.t; it[6 * i + 1] = T.jf; it[6 * i + 2] = T.jl; it[6 * i + 3] = T.e_in.elem; it[6 * i + 4] = T.e_out.elem; it[6 * i + 5] = 0;
        dt[6 * i + 0] = T.u_in; dt[6 * i + 1] = T.u_out; dt[6 * i + 2] = T.e_in.nx; dt[6 * i + 3] = T.e_in.ny; dt[6 * i + 4] = T.e_out.nx; dt[6 * i + 5] = T.e_out.ny;
        for (int s = 0; s < 2; ++s) { const Gather& g = s ? T.g_out : T.g_in;
            for (int q = 0; q < 4; ++q) { gidx[8 * i + 4 * s + q] = q < g.n ? g.idx[q] : -1; gw[8 * i + 4 * s + q] = q < g.n ? g.w[q] : 0.0; } }
    }
}

// Single steps and a synthetic-path march, exposed for the pins (P1, P2, P9, P10).
void orc_step(int stepper, const double* g, const double* De, const double* z, double l, double* out) {
    cd r = step(stepper, cd(g[0], g[1]), cd(De[0], De[1]), cd(z[0], z[1]), l); out[0] = r.real(); out[1] = r.imag();
}
void orc_gamma_h(const double* De, const double* z, double* out) {
    cd r = gamma_h(cd(De[0], De[1]), cd(z[0], z[1])); out[0] = r.real(); out[1] = r.imag();
}
// Real floating-point operations of ONE step (one trajectory-step update of the metric) as the oracle states it:
// counts[6] = mul, add, div, sqrt, exp, sincos.  The step is run on the counting scalar; its value is returned in out
// so that the caller can check it against orc_step.
void orc_opcount(int stepper, const double* g, const double* De, const double* z, double l, long* counts, double* out) {
    using opcount::CC;
    opcount::T = opcount::Tally{0, 0, 0, 0, 0, 0};
    CC r = stepper == 1 ? step_midpoint(CC(g[0], g[1]), CC(De[0], De[1]), CC(z[0], z[1]), l)
                        : step_closed(CC(g[0], g[1]), CC(De[0], De[1]), CC(z[0], z[1]), l);
    counts[0] = opcount::T.mul; counts[1] = opcount::T.add; counts[2] = opcount::T.div;
    counts[3] = opcount::T.sqrt; counts[4] = opcount::T.exp; counts[5] = opcount::T.sincos;
    out[0] = r.re; out[1] = r.im;
}
void orc_march(int stepper, int M, const double* len, const double* De, const double* a, const double* z0,
               const double* g_start, const double* gt_start, double* G, double* GT, double* ends) {
    cd ge, gte;
    march(stepper, M, len, (const cd*)De, a, cd(z0[0], z0[1]), cd(g_start[0], g_start[1]), cd(gt_start[0], gt_start[1]),
          (cd*)G, (cd*)GT, &ge, &gte);
    ends[0] = ge.real(); ends[1] = ge.imag(); ends[2] = gte.real(); ends[3] = gte.imag();
}

// R8: initial boundary stores (Algorithm 1 "Initialize gamma_dD"): gamma_end = gamma_h of
// the last piece (exit point, own direction); gamma-tilde_end = gamma-tilde_h of the first piece.
int orc_reset_stores(void* p, const double* delta, const double* Ax, const double* Ay, int ne,
                     const double* zre, const double* zim, double* g_store, double* gt_store) {
    Ctx* C = (Ctx*)p; const cd* D = (const cd*)delta; cd* gs = (cd*)g_store; cd* gts = (cd*)gt_store;
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : bad)
    for (int k = 0; k < C->nphi; ++k)
        for (size_t i = 0; i < C->traj[k].size(); ++i) {
            Pieces P; make_pieces(*C, C->traj[k][i], D, Ax, Ay, P, &bad);
            for (int n = 0; n < ne; ++n) {
                cd z0(zre[n], zim[n]);
                gs[(size_t)(C->off[k] + i) * ne + n] = gamma_h(P.De[P.M - 1], z0 + P.a[P.M - 1]);
                gts[(size_t)(C->off[k] + i) * ne + n] = gamma_h(-std::conj(P.De[0]), z0 + P.a[0]);
            }
        }
    return bad;
}

// Mask-renormalised bilinear gather of the per-angle node sums back to one grid point (R5 mirrored;
// PAPER.md:189 "summing over energies, and then rotating back to the reference frame").
static bool rotate_back_weights(const Ctx& C, const std::vector<unsigned char>& valid, int k, double x, double y,
                                int idx[4], double w[4], int* n) {
    double uu = (x * C.vx[k] + y * C.vy[k]) / C.h + C.c, ww = (-x * C.vy[k] + y * C.vx[k]) / C.h + C.c;
    int j0 = (int)std::floor(uu), t0 = (int)std::floor(ww);
    double fu = uu - j0, fw = ww - t0, sw = 0.0;
    *n = 0;
    for (int b = 0; b < 2; ++b) for (int a = 0; a < 2; ++a) {
        int jj = j0 + a, tt = t0 + b;
        if (jj < 0 || jj >= C.nrot || tt < 0 || tt >= C.nrot || !valid[(size_t)tt * C.nrot + jj]) continue;
        double wt = (a ? fu : 1.0 - fu) * (b ? fw : 1.0 - fw);
        idx[*n] = tt * C.nrot + jj; w[*n] = wt; sw += wt; ++*n;
    }
    if (sw > 1e-12) { for (int i = 0; i < *n; ++i) w[i] /= sw; return true; }
    double bd = 1e300; int best = -1;
    for (int tt = t0 - 2; tt <= t0 + 3; ++tt) for (int jj = j0 - 2; jj <= j0 + 3; ++jj) {
        if (jj < 0 || jj >= C.nrot || tt < 0 || tt >= C.nrot || !valid[(size_t)tt * C.nrot + jj]) continue;
        double d = (uu - jj) * (uu - jj) + (ww - tt) * (ww - tt);
        if (d < bd) { bd = d; best = tt * C.nrot + jj; }
    }
    if (best < 0) { *n = 0; return false; }
    idx[0] = best; w[0] = 1.0; *n = 1; return true;
}

// One Jacobi sweep (Algorithm 1 :203-205 inner part) over the angles in
// angle_list (NULL = all).  Energies z0[n] = zre + i zim with weights w[n]; z = z0 + sigma_e v.A (C3 :979).
// Accumulates (not finalised):
//   num  = sum_k W_k conj(eta_k) SF_k,  SF_k = sum_n w_n gamma/(1+P)            (c128 [ny][nx])
//   Jx,Jy= sum_k W_k v_k SG_k,          SG_k = sum_n w_n Im[(1-P)/(1+P)]
//   Iacc = sum_k W_k SI_k,              SI_k = sum_n w_n Re[i(D gt - conj(D) g)]   (Eq. 19 :128)
//   Racc = sum_k W_k SR_k,              SR_k = sum_n w_n Re[(1-P)/(1+P)]            (Eq. 14 :100 -> LDOS)
// with P = gamma gamma-tilde at every lattice node (Eq. 24 :165).  Reads the old stores, writes the new.
int orc_sweep(void* p, const double* delta, const double* Ax, const double* Ay,
              int ne, const double* zre, const double* zim, const double* wn,
              const double* g_old, const double* gt_old, double* g_new, double* gt_new,
              double* num, double* Jx, double* Jy, double* Iacc, double* Racc,
              const int* angle_list, int n_angle_list,
              int dbg_angle, double* dbg_SF, double* dbg_SG, double* dbg_SI, double* dbg_SR,
              double* stat_min_one_minus_abs, long long* stat_updates, int* stat_bad) {
    Ctx* C = (Ctx*)p; const cd* D = (const cd*)delta;
    const cd* go = (const cd*)g_old; const cd* gto = (const cd*)gt_old; cd* gn = (cd*)g_new; cd* gtn = (cd*)gt_new;
    size_t ng = (size_t)C->nx * C->ny, nl = (size_t)C->nrot * C->nrot;
    std::vector<int> angles;
    if (angle_list) angles.assign(angle_list, angle_list + n_angle_list);
    else for (int k = 0; k < C->nphi; ++k) angles.push_back(k);
    const size_t ncomp = C->syms.size();
    for (size_t q = 0; q < 2 * ng * ncomp; ++q) num[q] = 0.0;
    for (size_t q = 0; q < ng; ++q) { Jx[q] = Jy[q] = Iacc[q] = Racc[q] = 0.0; }
    double gmin = 1e300; long long nupd = 0; int bad = 0;
#pragma omp parallel for ordered schedule(dynamic, 1) reduction(min : gmin) reduction(+ : nupd, bad)
    for (int ia = 0; ia < (int)angles.size(); ++ia) {
        int k = angles[ia];
        std::vector<cd> SF(nl, 0.0); std::vector<double> SG(nl, 0.0), SI(nl, 0.0), SR(nl, 0.0);
        std::vector<unsigned char> valid(nl, 0);
        std::vector<cd> G, GT; Pieces P;
        for (size_t i = 0; i < C->traj[k].size(); ++i) {
            const Traj& T = C->traj[k][i];
            make_pieces(*C, T, D, Ax, Ay, P, &bad);
            int nn = P.M - 1; G.resize(nn); GT.resize(nn);
            size_t gid = (size_t)C->off[k] + i;
            for (int n = 0; n < ne; ++n) {
                cd z0(zre[n], zim[n]);
                cd gs = start_gamma(*C, T, P, D, Ax, Ay, go, ne, n, z0);
                cd gts = start_gammat(*C, T, P, D, Ax, Ay, gto, ne, n, z0);
                cd ge, gte;
                march(C->stepper, P.M, P.len.data(), P.De.data(), P.a.data(), z0, gs, gts, G.data(), GT.data(), &ge, &gte);
                gn[gid * ne + n] = ge; gtn[gid * ne + n] = gte;
                nupd += 2LL * P.M;
                for (int m = 0; m < nn; ++m) {
                    size_t q = (size_t)T.t * C->nrot + (T.jf + m);
                    cd Pq = G[m] * GT[m];
                    cd gnorm = (1.0 - Pq) / (1.0 + Pq);
                    SF[q] += wn[n] * G[m] / (1.0 + Pq);
                    SG[q] += wn[n] * gnorm.imag();
                    SR[q] += wn[n] * gnorm.real();
                    SI[q] += wn[n] * (I_ * (P.Dn[m] * GT[m] - std::conj(P.Dn[m]) * G[m])).real();
                    gmin = std::min(gmin, std::min(1.0 - std::abs(G[m]), 1.0 - std::abs(GT[m])));
                }
            }
            for (int m = 0; m < nn; ++m) valid[(size_t)T.t * C->nrot + (T.jf + m)] = 1;
        }
        // parity tap: the per-angle node sums of angle dbg_angle, or (dbg_angle == -2) of every angle of angle_list,
        // [position in angle_list][N_rot][N_rot]
        if ((k == dbg_angle || dbg_angle == -2) && dbg_SF) {
            size_t o = dbg_angle == -2 ? (size_t)ia * nl : 0;
            std::memcpy(dbg_SF + 2 * o, SF.data(), nl * sizeof(cd)); std::memcpy(dbg_SG + o, SG.data(), nl * sizeof(double));
            std::memcpy(dbg_SI + o, SI.data(), nl * sizeof(double)); std::memcpy(dbg_SR + o, SR.data(), nl * sizeof(double));
        }
#pragma omp ordered
        {
            for (int j = 0; j < C->ny; ++j) for (int i = 0; i < C->nx; ++i) {
                size_t q = (size_t)j * C->nx + i;
                if (!C->mask[q]) continue;
                double x = (i - 0.5 * (C->nx - 1)) * C->h, y = (j - 0.5 * (C->ny - 1)) * C->h;
                int idx[4], n; double w[4];
                if (!rotate_back_weights(*C, valid, k, x, y, idx, w, &n)) { ++bad; continue; }
                cd F = 0.0; double Gv = 0.0, Iv = 0.0, Rv = 0.0;
                for (int s = 0; s < n; ++s) { F += w[s] * SF[idx[s]]; Gv += w[s] * SG[idx[s]]; Iv += w[s] * SI[idx[s]]; Rv += w[s] * SR[idx[s]]; }
                for (size_t cc = 0; cc < ncomp; ++cc) {      // eta real: conj(eta_G,k) = eta_G,k
                    cd c = C->W[k] * basis(C->syms[cc], 2.0 * PI * k / C->nphi, C->rot) * F;
                    num[2 * (cc * ng + q)] += c.real(); num[2 * (cc * ng + q) + 1] += c.imag();
                }
                Jx[q] += C->W[k] * C->vx[k] * Gv; Jy[q] += C->W[k] * C->vy[k] * Gv;
                Iacc[q] += C->W[k] * Iv; Racc[q] += C->W[k] * Rv;
            }
        }
    }
    if (stat_min_one_minus_abs) *stat_min_one_minus_abs = gmin;
    if (stat_updates) *stat_updates = nupd;
    if (stat_bad) *stat_bad = bad;
    return 0;
}

// gamma, gamma-tilde at the nodes of one trajectory for one energy (parity tap).
int orc_debug_trajectory(void* p, const double* delta, const double* Ax, const double* Ay, int k, int local,
                         int ne, int n, const double* zre, const double* zim, const double* g_old, const double* gt_old,
                         double* G, double* GT, double* ends) {
    Ctx* C = (Ctx*)p; const cd* D = (const cd*)delta; const Traj& T = C->traj[k][local];
    Pieces P; int bad = 0; make_pieces(*C, T, D, Ax, Ay, P, &bad);
    cd z0(zre[n], zim[n]);
    cd gs = start_gamma(*C, T, P, D, Ax, Ay, (const cd*)g_old, ne, n, z0);
    cd gts = start_gammat(*C, T, P, D, Ax, Ay, (const cd*)gt_old, ne, n, z0);
    cd ge, gte;
    march(C->stepper, P.M, P.len.data(), P.De.data(), P.a.data(), z0, gs, gts, (cd*)G, (cd*)GT, &ge, &gte);
    ends[0] = ge.real(); ends[1] = ge.imag(); ends[2] = gte.real(); ends[3] = gte.imag();
    ends[4] = gs.real(); ends[5] = gs.imag(); ends[6] = gts.real(); ends[7] = gts.imag();
    return P.M - 1;
}
// node coefficients of one trajectory (rotate-in parity tap): Dn c128[nn], an f64[nn]
int orc_debug_nodes(void* p, const double* delta, const double* Ax, const double* Ay, int k, int local, double* Dn, double* an) {
    Ctx* C = (Ctx*)p; Pieces P; int bad = 0; make_pieces(*C, C->traj[k][local], (const cd*)delta, Ax, Ay, P, &bad);
    std::memcpy(Dn, P.Dn.data(), P.Dn.size() * sizeof(cd)); std::memcpy(an, P.an.data(), P.an.size() * sizeof(double));
    return (int)P.Dn.size();
}

// Vector potential (App. D): G_{m,n} closed form D3-D6 (:1014-1021), lengths in xi0.
static double Gam(double m, double n) {
    auto alpha = [](double m, double n) { return (1 + 2 * m) * (1 + 2 * n) * std::log(0.5 * (1 + 2 * m) * (1 + 2 * m) + 0.5 * (1 + 2 * n) * (1 + 2 * n)); };
    auto beta = [](double m, double n) { return (-2 * m * m + 2 * n * n + 4 * n + 1) * std::atan((1 + 2 * m) / (1 + 2 * n)); };
    return alpha(m, n) + beta(m, n) + beta(n, m);
}
double orc_G(int m, int n, double h) {
    double s = 0.0;
    for (int a = -1; a <= 1; a += 2) for (int b = -1; b <= 1; b += 2) s += Gam(a * (double)m, b * (double)n);
    return h * h / (4.0 * PI) * (2.0 * std::log(h) - std::log(2.0) - 3.0 + 0.25 * s);
}
// D1 (:1009) by direct summation with the mask-mean of j subtracted first (:1040; R17: mean over mask
// points): A_ind = -(1/kappa^2) sum_{m'n'} G_{|m'-m|,|n'-n|} (j - <j>)_{m'n'} on the whole grid.
void orc_vector_potential(int nx, int ny, double h, const unsigned char* mask, double kappa,
                          const double* jx, const double* jy, double* Ax, double* Ay) {
    size_t ng = (size_t)nx * ny;
    double mx = 0, my = 0; long cnt = 0;
    for (size_t q = 0; q < ng; ++q) if (mask[q]) { mx += jx[q]; my += jy[q]; ++cnt; }
    if (cnt) { mx /= cnt; my /= cnt; }
    std::vector<double> G((size_t)nx * ny);
    for (int n = 0; n < ny; ++n) for (int m = 0; m < nx; ++m) G[(size_t)n * nx + m] = orc_G(m, n, h);
    std::vector<double> sx(ng, 0.0), sy(ng, 0.0);
    for (size_t q = 0; q < ng; ++q) if (mask[q]) { sx[q] = jx[q] - mx; sy[q] = jy[q] - my; }
#pragma omp parallel for schedule(static)
    for (int n = 0; n < ny; ++n) for (int m = 0; m < nx; ++m) {
        double ax = 0, ay = 0;
        for (int n2 = 0; n2 < ny; ++n2) for (int m2 = 0; m2 < nx; ++m2) {
            size_t q = (size_t)n2 * nx + m2; if (!mask[q]) continue;
            double g = G[(size_t)std::abs(n2 - n) * nx + std::abs(m2 - m)];
            ax += g * sx[q]; ay += g * sy[q];
        }
        Ax[(size_t)n * nx + m] = -ax / (kappa * kappa); Ay[(size_t)n * nx + m] = -ay / (kappa * kappa);
    }
}

}  // extern "C"
