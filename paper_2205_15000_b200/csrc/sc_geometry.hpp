// sc_geometry.hpp — host-side trajectory generator of the CUDA library (step a1 of DESIGN.md §2).
//
// For every Fermi angle phi_k it lays the rotated square lattice of spacing h over the grain
// (Fig. 2 d-f :195), clips every lattice line against the exact grain boundary
// (:189 "exact location and shape of boundaries"), and builds the specular boundary-gather tables
// (:155, :161, :191-197).  Readings R1-R9 of DESIGN.md §3.  Product code: shares nothing with oracle/.
//
// Method (deliberately different from a per-shape interval algebra): all crossings of a line with all
// shape boundaries are collected as events, sorted along the line, and the segment between consecutive
// events is kept iff its midpoint is inside the CSG; kept neighbours are fused.  Angles k >= N_phi/2 are
// the exact mirror images (j,t) -> (N_rot-1-j, N_rot-1-t) of angle k - N_phi/2 (v -> -v), which is what
// lets the march kernel obtain gamma-tilde_k from gamma_{k+N/2} (Eq. 13 :95).
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <string>
#include <vector>

namespace scgeo {

struct ShapeH { int kind, add; double cx, cy, r; std::vector<double> vx, vy; };

struct Crossing { double u; int elem; double nx, ny; };   // normal = outward of the GRAIN

struct DTraj {                 // one directed trajectory (angle k, line t)
    int k, t, jf, jl;
    double u_in, u_out;
    int elem_in, elem_out;
    double nin[2], nout[2];
    int gn; int gidx[4]; double gw[4];     // entry gather (start value of gamma): directed-trajectory ids
    double mdir[2];                        // mirrored direction at the entry point (fallback)
};

struct Geometry {
    int nx, ny; double h;
    int nphi, nrot; double c;
    std::vector<ShapeH> shapes;
    std::vector<double> vx, vy, eta, W;
    std::vector<DTraj> dt;                 // angle-major, then line order
    std::vector<int> aoff;                 // first directed trajectory of each angle (size nphi+1)
    std::vector<int> line_first;           // [k*nrot + t] -> id of first directed trajectory on that line, or -1
    std::vector<int> line_count;
    int n_fallback = 0;
    std::string err;
};

static const double kPi = 3.141592653589793238462643383279502884;

inline double eta_of(int sym, double phi, double rot_turns) {
    const double a = phi - 2.0 * kPi * rot_turns;
    if (sym == 1) return std::sqrt(2.0) * std::cos(2.0 * a);
    if (sym == 2) return std::sqrt(2.0) * std::sin(2.0 * a);
    if (sym == 3) return std::sqrt(2.0) * std::sin(4.0 * a);
    return 1.0;
}

inline bool in_shape_strict(const ShapeH& s, double x, double y, bool closed) {
    if (s.kind == 0) {
        const double d2 = (x - s.cx) * (x - s.cx) + (y - s.cy) * (y - s.cy);
        return closed ? d2 <= s.r * s.r : d2 < s.r * s.r;
    }
    const size_t nv = s.vx.size();
    for (size_t e = 0; e < nv; ++e) {
        const double ax = s.vx[e], ay = s.vy[e], bx = s.vx[(e + 1) % nv], by = s.vy[(e + 1) % nv];
        const double ex = bx - ax, ey = by - ay, len = std::hypot(ex, ey);
        // signed distance to the edge line, positive outside for CCW order
        const double sd = (ey * (x - ax) - ex * (y - ay)) / len;
        if (!(sd < 0.0)) return false;
    }
    return true;
}

inline bool in_grain(const std::vector<ShapeH>& S, double x, double y) {
    bool in = false;
    for (const auto& s : S) {
        if (s.add) { if (in_shape_strict(s, x, y, false)) in = true; }
        else if (in_shape_strict(s, x, y, true)) in = false;
    }
    return in;
}

// crossings of the line P(u) = u*v + w*n with the boundary of one shape
inline void shape_events(const ShapeH& s, int sid, double vx, double vy, double w, std::vector<Crossing>& ev) {
    const double px = -w * vy, py = w * vx;     // foot point of the line (u = 0)
    const double sgn = s.add ? 1.0 : -1.0;      // removed shape: grain normal points into the shape
    if (s.kind == 0) {
        const double qx = px - s.cx, qy = py - s.cy;
        const double b = qx * vx + qy * vy;             // u^2 + 2 b u + cc = 0
        const double cc = qx * qx + qy * qy - s.r * s.r;
        const double disc = b * b - cc;
        if (!(disc > 0.0)) return;
        const double sq = std::sqrt(disc);
        for (int side = 0; side < 2; ++side) {
            const double u = side ? -b + sq : -b - sq;
            Crossing c; c.u = u; c.elem = sid * 65536;
            c.nx = sgn * (qx + u * vx) / s.r; c.ny = sgn * (qy + u * vy) / s.r;
            ev.push_back(c);
        }
        return;
    }
    // Cyrus-Beck against a convex CCW polygon
    const size_t nv = s.vx.size();
    double ulo = -1e300, uhi = 1e300; int elo = -1, ehi = -1; double nlo[2] = {0, 0}, nhi[2] = {0, 0};
    for (size_t e = 0; e < nv; ++e) {
        const double ax = s.vx[e], ay = s.vy[e], bx = s.vx[(e + 1) % nv], by = s.vy[(e + 1) % nv];
        const double ex = bx - ax, ey = by - ay, len = std::hypot(ex, ey);
        const double ox = ey / len, oy = -ex / len;                 // outward normal
        const double denom = ox * vx + oy * vy;
        const double dist0 = ox * (ax - px) + oy * (ay - py);       // inside iff u*denom < dist0
        if (std::fabs(denom) <= 1e-12) { if (!(dist0 > 0.0)) return; continue; }
        const double uc = dist0 / denom;
        if (denom > 0.0) { if (uc < uhi) { uhi = uc; ehi = (int)e; nhi[0] = ox; nhi[1] = oy; } }
        else if (uc > ulo) { ulo = uc; elo = (int)e; nlo[0] = ox; nlo[1] = oy; }
    }
    if (elo < 0 || ehi < 0 || !(uhi > ulo)) return;
    ev.push_back(Crossing{ulo, sid * 65536 + elo, sgn * nlo[0], sgn * nlo[1]});
    ev.push_back(Crossing{uhi, sid * 65536 + ehi, sgn * nhi[0], sgn * nhi[1]});
}

struct Seg { Crossing a, b; };

inline std::vector<Seg> clip(const std::vector<ShapeH>& S, double vx, double vy, double w) {
    std::vector<Crossing> ev;
    for (size_t s = 0; s < S.size(); ++s) shape_events(S[s], (int)s, vx, vy, w, ev);
    std::stable_sort(ev.begin(), ev.end(), [](const Crossing& p, const Crossing& q) { return p.u < q.u; });
    std::vector<Seg> out;
    for (size_t i = 0; i + 1 < ev.size(); ++i) {
        if (!(ev[i + 1].u - ev[i].u > 0.0)) continue;
        // between two consecutive crossings the line is either inside or outside, except at a point where it only
        // touches a boundary (a lattice line tangent to a hole): sample two points, neither the midpoint
        const double u1 = ev[i].u + 0.37 * (ev[i + 1].u - ev[i].u), u2 = ev[i].u + 0.71 * (ev[i + 1].u - ev[i].u);
        if (!in_grain(S, u1 * vx - w * vy, u1 * vy + w * vx) && !in_grain(S, u2 * vx - w * vy, u2 * vy + w * vx)) continue;
        if (!out.empty() && out.back().b.u == ev[i].u) out.back().b = ev[i + 1];   // fuse through an interior crossing
        else out.push_back(Seg{ev[i], ev[i + 1]});
    }
    return out;
}

inline std::vector<double> fs_weights(int n, int mode) {
    std::vector<double> W(n, 1.0 / n);
    if (mode == 1) return W;
    if (n % 4 == 0) { const double p[4] = {28.0, 64.0, 24.0, 64.0}; for (int k = 0; k < n; ++k) W[k] = p[k & 3] / (45.0 * n); }
    else if (n % 3 == 0) { const double p[3] = {6.0, 9.0, 9.0}; for (int k = 0; k < n; ++k) W[k] = p[k % 3] / (8.0 * n); }
    else if (n % 2 == 0) { for (int k = 0; k < n; ++k) W[k] = (k & 1 ? 4.0 : 2.0) / (3.0 * n); }
    return W;
}

inline int build(Geometry& G, int sym, double rot, int quad) {
    if (G.nphi < 2 || (G.nphi & 1)) { G.err = "n_angles must be even"; return 2; }
    double rmax = 0.0;
    for (const auto& s : G.shapes) {
        if (!s.add) continue;
        if (s.kind == 0) rmax = std::max(rmax, std::hypot(s.cx, s.cy) + s.r);
        else for (size_t i = 0; i < s.vx.size(); ++i) rmax = std::max(rmax, std::hypot(s.vx[i], s.vy[i]));
    }
    G.nrot = (int)std::ceil(2.0 * rmax / G.h + 2.0 - 1e-9);
    if (((G.nrot - G.nx) & 1) != 0) ++G.nrot;
    G.c = 0.5 * (G.nrot - 1);
    const int N = G.nphi, H = N / 2, NR = G.nrot;
    G.vx.resize(N); G.vy.resize(N); G.eta.resize(N);
    for (int k = 0; k < N; ++k) {
        const double phi = 2.0 * kPi * k / N;
        G.eta[k] = eta_of(sym, phi, rot);
        if (k < H) { G.vx[k] = std::cos(phi); G.vy[k] = std::sin(phi); }
        else { G.vx[k] = -G.vx[k - H]; G.vy[k] = -G.vy[k - H]; }
    }
    G.W = fs_weights(N, quad);
    auto U = [&](int j) { return (j - G.c) * G.h; };
    // first half of the angles: clip; second half: mirror
    std::vector<std::vector<DTraj>> per(N);
    for (int k = 0; k < H; ++k) {
        for (int t = 0; t < NR; ++t) {
            for (const Seg& sg : clip(G.shapes, G.vx[k], G.vy[k], U(t))) {
                int jf = (int)std::floor(sg.a.u / G.h + G.c) - 1;
                while (!(U(jf) > sg.a.u)) ++jf;
                int jl = (int)std::floor(sg.b.u / G.h + G.c) + 2;
                while (!(U(jl) < sg.b.u)) --jl;
                if (jf > jl) continue;
                if (jf < 0 || jl >= NR) { G.err = "rotated lattice too small"; return 2; }
                DTraj d{}; d.k = k; d.t = t; d.jf = jf; d.jl = jl; d.u_in = sg.a.u; d.u_out = sg.b.u;
                d.elem_in = sg.a.elem; d.elem_out = sg.b.elem;
                d.nin[0] = sg.a.nx; d.nin[1] = sg.a.ny; d.nout[0] = sg.b.nx; d.nout[1] = sg.b.ny;
                per[k].push_back(d);
            }
        }
        // mirror: line t -> NR-1-t, node j -> NR-1-j, u -> -u; keep ascending (t, u) order
        for (auto it = per[k].rbegin(); it != per[k].rend(); ++it) {
            DTraj m{}; m.k = k + H; m.t = NR - 1 - it->t; m.jf = NR - 1 - it->jl; m.jl = NR - 1 - it->jf;
            m.u_in = -it->u_out; m.u_out = -it->u_in; m.elem_in = it->elem_out; m.elem_out = it->elem_in;
            m.nin[0] = it->nout[0]; m.nin[1] = it->nout[1]; m.nout[0] = it->nin[0]; m.nout[1] = it->nin[1];
            per[k + H].push_back(m);
        }
    }
    G.aoff.assign(N + 1, 0); G.dt.clear();
    G.line_first.assign((size_t)N * NR, -1); G.line_count.assign((size_t)N * NR, 0);
    for (int k = 0; k < N; ++k) {
        for (const auto& d : per[k]) {
            const size_t li = (size_t)k * NR + d.t;
            if (G.line_first[li] < 0) G.line_first[li] = (int)G.dt.size();
            ++G.line_count[li];
            G.dt.push_back(d);
        }
        G.aoff[k + 1] = (int)G.dt.size();
    }
    // entry gathers (R6): start value of gamma on (k,t) = interpolation over directed trajectories that
    // EXIT on the same wall element, bracketing the mirrored direction in angle and the entry point in
    // perpendicular offset.
    const double dphi = 2.0 * kPi / N;
    G.n_fallback = 0;
    for (auto& d : G.dt) {
        const double vx = G.vx[d.k], vy = G.vy[d.k], w = U(d.t);
        const double Rx = d.u_in * vx - w * vy, Ry = d.u_in * vy + w * vx;
        const double vn = vx * d.nin[0] + vy * d.nin[1];
        const double mx = vx - 2.0 * vn * d.nin[0], my = vy - 2.0 * vn * d.nin[1];
        d.mdir[0] = mx; d.mdir[1] = my;
        double kap = std::atan2(my, mx) / dphi;
        kap -= N * std::floor(kap / N);
        const int k1 = (int)std::floor(kap);
        const double om = kap - k1;
        int ang[2]; double wa[2]; int na;
        if (om < 1e-12) { ang[0] = k1 % N; wa[0] = 1.0; na = 1; }
        else if (om > 1.0 - 1e-12) { ang[0] = (k1 + 1) % N; wa[0] = 1.0; na = 1; }
        else { ang[0] = k1 % N; wa[0] = 1.0 - om; ang[1] = (k1 + 1) % N; wa[1] = om; na = 2; }
        d.gn = 0; double sw = 0.0;
        for (int q = 0; q < na; ++q) {
            const int a = ang[q];
            const double tau = (-Rx * G.vy[a] + Ry * G.vx[a]) / G.h + G.c;
            const int t1 = (int)std::floor(tau);
            const double nu = tau - t1;
            for (int s = 0; s < 2; ++s) {
                const int tt = t1 + s;
                const double wt = wa[q] * (s ? nu : 1.0 - nu);
                if (wt < 1e-9 || tt < 0 || tt >= NR) continue;
                const size_t li = (size_t)a * NR + tt;
                int best = -1; double bd = 1e300;
                for (int c = 0; c < G.line_count[li]; ++c) {
                    const DTraj& o = G.dt[G.line_first[li] + c];
                    if (o.elem_out != d.elem_in) continue;
                    const double ex = o.u_out * G.vx[a] - U(tt) * G.vy[a], ey = o.u_out * G.vy[a] + U(tt) * G.vx[a];
                    const double dd = (ex - Rx) * (ex - Rx) + (ey - Ry) * (ey - Ry);
                    if (dd < bd) { bd = dd; best = G.line_first[li] + c; }
                }
                if (best < 0) continue;
                d.gidx[d.gn] = best; d.gw[d.gn] = wt; sw += wt; ++d.gn;
            }
        }
        for (int i = 0; i < d.gn; ++i) d.gw[i] /= sw;
        if (d.gn == 0) ++G.n_fallback;
    }
    return 0;
}

}  // namespace scgeo
