"""Pins of the oracle's self-consistency driver (`oracle.Driver`, Algorithm 1) and of its handling of
crystal-axes rotation, against what the theory fixes (VERDICT r1 "weak #2", north_star "div j ~ 0"):

  * charge conservation: at self-consistency div j = 0 (:114 "the gap equation ... guarantees current conservation").
    Integrated over a full cross-section of an isolated grain this says that NO net current crosses it; the discrete
    scheme obeys that to the level of the residual, and violates it by 30 % of the circulating current for a
    non-self-consistent Delta.  The pointwise divergence falls to its discretisation floor.
  * the converged (Delta, A_ind) is a fixed point of the independently composed map sweep -> D1 A-solve (hook-up of the
    kappa^2-scaled iterate x of E3 :1053), and the induced field screens the applied one (Meissner, Eq. 45 :602).
  * rotation covariance (P11, A12): a square rotated by 1/8 turn with d_{x^2-y^2} pairing is the axis-aligned square
    with the crystal axes rotated by 1/8 turn (:890): same lattice sums, angle index shifted by N_phi/8.
"""
import math

import numpy as np
import pytest

import oracle
import workloads as wlmod
from workloads import make_mask, square


def _div(jx, jy, mask, h):
    m = mask > 0
    inner = np.zeros_like(m)
    inner[1:-1, 1:-1] = m[1:-1, 1:-1] & m[1:-1, 2:] & m[1:-1, :-2] & m[2:, 1:-1] & m[:-2, 1:-1]
    d = np.zeros_like(jx)
    d[1:-1, 1:-1] = (jx[1:-1, 2:] - jx[1:-1, :-2] + jy[2:, 1:-1] - jy[:-2, 1:-1]) / (2 * h)
    return np.max(np.abs(d[inner]))


def _grain(kappa):
    """configs[0]-sized grain (square side 5 xi0, h = 0.1, 16 angles, 16 Matsubara energies, t = 0.5) in a field of 1.5
    flux quanta, seeded amplitude and phase noise on the bulk gap"""
    L, h, nphi, ne, t, flux = 5.0, 0.1, 16, 16, 0.5, 1.5
    n = int(round(L / h))
    shapes = [square(L)]
    mask = make_mask(shapes, n, n, h)
    X, Y = wlmod.grid_xy(n, n, h)
    B = math.pi * flux / (L * L)                                   # B_ext = Phi / area in units of Phi0 / (pi xi0^2)
    rng = np.random.default_rng(1)
    d0 = wlmod.BULK_GAP[("s", 0.5, 16)] * (1 + 0.1 * rng.uniform(-1, 1, (n, n))) * np.exp(0.3j * rng.uniform(-1, 1, (n, n))) * mask
    o = oracle.Oracle(n, n, h, mask, shapes, t, wlmod.SYM_S, nphi, kappa=kappa)
    return dict(o=o, n=n, h=h, ne=ne, mask=mask, B=B, Aext=(-0.5 * B * Y, 0.5 * B * X), d0=d0)


def _converge(G, accelerator, step, nit=300, tol=1e-8):
    o, n, h = G["o"], G["n"], G["h"]
    drv = oracle.Driver(o, G["Aext"][0], G["Aext"][1], G["ne"], accelerator=accelerator, step=step)
    d, ax, ay = G["d0"], np.zeros((n, n)), np.zeros((n, n))
    hist = []
    for _ in range(nit):
        r = drv.iterate(d, ax, ay)
        net = max(np.max(np.abs(h * np.sum(r["jx"], axis=0))), np.max(np.abs(h * np.sum(r["jy"], axis=1))))   # through x = x_i, y = y_j
        circ = np.max(h * np.sum(np.abs(r["jx"]), axis=0))
        hist.append((r["res_delta"], _div(r["jx"], r["jy"], G["mask"], h), net, circ))
        d, ax, ay = r["delta"], r["Aind_x"], r["Aind_y"]
        if r["res_delta"] < tol:
            break
    return drv, d, ax, ay, r, np.array(hist)


@pytest.mark.parametrize("kappa,accelerator,step", [(-1.0, 0, 0.7), (3.0, 1, 1.0)])
def test_current_is_conserved_at_self_consistency(kappa, accelerator, step):
    G = _grain(kappa)
    drv, d, ax, ay, r, hist = _converge(G, accelerator, step)
    res, div, net, circ = hist.T
    assert res[-1] < 1e-8 and len(res) < 300
    # the start is far from conserving: 11 % of the circulating current leaks through a cross-section, |div j| xi0 ~ |j|
    assert net[0] > 0.1 * circ[0] and div[0] > 0.15
    # integral form: the net current through every full cross-section vanishes WITH the residual
    assert net[-1] < 1e-6 * circ[-1]
    late = res < 1e-3
    assert np.all(net[late] < 100.0 * res[late] * circ[late] + 1e-9)    # residual = last step; the distance to the fixed point is res / (1 - rate)
    # pointwise: falls to the discretisation floor (measured 6.1e-3 at h = 0.1, 16 angles) and stays there
    assert div[-1] < div[0] / 25 and div[-1] < 0.05 * np.max(np.hypot(r["jx"], r["jy"])) / 1.0
    assert np.all(np.abs(div[late] - div[-1]) < 0.05 * div[-1])
    assert np.max(np.hypot(r["jx"], r["jy"])) > 0.1                      # a real circulating Meissner current


def test_driver_fixed_point_is_the_fixed_point_of_sweep_and_D1():
    """kappa = 3: the converged (Delta*, A*) must satisfy Delta* = Delta_new(Delta*, A_ext + A*) and A* = D1[j(Delta*, A_ext + A*)]
    with the sweep and `oracle.vector_potential` called directly (none of Driver's bookkeeping: kappa^2 scaling of the
    iterate E3 :1053, the accelerator, the mask multiply), and the induced field must screen the applied one."""
    G = _grain(3.0)
    o, n, h, ne = G["o"], G["n"], G["h"], G["ne"]
    drv, d, ax, ay, r, hist = _converge(G, 1, 1.0, tol=1e-9)
    Ax, Ay = G["Aext"][0] + ax, G["Aext"][1] + ay
    st = o.reset_stores(d, Ax, Ay, o.matsubara(ne)[0])
    for _ in range(40):                                                   # boundary values at frozen fields
        rr = o.sweep(d, Ax, Ay, ne, st)
        st = rr["stores"]
    assert np.max(np.abs(rr["delta_new"] - d)) < 1e-7 * np.max(np.abs(d))
    gax, gay = oracle.vector_potential(G["mask"], h, 3.0, rr["jx"], rr["jy"])
    assert np.max(np.abs(gax - ax)) < 1e-6 * np.max(np.abs(ax)) and np.max(np.abs(gay - ay)) < 1e-6 * np.max(np.abs(ay))
    assert np.all(d[G["mask"] == 0] == 0)
    # Meissner screening (Eq. 45 :602): B_ind = curl A_ind opposes B_ext at the centre and is weaker
    c = n // 2
    Bind = ((ay[c, c + 1] - ay[c, c - 1]) - (ax[c + 1, c] - ax[c - 1, c])) / (2 * h)
    assert Bind * G["B"] < 0 and 0.02 * G["B"] < abs(Bind) < G["B"]
    # and the screening current flows against A in the interior (diamagnetic)
    assert rr["jx"][c + 10, c] * Ax[c + 10, c] < 0


def test_P11_rotated_square_equals_axis_aligned_square_with_rotated_crystal_axes():
    """Uniform d_{x^2-y^2} gap and a uniform vector potential.  Grain A: square rotated by 1/8 turn ([110] walls).  Grain B:
    the same square axis-aligned with the crystal axes (and A) rotated by -1/8 turn.  B is A turned by -45 degrees, so with
    N_phi a multiple of 8 trajectory set k of A is set k - N_phi/8 of B: the lattices coincide node for node (same N_rot
    parity), hence after 3 Jacobi sweeps the per-angle lattice sums agree to rounding, and so does Delta_new at the centre."""
    L, h, nphi, ne, t = 2.03, 0.1, 32, 6, 0.3       # N_phi / 8 = 4: the period of Boole's weight pattern (:189)
    D0 = 0.2 * np.exp(0.4j)
    A0 = np.array([0.05, -0.02])
    c8, s8 = math.cos(math.pi / 4), math.sin(math.pi / 4)
    res = {}
    for name, rot_shape, rot_crystal, n, Avec in (("A", 0.125, 0.0, 31, A0),
                                                  ("B", 0.0, -0.125, 21, np.array([c8 * A0[0] + s8 * A0[1], -s8 * A0[0] + c8 * A0[1]]))):
        # centre of the square off the origin (at (0.013, 0.007) in B's frame), so that no lattice line runs through a corner
        ca_, sa_ = math.cos(2 * math.pi * rot_shape), math.sin(2 * math.pi * rot_shape)
        base = [(-L / 2 + 0.013, -L / 2 + 0.007), (L / 2 + 0.013, -L / 2 + 0.007), (L / 2 + 0.013, L / 2 + 0.007), (-L / 2 + 0.013, L / 2 + 0.007)]
        shapes = [wlmod.Shape(kind=1, vx=[ca_ * x - sa_ * y for x, y in base], vy=[sa_ * x + ca_ * y for x, y in base])]
        mask = make_mask(shapes, n, n, h)
        o = oracle.Oracle(n, n, h, mask, shapes, t, wlmod.SYM_DX2Y2, nphi, crystal_rotation=rot_crystal)
        delta = np.full((n, n), D0) * mask
        Ax = np.full((n, n), Avec[0]); Ay = np.full((n, n), Avec[1])
        z, w = o.matsubara(ne)
        st = o.reset_stores(delta, Ax, Ay, z)
        for _ in range(2):
            st = o.raw_sweep(delta, Ax, Ay, z, w, st)["stores"]
        per_angle = [o.raw_sweep(delta, Ax, Ay, z, w, st, angle_list=[k], dbg_angle=k)["dbg"] for k in range(nphi)]
        full = o.sweep(delta, Ax, Ay, ne, st)
        res[name] = dict(o=o, dbg=per_angle, full=full, n=n)
    assert res["A"]["o"].nrot == res["B"]["o"].nrot and res["A"]["o"].n_gather_fallback == res["B"]["o"].n_gather_fallback
    sh = nphi // 8
    worst = 0.0
    for k in range(nphi):
        a, b = res["A"]["dbg"][k], res["B"]["dbg"][(k - sh) % nphi]
        for key in ("SF", "SG", "SI", "SR"):
            worst = max(worst, float(np.max(np.abs(a[key] - b[key]))))
        assert np.count_nonzero(a["SR"]) == np.count_nonzero(b["SR"]) > 100
    assert worst < 1e-12
    ca, cb = res["A"]["n"] // 2, res["B"]["n"] // 2                        # the origin is a grid point of both grids
    fa, fb = res["A"]["full"], res["B"]["full"]
    assert abs(fa["delta_new"][ca, ca] - fb["delta_new"][cb, cb]) < 1e-13
    ja = np.array([fa["jx"][ca, ca], fa["jy"][ca, ca]]); jb = np.array([fb["jx"][cb, cb], fb["jy"][cb, cb]])
    assert np.max(np.abs(np.array([c8 * ja[0] + s8 * ja[1], -s8 * ja[0] + c8 * ja[1]]) - jb)) < 1e-13 and np.linalg.norm(ja) > 1e-3
    # [110] walls are pair breaking, [100] walls are not: the gap at the wall is suppressed in A / B and not in a [100] square
    assert abs(fa["delta_new"][ca, ca + int(0.9 * L / math.sqrt(2) / h)]) < 0.8 * abs(fa["delta_new"][ca, ca])
