"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these re-types an oracle formula: each compares an oracle routine with an independent
statement — an adaptive ODE solve of the Riccati equation itself, a closed form, an invariant, a
numerical quadrature of the defining integral, or a brute-force ray-tracing path.
"""
import math
import os

import numpy as np
import pytest
from scipy.integrate import dblquad, solve_ivp

import oracle
import workloads as wlmod
from workloads import Shape, make_mask, square

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "constants.txt")) as f:
    for line in f:
        if line.strip() and not line.startswith("#"):
            k, v = line.split()[:2]
            GOLD[k] = float(v)


def riccati_rhs(De, z):
    # PAPER.md C1-C2 (:972-974), v_F = 1: d gamma/ds = i[conj(De) gamma^2 + 2 z gamma + De]
    def f(s, y):
        g = y[0] + 1j * y[1]
        d = 1j * (np.conj(De) * g * g + 2 * z * g + De)
        return [d.real, d.imag]
    return f


def ode(De, z, g0, l):
    r = solve_ivp(riccati_rhs(De, z), [0, l], [g0.real, g0.imag], method="DOP853", rtol=1e-13, atol=1e-15)
    return r.y[0, -1] + 1j * r.y[1, -1]


# ---- P1: one step vs an adaptive integration of the same constant-coefficient ODE -----------------
@pytest.mark.parametrize("De,z,g0,l", [
    (0.3 + 0.1j, 0.25j + 0.04, 0.2 - 0.3j, 0.1),
    (0.25 + 0j, 12.7j - 0.1, -0.01 + 0.02j, 0.05),
    (0.0 + 0j, 0.5j + 0.2, 0.3 + 0.3j, 0.1),            # Delta = 0 (vortex core)
    (0.34 - 0.02j, 0.3 + 0.003j, 0.1 + 0.6j, 0.05),      # retarded, inside the gap
    (0.2 + 0.1j, -0.6 + 0.002j, -0.4 + 0.1j, 0.08),      # retarded, outside the gap, negative energy
    (-0.3 + 0.2j, 0.025j + 0.3, 0.5j, 0.031),            # Doppler shift larger than eps_0 and |Delta|~a
])
def test_P1_closed_form_step_vs_ode(De, z, g0, l):
    ref = ode(De, z, g0, l)
    got = oracle.step(g0, De, z, l, stepper=0)
    assert abs(got - ref) < 1e-12
    mid = oracle.step(g0, De, z, l, stepper=1)
    assert abs(mid - ref) < 40 * l ** 3 * (abs(z) + abs(De) + 1) ** 3   # one step of a 2nd-order rule


def test_P1_tilde_equation_is_the_gamma_equation_backwards():
    # Eq. 26 (:172): d gt/ds = i[D gt^2 - 2 z gt + conj(D)] integrated from s=l down to 0
    D, z, gt1, l = 0.3 - 0.2j, 0.4j + 0.07, 0.1 + 0.2j, 0.1
    r = solve_ivp(lambda s, y: (lambda g: [(1j * (D * g * g - 2 * z * g + np.conj(D))).real,
                                           (1j * (D * g * g - 2 * z * g + np.conj(D))).imag])(y[0] + 1j * y[1]),
                  [l, 0], [gt1.real, gt1.imag], method="DOP853", rtol=1e-13, atol=1e-15)
    ref = r.y[0, -1] + 1j * r.y[1, -1]
    _, _, _, gt_end = oracle.march([l], [D], [0.0], z, 0j, gt1)
    assert abs(gt_end - ref) < 1e-12


# ---- P2: homogeneous bulk (north_star's bulk check, convention-free form) --------------------------
@pytest.mark.parametrize("eps", [0.05, 0.25, 3.0, 25.0])
def test_P2_bulk_fixed_point(eps):
    D = 0.28 * np.exp(0.7j)
    z = 1j * eps
    gh = oracle.gamma_h(D, z)
    Lam = math.sqrt(eps ** 2 + abs(D) ** 2)
    assert abs(abs(gh) - abs(D) / (eps + Lam)) < 1e-15               # |gamma| = |Delta|/(eps_n + Lambda_n)
    for l in (0.01, 0.1, 1.0):
        assert abs(oracle.step(gh, D, z, l) - gh) < 1e-15            # fixed point of the step
        assert abs(oracle.step(gh, D, z, l, 1) - gh) < 1e-15
    gth = oracle.gamma_h(-np.conj(D), z)
    P = gh * gth
    assert abs((1 - P) / (1 + P) - eps / Lam) < 1e-14                # g_n = eps_n / Lambda_n
    assert abs(-2j * gh / (1 + P) - D / Lam) < 1e-14                 # f / pi = Delta / Lambda_n


# ---- P3: exact discrete pin — uniform gap in an axis-aligned square -------------------------------
@pytest.mark.parametrize("sym,nphi", [(wlmod.SYM_S, 16), (wlmod.SYM_DX2Y2, 16), (wlmod.SYM_S, 12), (wlmod.SYM_DX2Y2, 6)])
def test_P3_uniform_gap_closed_form(sym, nphi):
    n, h, t, ne, D0 = 20, 0.1, 0.5, 16, 0.22 * np.exp(0.3j)
    shapes = [square(n * h)]
    mask = make_mask(shapes, n, n, h)
    o = oracle.Oracle(n, n, h, mask, shapes, t, sym, nphi)
    assert o.n_gather_fallback == 0
    delta = np.full((n, n), D0)
    r = o.sweep(delta, None, None, ne)
    eps = t * (np.arange(ne) + 0.5)
    acc = 0.0
    for k in range(nphi):
        _, eta, W = o.angle_info(k)
        acc += W * eta ** 2 * t * np.sum(1.0 / np.sqrt(eps ** 2 + abs(D0) ** 2 * eta ** 2))
    expect = D0 * acc / oracle.matsubara_denominator(t, ne)
    assert np.max(np.abs(r["delta_new"] - expect)) < 1e-13
    assert np.max(np.abs(r["jx"])) < 1e-14 and np.max(np.abs(r["jy"])) < 1e-14
    assert r["stats"]["n_bad"] == 0


def _bulk_gap(sym, t, ne, nphi, D0=0.25):
    """Fixed point of the oracle's own sweep on a 2x2 uniform grain (Steffensen-accelerated)."""
    n, h = 2, 0.1
    shapes = [square(n * h)]
    mask = make_mask(shapes, n, n, h)
    o = oracle.Oracle(n, n, h, mask, shapes, t, sym, nphi)
    F = lambda d: float(o.sweep(np.full((n, n), d + 0j), None, None, ne)["delta_new"][0, 0].real)
    d = D0
    for _ in range(30):
        d1 = F(d); d2 = F(d1)
        den = d2 - 2 * d1 + d
        dn = d2 if abs(den) < 1e-15 else d - (d1 - d) ** 2 / den
        if abs(dn - d) < 1e-13:
            d = dn
            break
        d = dn
    return d


# ---- P4: weak-coupling BCS gap from the gap equation ----------------------------------------------
def test_P4_bcs_gap_swave():
    d = _bulk_gap(wlmod.SYM_S, 0.02, 4000, 4)
    assert abs(2 * math.pi * d - GOLD["bcs_ratio_swave"]) < 2e-5


def test_P4_bcs_gap_dwave():
    d = _bulk_gap(wlmod.SYM_DX2Y2, 0.02, 2000, 64)
    assert abs(2 * math.pi * math.sqrt(2) * d - GOLD["bcs_ratio_dwave_max"]) < 1e-3


# ---- P5: the literal bulk gaps the workloads use as initial amplitudes ----------------------------
@pytest.mark.parametrize("key,sym,nphi", [(("s", 0.5, 16), wlmod.SYM_S, 4), (("s", 0.1, 128), wlmod.SYM_S, 4),
                                          (("s", 0.05, 512), wlmod.SYM_S, 4), (("d", 0.1, 256), wlmod.SYM_DX2Y2, 64)])
def test_P5_workload_bulk_gaps(key, sym, nphi):
    d = _bulk_gap(sym, key[1], key[2], nphi)
    assert abs(d - wlmod.BULK_GAP[key]) < 1e-6


# ---- P6: Doppler shift (exact nonlinear with bc_mode=1) and linear response (Eq. 33-34) -----------
def test_P6_doppler_current_exact_and_linear_response():
    n, h, t, ne, nphi, D0, sig = 12, 0.1, 0.3, 24, 16, 0.25, -1
    shapes = [square(n * h)]
    mask = make_mask(shapes, n, n, h)
    o = oracle.Oracle(n, n, h, mask, shapes, t, wlmod.SYM_S, nphi, bc_mode=1, charge_sign=sig)
    eps = t * (np.arange(ne) + 0.5)
    for A0 in ((0.11, -0.07), (1e-4, 0.0)):
        Ax = np.full((n, n), A0[0]); Ay = np.full((n, n), A0[1])
        r = o.sweep(np.full((n, n), D0 + 0j), Ax, Ay, ne)
        jx = jy = 0.0
        for k in range(nphi):
            v, _, W = o.angle_info(k)
            z = 1j * eps + sig * (v[0] * A0[0] + v[1] * A0[1])
            Om = np.sqrt(D0 ** 2 - z * z)
            s = np.sum((-1j * z / Om).imag)
            jx += 2 * sig * t * W * v[0] * s; jy += 2 * sig * t * W * v[1] * s
        assert np.max(np.abs(r["jx"] - jx)) < 1e-13 and np.max(np.abs(r["jy"] - jy)) < 1e-13
    # linear response: j = sigma_e Y p_s, p_s = -sigma_e A, Y = t sum |D|^2 / Lambda^3  (Eq. 34 :502)
    Y = t * np.sum(D0 ** 2 / (eps ** 2 + D0 ** 2) ** 1.5)
    assert abs(r["jx"][5, 5] - (-Y * 1e-4)) < 1e-4 * Y * 1e-4 + 1e-10
    assert abs(r["jy"][5, 5]) < 1e-14


# ---- P7: vector-potential kernel: closed form D3-D6 vs quadrature of D2; discrete London equation -
@pytest.mark.parametrize("m,n,h", [(0, 0, 0.05), (1, 0, 0.05), (0, 1, 0.05), (3, 2, 0.1), (7, 0, 0.2), (2, 9, 0.05)])
def test_P7_G_closed_form_vs_quadrature(m, n, h):
    f = lambda yp, xp: np.log((xp + h * m) ** 2 + (yp + h * n) ** 2) / (4 * math.pi)
    if m == 0 and n == 0:   # integrable log singularity at the origin: use the 4-fold symmetry
        ref = 4 * dblquad(f, 0, h / 2, 0, h / 2, epsabs=1e-14, epsrel=1e-12)[0]
    else:
        ref = dblquad(f, -h / 2, h / 2, -h / 2, h / 2, epsabs=1e-15, epsrel=1e-13)[0]
    assert abs(oracle.G_table_entry(m, n, h) - ref) < 1e-10 * max(1.0, abs(ref) / 1e-3) * 1e-2 + 1e-12


def test_P7_vector_potential_solves_discrete_london():
    # laplace(A_ind) = -(j - <j>)/kappa^2 (Eq. 45 :602 with our units; App. D :1007)
    n, h, kappa = 40, 0.1, 2.0
    mask = np.ones((n, n), np.uint8)
    X, Y = wlmod.grid_xy(n, n, h)
    jx = -Y * np.exp(-(X ** 2 + Y ** 2)); jy = X * np.exp(-(X ** 2 + Y ** 2))   # zero-mean circulating current
    Ax, Ay = oracle.vector_potential(mask, h, kappa, jx, jy)
    lap = (Ax[1:-1, 2:] + Ax[1:-1, :-2] + Ax[2:, 1:-1] + Ax[:-2, 1:-1] - 4 * Ax[1:-1, 1:-1]) / h ** 2
    rhs = -(jx - jx.mean())[1:-1, 1:-1] / kappa ** 2
    assert np.max(np.abs(lap - rhs)) < 0.02 * np.max(np.abs(rhs))
    assert np.max(np.abs(Ax)) > 1e-3    # not trivially zero


# ---- P8: bulk free energy, Eq. 38 (:525-533) ------------------------------------------------------
def test_P8_bulk_free_energy():
    n, h, ne, nphi = 4, 0.1, 64, 16
    shapes = [square(n * h)]
    mask = make_mask(shapes, n, n, h)
    for sym, t, D0 in ((wlmod.SYM_S, 0.3, 0.26), (wlmod.SYM_DX2Y2, 0.2, 0.2)):
        o = oracle.Oracle(n, n, h, mask, shapes, t, sym, nphi)
        delta = np.full((n, n), D0 + 0j)
        r = o.sweep(delta, None, None, ne)
        om = o.free_energy_density(delta, ne, r["fe_I"])
        eps = t * (np.arange(ne) + 0.5)
        ref = 0.0
        for k in range(nphi):
            _, eta, W = o.angle_info(k)
            d2 = (D0 * eta) ** 2
            Lam = np.sqrt(eps ** 2 + d2)
            ref += W * (d2 * math.log(t) + t * np.sum(d2 ** 2 / (eps * (Lam + eps) ** 2)))
        assert np.max(np.abs(om - ref)) < 1e-13


def test_P8_condensation_energy_T0():
    t, ne = 0.02, 4000
    d = _bulk_gap(wlmod.SYM_S, t, ne, 4)
    n, h = 2, 0.1
    shapes = [square(n * h)]
    o = oracle.Oracle(n, n, h, make_mask(shapes, n, n, h), shapes, t, wlmod.SYM_S, 4)
    delta = np.full((n, n), d + 0j)
    om = o.free_energy_density(delta, ne, o.sweep(delta, None, None, ne)["fe_I"])
    assert abs(om[0, 0] - GOLD["omega_bulk_T0"]) < 1e-4


# ---- P9: convergence order through a smooth inhomogeneous profile ---------------------------------
def test_P9_second_order_convergence_both_steppers():
    z = 0.15j + 0.0
    Dfun = lambda s: 0.28 * np.tanh(s) * np.exp(0.4j * np.sin(s))     # vortex-like: amplitude zero, phase varies
    afun = lambda s: 0.05 * np.cos(0.7 * s)
    s0, s1 = -4.0, 4.0
    g0 = oracle.gamma_h(Dfun(s0), z + afun(s0))
    rhs = lambda s, y: (lambda g: [(1j * (np.conj(Dfun(s)) * g * g + 2 * (z + afun(s)) * g + Dfun(s))).real,
                                   (1j * (np.conj(Dfun(s)) * g * g + 2 * (z + afun(s)) * g + Dfun(s))).imag])(y[0] + 1j * y[1])
    ref = solve_ivp(rhs, [s0, s1], [g0.real, g0.imag], method="DOP853", rtol=1e-12, atol=1e-14)
    ref = ref.y[0, -1] + 1j * ref.y[1, -1]
    errs = {0: [], 1: []}
    for N in (80, 160, 320):
        h = (s1 - s0) / N
        nodes = s0 + h * np.arange(N + 1)
        Dn = Dfun(nodes); an = afun(nodes)
        De = 0.5 * (Dn[:-1] + Dn[1:]); a = 0.5 * (an[:-1] + an[1:])
        for st in (0, 1):
            _, _, ge, _ = oracle.march(np.full(N, h), De, a, z, g0, 0j, stepper=st)
            errs[st].append(abs(ge - ref))
    for st in (0, 1):
        assert 3.5 < errs[st][0] / errs[st][1] < 4.5 and 3.5 < errs[st][1] / errs[st][2] < 4.5


# ---- P10: Andreev bound state at a sign-changing (unfolded [110]) reflection ----------------------
def test_P10_abs_kink_exact():
    Deta, M, h = 0.24 * math.sqrt(2) * math.cos(2 * 0.3), 400, 0.05
    De = np.array([Deta] * M + [-Deta] * M, dtype=complex)
    lengths = np.full(2 * M, h); a = np.zeros(2 * M)
    for z in (0.05j, 0.7j, 0.0 + 0.0024j, 0.1 + 0.0024j, -0.2 + 0.001j):
        gs = oracle.gamma_h(Deta, z)                      # gamma_h(+) at the left end
        gts = oracle.gamma_h(-np.conj(-Deta + 0j), z)     # gamma-tilde_h(-) at the right end
        G, GT, _, _ = oracle.march(lengths, De, a, z, gs, gts)
        P = G[M - 1] * GT[M - 1]                          # node at the kink
        g = (1 - P) / (1 + P)
        Om = np.sqrt(Deta ** 2 - z * z + 0j)
        assert abs(g - 1j * Om / z) < 1e-12 * abs(g)      # g_n = i Omega / z = 1 / g_bulk exactly
    # zero-energy peak height |Delta eta| / delta, absent in the bulk
    delta = 0.0024
    z = 0.0 + 1j * delta
    G, GT, _, _ = oracle.march(lengths, De, a, z, oracle.gamma_h(Deta, z), oracle.gamma_h(Deta + 0j, z))
    P = G[M - 1] * GT[M - 1]
    assert abs(((1 - P) / (1 + P)).real - abs(Deta) / delta) < 1e-4 * abs(Deta) / delta   # height |D eta|/delta up to O(delta^2/D^2)
    P0 = G[5] * GT[5]                                   # 20 xi0 away: bound-state tail e^{-2 Omega s} is gone
    assert ((1 - P0) / (1 + P0)).real < 0.05


# ---- P12: invariants of a full sweep on a noisy field with a vector potential ----------------------
@pytest.fixture(scope="module")
def noisy_disc():
    rng = np.random.default_rng(7)
    R, h = 1.5, 0.1
    n = 30
    shapes = [wlmod.disc(R)]
    mask = make_mask(shapes, n, n, h)
    X, Y = wlmod.grid_xy(n, n, h)
    delta = 0.25 * (1 + 0.2 * rng.uniform(-1, 1, (n, n))) * np.exp(1j * (0.5 * rng.uniform(-1, 1, (n, n)) - np.arctan2(Y - 0.13, X + 0.21)))
    Ax = -0.05 * Y; Ay = 0.05 * X
    return dict(n=n, h=h, shapes=shapes, mask=mask, delta=delta * mask, Ax=Ax, Ay=Ay, X=X, Y=Y)


def test_P12_tilde_symmetry_eq13(noisy_disc):
    d = noisy_disc
    nphi, ne, t = 8, 5, 0.3
    o = oracle.Oracle(d["n"], d["n"], d["h"], d["mask"], d["shapes"], t, wlmod.SYM_DX2Y2, nphi)
    z, w = o.matsubara(ne)
    st = o.reset_stores(d["delta"], d["Ax"], d["Ay"], z)
    for _ in range(3):
        r = o.raw_sweep(d["delta"], d["Ax"], d["Ay"], z, w, st)
        st = r["stores"]
    g, gt = st
    for k in range(nphi // 2):
        k2 = k + nphi // 2
        n1, n2 = o.ntraj_angle(k), o.ntraj_angle(k2)
        assert n1 == n2
        a = gt[o.traj_offset(k):o.traj_offset(k) + n1]
        b = g[o.traj_offset(k2):o.traj_offset(k2) + n2][::-1]      # lattices coincide under (j,t)->(-j,-t)
        assert np.max(np.abs(a - np.conj(b))) < 1e-13               # x~(p,e) = x(-p,-e*)*  (Eq. 13 :95)
    assert r["stats"]["min_one_minus_abs_gamma"] > 0                # |gamma|, |gamma~| < 1
    assert np.all(r["R"][d["mask"] > 0] > 0)                        # Re g_n(Matsubara) > 0


def test_P12_global_phase_covariance(noisy_disc):
    d = noisy_disc
    o = oracle.Oracle(d["n"], d["n"], d["h"], d["mask"], d["shapes"], 0.3, wlmod.SYM_S, 8)
    r0 = o.sweep(d["delta"], d["Ax"], d["Ay"], 6)
    ph = np.exp(0.9j)
    r1 = o.sweep(d["delta"] * ph, d["Ax"], d["Ay"], 6)
    assert np.max(np.abs(r1["delta_new"] - ph * r0["delta_new"])) < 1e-14
    assert np.max(np.abs(r1["jx"] - r0["jx"])) < 1e-15 and np.max(np.abs(r1["fe_I"] - r0["fe_I"])) < 1e-15


def test_P12_local_gauge_covariance_second_order():
    # Delta -> Delta e^{i theta(R)}, A -> A + sigma_e grad(theta)/2 (Eq. 2 :41, Eq. 31 :479) leaves |Delta_new| and j
    # invariant.  Piecewise-constant coefficients are not gauge covariant, so this holds to O(h^2) in the interior
    # (at the wall the angle interpolation of the specular gather adds O(dphi^2)); boundary values converged first.
    errs = []
    for n, h in ((20, 0.2), (40, 0.1)):
        shapes = [wlmod.disc(1.9)]
        mask = make_mask(shapes, n, n, h)
        X, Y = wlmod.grid_xy(n, n, h)
        o = oracle.Oracle(n, n, h, mask, shapes, 0.4, wlmod.SYM_S, 16, charge_sign=-1)
        delta = 0.25 * (1 - 0.3 * np.exp(-(X ** 2 + Y ** 2))) * mask
        Ax = -0.08 * Y; Ay = 0.08 * X
        theta = 0.3 * X + 0.2 * X * Y

        def converged(d, ax, ay):
            st = None
            for _ in range(16):
                r = o.sweep(d, ax, ay, 6, st); st = r["stores"]
            return r
        r0 = converged(delta, Ax, Ay)
        r1 = converged(delta * np.exp(1j * theta), Ax + (-1) * 0.5 * (0.3 + 0.2 * Y), Ay + (-1) * 0.5 * (0.2 * X))
        m = (mask > 0) & (np.hypot(X, Y) < 1.2)
        errs.append(max(np.max(np.abs(np.abs(r1["delta_new"]) - np.abs(r0["delta_new"]))[m]),
                        np.max(np.abs(r1["jx"] - r0["jx"])[m])))
        assert np.max(np.abs(r0["jx"])) > 0.05
    assert errs[1] < errs[0] / 2.5 and errs[1] < 4e-4


def test_P12_current_sign_is_diamagnetic(noisy_disc):
    # Meissner response: j = -Y A for uniform Delta (London, Eq. 45 :602): j antiparallel to A
    d = noisy_disc
    o = oracle.Oracle(d["n"], d["n"], d["h"], d["mask"], d["shapes"], 0.3, wlmod.SYM_S, 16)
    r = o.sweep(0.25 * d["mask"] + 0j, d["Ax"], d["Ay"], 12)
    c = d["n"] // 2
    i, j = c + 4, c + 2
    assert r["jx"][j, i] * d["Ax"][j, i] + r["jy"][j, i] * d["Ay"][j, i] < 0


# ---- P13: brute force — trace each start value back through the grain instead of using stores -----
def test_P13_brute_force_ray_tracing_equals_store_based_sweeps():
    m, h, nphi, t = 8, 0.1, 8, 0.4
    L = math.sqrt(2) * h * m          # L/(sqrt(2) h) integer: 45-degree reflections land on lattice lines
    n = 10                            # even: no lattice line passes exactly through a corner
    shapes = [square(L)]
    mask = make_mask(shapes, n, n, h)
    assert mask.all()
    rng = np.random.default_rng(3)
    delta = 0.25 * (1 + 0.4 * rng.uniform(-1, 1, (n, n))) * np.exp(1j * rng.uniform(-1, 1, (n, n)))
    Ax = 0.1 * rng.uniform(-1, 1, (n, n)); Ay = 0.1 * rng.uniform(-1, 1, (n, n))
    o = oracle.Oracle(n, n, h, mask, shapes, t, wlmod.SYM_DX2Y2, nphi)
    assert o.n_gather_fallback == 0
    z = np.array([0.2j, 0.35 + 0.01j, 1.0j]); w = np.ones(3)
    B = 3
    st = o.reset_stores(delta, Ax, Ay, z)
    init = st
    for _ in range(B):
        st = o.raw_sweep(delta, Ax, Ay, z, w, st)["stores"]
    tabs = [o.tables(k) for k in range(nphi)]
    vs = [o.angle_info(k)[0] for k in range(nphi)]
    c = 0.5 * (o.nrot - 1)

    def endpoint(k, i, which):
        T = tabs[k]; u = T["u_out"][i] if which == "out" else T["u_in"][i]
        wv = (T["t"][i] - c) * h
        return np.array([u * vs[k][0] - wv * vs[k][1], u * vs[k][1] + wv * vs[k][0]])

    def normal(k, i, which):
        return tabs[k]["n_out"][i] if which == "out" else tabs[k]["n_in"][i]

    def find(pt, direction, which):
        """the unique trajectory with direction `direction` whose `which` end is the point pt"""
        ang = math.atan2(direction[1], direction[0]) / (2 * math.pi / nphi)
        k = int(round(ang)) % nphi
        assert abs(ang - round(ang)) < 1e-9
        for i in range(len(tabs[k]["t"])):
            if np.linalg.norm(endpoint(k, i, which) - pt) < 1e-9:
                return k, i
        raise AssertionError("reflection not on the lattice")

    def pieces(k, i):
        Dn, an = o.debug_nodes(delta, Ax, Ay, k, i)
        T = tabs[k]
        uf = (T["jf"][i] - c) * h; ul = (T["jl"][i] - c) * h
        ln = np.concatenate([[uf - T["u_in"][i]], np.full(len(Dn) - 1, h), [T["u_out"][i] - ul]])
        De = np.concatenate([[Dn[0]], 0.5 * (Dn[:-1] + Dn[1:]), [Dn[-1]]])
        a = np.concatenate([[an[0]], 0.5 * (an[:-1] + an[1:]), [an[-1]]])
        return ln, De, a

    def gamma_end(k, i, e, depth):
        """gamma at the exit of trajectory (k,i) after `depth` Jacobi sweeps"""
        if depth == 0:
            return init[0][o.traj_offset(k) + i, e]
        nrm = normal(k, i, "in"); v = vs[k]
        vin = v - 2 * np.dot(v, nrm) * nrm
        kp, ip = find(endpoint(k, i, "in"), vin, "out")
        ln, De, a = pieces(k, i)
        return oracle.march(ln, De, a, complex(z[e]), gamma_end(kp, ip, e, depth - 1), 0j)[2]

    def gammat_end(k, i, e, depth):
        if depth == 0:
            return init[1][o.traj_offset(k) + i, e]
        nrm = normal(k, i, "out"); v = vs[k]
        vout = v - 2 * np.dot(v, nrm) * nrm
        kp, ip = find(endpoint(k, i, "out"), vout, "in")
        ln, De, a = pieces(k, i)
        return oracle.march(ln, De, a, complex(z[e]), 0j, gammat_end(kp, ip, e, depth - 1))[3]

    worst = 0.0
    for k in range(nphi):
        for i in range(0, len(tabs[k]["t"]), 3):
            for e in range(3):
                worst = max(worst, abs(gamma_end(k, i, e, B) - st[0][o.traj_offset(k) + i, e]),
                            abs(gammat_end(k, i, e, B) - st[1][o.traj_offset(k) + i, e]))
    assert worst < 1e-12


# ---- geometry sanity: node count = area / h^2, no fallbacks, on the shapes of the five configs -----
@pytest.mark.parametrize("cfg,kw", [(0, {}), (1, dict(pts_per_xi=5, n_angles=16)), (2, dict(pts_per_xi=4, n_angles=16, size_scale=0.5))])
def test_geometry_tables(cfg, kw):
    wl = wlmod.make_workload(cfg, **kw)
    o = oracle.Oracle.from_workload(wl)
    assert o.n_gather_fallback == 0
    for k in range(0, wl.n_angles, 3):
        T = o.tables(k)
        nodes = int(np.sum(T["jl"] - T["jf"] + 1))
        assert abs(nodes * wl.h ** 2 - wl.area()) < 0.03 * wl.area()
        assert np.all(T["u_out"] > T["u_in"])
        assert np.all(np.abs(np.sum(T["g_w"], axis=2) - 1.0) < 1e-12)


def test_abs_peak_at_110_wall_in_closed_grain():
    """north_star's ABS check: zero-energy peak at pair-breaking [110] d-wave edges, absent in the bulk."""
    wl = wlmod.make_workload(3, pts_per_xi=5, n_angles=32, size_scale=0.5, n_energies=3)
    o = oracle.Oracle.from_workload(wl)
    ld = o.ldos(wl.delta0, None, None, [0.0], 0.02 * wl.bulk_gap, 6)[0]
    c = wl.nx // 2
    # wall point: midway along the upper-right [110] wall, one cell inside; bulk: the centre
    d = 0.5 * 10.0 / math.sqrt(2) / math.sqrt(2)
    i = int(round(c + (d - 0.15) / wl.h)); j = i
    assert wl.mask[j, i]
    assert ld[j, i] > 5.0 * ld[c, c] and ld[c, c] < 1.0
    assert np.all(ld[wl.mask > 0] > 0)


# ---- accelerators of App. E on fixed-point problems with known answers ---------------------------------
def _run_linear(acc, lam, x0, xstar, n):
    """iterate x <- x + acc.update(g(x) - x) for the linear map g(x) = x - lam (x - x*) (lam: per-element)."""
    x = np.array(x0, float)
    hist = [x.copy()]
    for _ in range(n):
        x = x + acc.update(-lam * (x - xstar))
        hist.append(x.copy())
    return np.array(hist)


def test_accelerator_picard_geometric_rate():
    # E5 (:1070): e_n = (1 - alpha lam)^n e_0
    lam, xs = np.array([0.3, 0.9, 1.4]), np.array([1.0, -2.0, 0.5])
    h = _run_linear(oracle.Accelerator(0, step=0.8), lam, [0, 0, 0], xs, 7)
    assert np.allclose(h[7] - xs, (1 - 0.8 * lam) ** 7 * (0 - xs), rtol=1e-12, atol=1e-14)


def test_accelerator_bb_is_the_secant_step_on_an_isotropic_problem():
    # E8-E11 (:1107-1115): for g(x) = x - lam (x - x*) with one scalar lam, d_i - d_{i-1} = -lam alpha_i d_{i-1},
    # so s^BB1 = s^BB2 = 1/(lam alpha_i) and alpha_{i+1} = 1/lam: the second update lands on x* exactly
    xs = np.array([1.0, -2.0, 0.5, 3.0])
    acc = oracle.Accelerator(1, step=1.0)
    h = _run_linear(acc, 0.37, [0.2, 0.1, -1.0, 4.0], xs, 2)
    assert abs(acc.alpha - 1 / 0.37) < 1e-12
    assert np.max(np.abs(h[2] - xs)) < 1e-13
    # the step size is clipped to [1e-3, 100] (Listing 15 :1121-1127)
    acc = oracle.Accelerator(1, step=1.0)
    _run_linear(acc, 1e-4, [0.2, 0.1], xs[:2], 2)
    assert acc.alpha == 100.0


def test_accelerator_polyak_two_term_recurrence():
    # E6-E7 (:1087-1089) with v_0 = 0 on a scalar linear problem: eliminating v gives
    # e_{n+1} = (2 - beta - alpha lam) e_n - (1 - beta) e_{n-1},  e_1 = (1 - alpha lam) e_0
    al, be, lam = 2.0, 0.5, 0.21
    h = _run_linear(oracle.Accelerator(2, step=al, drag=be), lam, [1.0], np.array([0.0]), 12)[:, 0]
    e = [1.0, 1.0 - al * lam]
    for n in range(1, 12):
        e.append((2 - be - al * lam) * e[n] - (1 - be) * e[n - 1])
    assert np.allclose(h, e, rtol=1e-12, atol=1e-15)
    # closed form through the roots of r^2 - (2 - beta - alpha lam) r + (1 - beta) = 0
    r = np.roots([1.0, -(2 - be - al * lam), 1 - be])
    c = np.linalg.solve(np.array([[1, 1], [r[0], r[1]]]), np.array([e[0], e[1]], complex))
    assert abs((c[0] * r[0] ** 12 + c[1] * r[1] ** 12).real - h[12]) < 1e-12
    # drag = 1 forgets the velocity: Picard
    hp = _run_linear(oracle.Accelerator(2, step=0.7, drag=1.0), lam, [1.0], np.array([0.0]), 5)[:, 0]
    assert np.allclose(hp, (1 - 0.7 * lam) ** np.arange(6), rtol=1e-13)


def test_accelerator_congacc_step_growth_and_clip():
    # E12-E16 (:1134-1146) with a CONSTANT difference d (cos = 1 from the second iteration on, 0 at the first where
    # m = 0): alpha_1 = alpha_0, alpha_{i+1} = alpha_i k, m = d  =>  x_n = x_0 + d alpha_0 (1 + k + ... + k^{n-1})
    d = np.array([0.3, -0.2, 0.0, 1.0, 0.5, 0.5, -1.0, 2.0])
    acc = oracle.Accelerator(3, step=0.5, step_factor=1.234, ncomp=4)
    x = np.zeros(8)
    for _ in range(6):
        x = x + acc.update(d)
    assert np.allclose(x, d * 0.5 * sum(1.234 ** i for i in range(6)), rtol=1e-13)
    assert np.allclose(acc.alpha_c, 0.5 * 1.234 ** 5, rtol=1e-13) and acc.w_c == [0.0] * 4
    for _ in range(40):
        acc.update(d)
    assert acc.alpha_c == [100.0] * 4                      # step_size_max (Listing 16 :1157)
    # opposite direction: cos = -1, alpha shrinks by k per iteration (E13), down to step_size_min
    acc = oracle.Accelerator(3, step=0.5, ncomp=1)
    acc.update(np.array([1.0, 0.0])); a1 = acc.alpha_c[0]
    acc.update(np.array([-1.0, 0.0]))
    assert abs(acc.alpha_c[0] - a1 / 1.234) < 1e-15


def test_accelerator_congacc_weight_solves_E17():
    # E14, E17 (:1138-1149): m = (1,0), d = (0,1): cos(w m + (1-w) d, d) = (1-w)/sqrt(w^2 + (1-w)^2) = s_min
    # => w* = 1/(1 + s_min/sqrt(1 - s_min^2))
    for smin in (0.7, 0.3, 0.95):
        acc = oracle.Accelerator(3, step=0.5, cos_min=smin, ncomp=1)
        acc.update(np.array([1.0, 0.0]))                    # m_1 = d_0 = (1, 0), w_1 = 0
        upd = acc.update(np.array([0.0, 1.0]))              # cos(m, d) = 0 < s_min -> w* from E17
        wstar = 1.0 / (1.0 + smin / math.sqrt(1.0 - smin * smin))
        assert abs(acc.w_c[0] - wstar) < 1e-14
        m = np.array([wstar, 1.0 - wstar])
        assert abs(m[1] / np.linalg.norm(m) - smin) < 1e-14     # the mixed direction has exactly the tolerated similarity
        assert np.allclose(upd, acc.alpha_c[0] * m, rtol=1e-13)
        assert abs(acc.alpha_c[0] - 0.5) < 1e-15            # k^0: cos(m, d) = 0 leaves the step size
    # components are treated independently (E12 "component index c")
    acc = oracle.Accelerator(3, step=0.5, ncomp=2)
    acc.update(np.array([1.0, 0.0, 1.0, 0.0]))
    acc.update(np.array([1.0, 0.0, 0.0, 1.0]))
    assert acc.w_c[0] == 0.0 and acc.w_c[1] > 0.4 and abs(acc.alpha_c[0] - 0.5 * 1.234) < 1e-15


# ---- several order-parameter components (Eq. 1 :37, Eq. 20-22 :135-144, Listing 11 :909-926) --------------------
@pytest.mark.parametrize("Ds,Dd,tc_s", [(0.05, 0.20, 0.6), (0.05j, 0.20, 0.6), (0.18 * np.exp(0.4j), 0.07 * np.exp(-1.1j), 1.0)])
def test_two_component_uniform_gap_closed_form(Ds, Dd, tc_s):
    """Uniform Delta_s + Delta_d eta_d in an axis-aligned square ([100] walls: eta_s and eta_{dx2-y2} are both invariant
    under the specular reflections, so every start value stays the homogeneous solution): f/pi = Delta(phi)/Lambda_n(phi)
    with Delta(phi) = Delta_s + Delta_d sqrt2 cos 2phi, hence Delta_new,G = t sum_n <eta_G Delta/Lambda_n> / (ln(T/T_c^G)
    + sum 1/(n+1/2)) exactly on the discrete angle set — pins the sum over components at the nodes, the projection
    on each eta_G and each component's own T_c in the denominator.  d + s, d + is, and a general relative phase."""
    n, h, t, ne, nphi = 12, 0.1, 0.3, 24, 32
    shapes = [square(n * h)]
    mask = make_mask(shapes, n, n, h)
    tc = [tc_s, 1.0] if tc_s < 1.0 else [1.0, 0.5]
    o = oracle.Oracle(n, n, h, mask, shapes, t, 0, nphi)
    o.set_components([0, 1], tc)
    delta = np.stack([np.full((n, n), Ds, complex), np.full((n, n), Dd, complex)])
    r = o.sweep(delta, None, None, ne)
    eps = t * (np.arange(ne) + 0.5)
    num = np.zeros(2, complex)
    for k in range(nphi):
        phi = 2 * np.pi * k / nphi
        W = o.angle_info(k)[2]
        eta = np.array([1.0, np.sqrt(2.0) * np.cos(2 * phi)])
        Dphi = Ds * eta[0] + Dd * eta[1]
        num += W * eta * Dphi * t * np.sum(1.0 / np.sqrt(eps ** 2 + abs(Dphi) ** 2))
    for c in range(2):
        expect = num[c] / (np.log(t / tc[c]) + np.sum(1.0 / (np.arange(ne) + 0.5)))
        assert np.max(np.abs(r["delta_new"][c] - expect)) < 1e-13, c
    assert np.max(np.abs(r["jx"])) < 1e-14 and np.max(np.abs(r["jy"])) < 1e-14
    # free energy (Eq. 17 :120 with Eq. 19): sum_G |D_G|^2 ln(T/T_c^G) + <|Delta(phi)|^2> sum 1/(n+1/2) - I, and
    # I = t sum_n <2 |Delta(phi)|^2/(eps_n + Lambda_n)> for the homogeneous solution (Eq. 38's integrand)
    fe = o.free_energy_density(delta, ne, r["fe_I"])
    ref = abs(Ds) ** 2 * np.log(t / tc[0]) + abs(Dd) ** 2 * np.log(t / tc[1])
    for k in range(nphi):
        phi = 2 * np.pi * k / nphi
        W = o.angle_info(k)[2]
        d2 = abs(Ds + Dd * np.sqrt(2.0) * np.cos(2 * phi)) ** 2
        L = np.sqrt(eps ** 2 + d2)
        ref += W * (d2 * np.sum(1.0 / (np.arange(ne) + 0.5)) - t * np.sum(2.0 * d2 / (eps + L)))
    assert np.max(np.abs(fe[mask > 0] - ref)) < 1e-13


def test_second_component_with_zero_amplitude_changes_nothing():
    """Delta_2 = 0: the first component's Delta_new, j, I equal the one-component sweep bit for bit (the node gap is
    the same sum), and the projection on the second basis function is what a one-component run cannot see."""
    wl = wlmod.make_workload(1, pts_per_xi=4, n_angles=16, n_energies=12)
    o1 = oracle.Oracle.from_workload(wl)
    r1 = o1.sweep(wl.delta0, wl.Aext_x, wl.Aext_y, wl.n_energies)
    o2 = oracle.Oracle.from_workload(wl)
    o2.set_components([wl.symmetry, 2], [1.0, 0.3])
    d2 = np.stack([wl.delta0, np.zeros_like(wl.delta0)])
    r2 = o2.sweep(d2, wl.Aext_x, wl.Aext_y, wl.n_energies)
    assert np.array_equal(r2["delta_new"][0], r1["delta_new"]) and np.array_equal(r2["jx"], r1["jx"]) and np.array_equal(r2["fe_I"], r1["fe_I"])
    assert np.max(np.abs(r2["delta_new"][1])) > 1e-6        # a vortex + walls do induce a d_xy admixture


# ---- the paper's truncated eigen-decomposition of the vector-potential kernel (App. D, D7-D9 :1023-1038) -----------
def test_lowrank_vector_potential_against_the_full_correlation():
    """D8 with all N eigenpairs is D1 exactly (G = V Lambda V^T); with N* < N of them (D9) the error obeys the
    Cauchy-Schwarz bound |dA| <= (2/kappa^2) ||G - G_N*||_F ||J||_F = (2/kappa^2) sqrt(sum_{n>=N*} lambda_n^2) ||J||_F
    (each |m'-m|, |n'-n| entry of the table is visited at most four times), and N* grows as eps shrinks."""
    n, h, kappa = 24, 0.25, 1.7
    shapes = [Shape(kind=0, cx=0.0, cy=0.0, r=0.5 * n * h - 0.1)]
    mask = make_mask(shapes, n, n, h)
    rng = np.random.default_rng(5)
    jx = rng.normal(size=(n, n)) * mask; jy = rng.normal(size=(n, n)) * mask
    ex, ey = oracle.vector_potential(mask, h, kappa, jx, jy)
    fx, fy, nfull = oracle.vector_potential_lowrank(mask, h, kappa, jx, jy, 0.0)      # eps = 0: D9 is never met, all N pairs
    assert nfull == n
    assert np.max(np.abs(fx - ex)) < 1e-12 * np.max(np.abs(ex)) and np.max(np.abs(fy - ey)) < 1e-12 * np.max(np.abs(ey))
    G = np.array([[oracle.G_table_entry(a, b, h) for b in range(n)] for a in range(n)])
    lam = np.sort(np.abs(np.linalg.eigvalsh(G)))[::-1]
    last = n
    for eps in (1e-1, 1e-2, 1e-4, 1e-6):
        ax, ay, ns = oracle.vector_potential_lowrank(mask, h, kappa, jx, jy, eps)
        assert 1 <= ns <= n
        assert np.sqrt(1.0 - np.sum(lam[:ns] ** 2) / np.sum(lam ** 2)) < eps                       # D9 holds for N* ...
        assert ns == 1 or not np.sqrt(1.0 - np.sum(lam[:ns - 1] ** 2) / np.sum(lam ** 2)) < eps     # ... and not for N* - 1
        m = mask.astype(bool)
        Jn = np.sqrt(np.sum((jx - jx[m].mean()) ** 2 * mask))
        bound = 2.0 / kappa ** 2 * np.sqrt(np.sum(lam[ns:] ** 2)) * Jn
        assert np.max(np.abs(ax - ex)) <= bound * (1 + 1e-9) + 1e-15
        last = ns
    assert last > 3                                                                            # eps = 1e-6 needs several pairs


# ---- Fermi-surface quadrature (:189) and basis functions (Table III :1238-1246) ---------------------------------------
@pytest.mark.parametrize("nphi,order", [(64, 4), (20, 4), (18, 3), (10, 2), (7, 1)])
def test_quadrature_weights_are_the_composite_newton_cotes_rules(nphi, order):
    """:189 "Boole's rule, Simpson's 3/8 rule, Simpson's 1/3 rule or the trapezoidal rule depending on N_phi mod 4, 3, 2":
    the periodic composite rule built from scipy's closed Newton-Cotes coefficients of that order."""
    from scipy.integrate import newton_cotes
    an, _ = newton_cotes(order, 1)                       # weights on 0..order for spacing 1
    w = np.zeros(nphi)
    for start in range(0, nphi, order):
        for i, a in enumerate(an):
            w[(start + i) % nphi] += a
    w /= nphi                                            # spacing 1/N_phi of the unit circle average
    sq = make_mask([square(0.4)], 4, 4, 0.1)
    o = oracle.Oracle(4, 4, 0.1, sq, [square(0.4)], 0.5, 0, nphi)
    W = np.array([o.angle_info(k)[2] for k in range(nphi)])
    assert np.max(np.abs(W - w)) < 1e-15 and abs(W.sum() - 1.0) < 1e-14
    if nphi % 2 == 0:
        ot = oracle.Oracle(4, 4, 0.1, sq, [square(0.4)], 0.5, 0, nphi, quadrature=1)
        assert np.allclose([ot.angle_info(k)[2] for k in range(nphi)], 1.0 / nphi, rtol=0, atol=1e-16)


def test_basis_functions_are_orthonormal_on_the_angle_set():
    """<eta_i eta_j> = delta_ij (:143, used to divide Eq. 20 down to Eq. 22) for s, d_x2-y2, d_xy, g (Table III) with the
    paper's quadrature at N_phi = 64 (the products carry frequencies <= 8, none of which aliases with the period-4
    weight pattern), with and without a crystal-axes rotation."""
    sq = make_mask([square(0.4)], 4, 4, 0.1)
    for rot in (0.0, 0.031):
        eta = []
        for sym in range(4):
            o = oracle.Oracle(4, 4, 0.1, sq, [square(0.4)], 0.5, sym, 64, crystal_rotation=rot)
            info = [o.angle_info(k) for k in range(64)]
            eta.append(np.array([e for _, e, _ in info])); W = np.array([w for _, _, w in info])
        gram = np.array([[np.sum(W * a * b) for b in eta] for a in eta])
        assert np.max(np.abs(gram - np.eye(4))) < 1e-13
    # d_x2-y2 -> d_xy under a rotation of the crystal axes by 1/8 turn (:890)
    o1 = oracle.Oracle(4, 4, 0.1, sq, [square(0.4)], 0.5, 1, 64, crystal_rotation=0.125)
    o2 = oracle.Oracle(4, 4, 0.1, sq, [square(0.4)], 0.5, 2, 64)
    assert max(abs(o1.angle_info(k)[1] - o2.angle_info(k)[1]) for k in range(64)) < 1e-14


def test_opcount_scalar_runs_the_same_step():
    """bench.py's "textbook" flop count comes from running the oracle's own step statements on an operation-counting
    scalar: it must return the step's value, and the tallies must be those of the formula as printed (closed form: one
    complex square root, one complex exponential, three complex divisions and one real-by-complex; mid-point C4-C9: one
    square root, one division, no exponential)."""
    for st in (0, 1):
        for (g, De, z, l) in ((0.2 - 0.3j, 0.3 + 0.1j, 0.04 + 0.25j, 0.05), (0.1 + 0.6j, 0.34 - 0.02j, 0.3 + 0.003j, 0.1)):
            d = oracle.step_opcount(st, g, De, z, l)
            assert abs(d["value"] - oracle.step(g, De, z, l, st)) < 1e-15
    c, m = oracle.step_opcount(0), oracle.step_opcount(1)
    assert (c["sqrt"], c["exp"], c["sincos"]) == (2, 1, 1) and (m["sqrt"], m["exp"], m["sincos"]) == (2, 0, 0)
    assert c["div"] == 2 * 3 + 1 and m["div"] == 2 * 1 + 1          # 2 real divisions per complex division + 1 in the square root
    assert 40 <= c["mul"] <= 70 and 25 <= c["add"] <= 45
