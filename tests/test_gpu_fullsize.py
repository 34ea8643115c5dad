"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

cfg 1 and cfg 2 are small enough for the oracle to sweep in full on the box's host cores (2e9 / 1e10 updates), so
they are compared element by element.  cfg 3 is compared on sampled energy planes (the LDOS planes are independent
per energy).  cfg 4 (5.3e11 updates, ~an hour of oracle time) is compared on sampled outputs the oracle can compute
one by one — gamma and gamma-tilde along sampled trajectories at sampled energies of the full 512-energy sweep, and
the per-angle node sums of sampled angles on an energy subset — plus properties that hold at any size.
Tolerance: 1e-9 relative max-norm (north_star; R21).
"""
import numpy as np
import pytest

import oracle
import workloads as wlmod

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-9


def relerr(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.max(np.abs(a - b)) / max(float(np.max(np.abs(b))), 1e-6))


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), device="cuda") if a is not None else None


@pytest.fixture(scope="module")
def sc():
    import paper_2205_15000_b200 as m
    from paper_2205_15000_b200 import build
    build.build()
    return m


def gpu_sweep(ctx, wl, Ax, Ay):
    n = (wl.ny, wl.nx)
    dn = torch.zeros(n, dtype=torch.complex128, device="cuda")
    jx = torch.zeros(n, dtype=torch.float64, device="cuda"); jy = torch.zeros_like(jx); fe = torch.zeros_like(jx)
    st = ctx.sc_riccati_sweep(dn, jx, jy, fe, want_stats=True)
    torch.cuda.synchronize()
    return dict(delta_new=dn.cpu().numpy(), jx=jx.cpu().numpy(), jy=jy.cpu().numpy(), fe_I=fe.cpu().numpy(), stats=st)


@pytest.mark.parametrize("cfg", [1, 2])
def test_full_config_sweep_elementwise(sc, cfg):
    wl = wlmod.make_workload(cfg)
    Ax = wl.Aext_x if np.any(wl.Aext_x) else None
    Ay = wl.Aext_y if np.any(wl.Aext_x) else None
    ctx = sc.ScContext.from_workload(wl)
    ctx.sc_set_fields(dev(wl.delta0.astype(np.complex128)), dev(Ax), dev(Ay))
    rg = gpu_sweep(ctx, wl, Ax, Ay)
    o = oracle.Oracle.from_workload(wl)
    ro = o.sweep(wl.delta0, Ax, Ay, wl.n_energies)
    for key in ("delta_new", "jx", "jy", "fe_I"):
        assert relerr(rg[key], ro[key]) < TOL, key
    assert rg["stats"].n_updates == ro["stats"]["n_updates"] and rg["stats"].n_bad == 0
    assert abs(rg["stats"].min_one_minus_abs_gamma - ro["stats"]["min_one_minus_abs_gamma"]) < 1e-9
    ctx.close()


def test_full_config3_ldos_sampled_energy_planes(sc):
    wl = wlmod.make_workload(3)
    ctx = sc.ScContext.from_workload(wl)
    ctx.sc_set_fields(dev(wl.delta0.astype(np.complex128)))
    idx = np.array([0, 37, 255, 256, 300, 511])              # includes the +-eps pair 255/256 around zero energy
    energies = wl.ldos_energies[idx]
    o = oracle.Oracle.from_workload(wl)
    for iters in (1, 2):
        out = torch.zeros((len(idx), wl.ny, wl.nx), dtype=torch.float64, device="cuda")
        ctx.sc_ldos(energies, wl.ldos_broadening, iters, out)
        torch.cuda.synchronize()
        ref = o.ldos(wl.delta0, None, None, energies, wl.ldos_broadening, iters)
        assert relerr(out.cpu().numpy(), ref) < TOL, iters
    # north_star's ABS check on the full-size grain: zero-energy weight piles up at the [110] walls, not in the bulk
    zero = out.cpu().numpy()[2]
    cy, cx = wl.ny // 2, wl.nx // 2
    wall = zero[wl.mask > 0].max()
    assert wall > 10.0 * zero[cy, cx]
    ctx.close()


def test_full_config4_sampled_outputs_and_properties(sc):
    wl = wlmod.make_workload(4)
    Ax, Ay = wl.Aext_x, wl.Aext_y
    ctx = sc.ScContext.from_workload(wl)
    ctx.sc_set_fields(dev(wl.delta0.astype(np.complex128)), dev(Ax), dev(Ay))
    rg = gpu_sweep(ctx, wl, Ax, Ay)                           # the sweep bench.py times: 256 angles x 512 energies
    st = rg["stats"]
    o = oracle.Oracle.from_workload(wl)
    # --- sampled trajectories x sampled energies of the FULL sweep (start values from the reset stores) ---
    nsel = np.array([0, 31, 32, 300, 511])
    z_all, _ = o.matsubara(wl.n_energies)
    z_sub = z_all[nsel]
    stores = o.reset_stores(wl.delta0, Ax, Ay, z_sub)
    rng = np.random.default_rng(4)
    for k in (0, 1, 37, 64, 127):
        nt = o.ntraj_angle(k)
        for local in sorted({0, nt - 1, nt // 2, int(rng.integers(nt)), int(rng.integers(nt))}):
            for i, n in enumerate(nsel):
                Go, GTo, _ = o.debug_trajectory(wl.delta0, Ax, Ay, k, local, z_sub, i, stores)
                Gg, GTg = ctx.sc_debug_trajectory(k, local, int(n))
                assert len(Gg) == len(Go)
                assert relerr(Gg, Go) < TOL and relerr(GTg, GTo) < TOL, (k, local, n)
    # --- properties of the full outputs ---
    assert st.n_bad == 0 and st.n_updates == 4 * (ctx.n_pieces // 2) * wl.n_energies
    assert 0.0 < st.min_one_minus_abs_gamma < 1.0
    for key in ("delta_new", "jx", "jy", "fe_I"):
        assert np.all(np.isfinite(rg[key])) and np.all(rg[key][wl.mask == 0] == 0)
    # the phase of Delta_new winds -20 times around the rim (20 vortices, R11/R19)
    R = 0.95 * 40.0
    th = np.linspace(0, 2 * np.pi, 4001)
    ii = np.rint(R * np.cos(th) / wl.h + 0.5 * (wl.nx - 1)).astype(int); jj = np.rint(R * np.sin(th) / wl.h + 0.5 * (wl.ny - 1)).astype(int)
    ph = np.unwrap(np.angle(rg["delta_new"][jj, ii]))
    assert round((ph[-1] - ph[0]) / (2 * np.pi)) == -20
    ctx.close()
    # --- per-angle node sums of sampled angles, same grid / trajectories / angles, energy subset (ragged: 5 of 512) ---
    ctx2 = sc.ScContext.from_workload(wl)
    ctx2.sc_set_energies(z_sub, np.ones(len(z_sub)))
    ctx2.sc_set_fields(dev(wl.delta0.astype(np.complex128)), dev(Ax), dev(Ay))
    ctx2.sc_riccati_sweep()
    torch.cuda.synchronize()
    for k in (3, 200):                                       # one from each half of the angle set (Eq. 13 partner)
        ro = o.raw_sweep(wl.delta0, Ax, Ay, z_sub, np.ones(len(z_sub)), stores, angle_list=[k], dbg_angle=k)
        SF, SG, SI = ctx2.sc_debug_partial(k)
        assert relerr(SF, ro["dbg"]["SF"]) < TOL and relerr(SG, ro["dbg"]["SG"]) < TOL and relerr(SI, ro["dbg"]["SI"]) < TOL
    ctx2.close()
