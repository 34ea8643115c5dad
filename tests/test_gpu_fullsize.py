"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

cfg 1 and cfg 2 are small enough for the oracle to sweep in full on the box's host cores (2e9 / 1e10 updates): every
output is compared element by element, once through the stats instantiation of the march and once through the
stats-free one (the one sc_iterate and bench.py launch; cfg 1 / cfg 2 have 128 / 256 Matsubara energies, whole warps,
so that is the unit-weight kernel).  cfg 3 runs sc_ldos at its full 512 energies and compares 18 sampled energy planes
(the planes are independent per energy) at 1 and 4 boundary iterations.  cfg 4 (5.3e11 updates, ~an hour of oracle
time) follows §8(d)'s rule: the production launch itself (256 angles x 512 energies, no stats) is compared on every
16th angle x ALL 512 energies — the per-angle node sums SF, SG, SI at every lattice node and the boundary values
gamma_end, gamma-tilde_end of every trajectory — plus the N_phi = 16, N_eps = 32 twin on the full 1600 x 1600 grid
element by element in FP64 and FP32, plus properties that hold at any size.
Tolerance: 1e-9 relative max-norm in FP64, 2e-4 in FP32 mode (north_star; R21).
"""
import numpy as np
import pytest

import oracle
import workloads as wlmod

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-9
TOL32 = 2e-4
BENCH_KERNEL = {64: "march_kernel<0,false,0,double,1,true>", 32: "march_kernel<0,false,0,float,1,true>"}   # what bench.py times


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


def gpu_sweep(ctx, wl, stats):
    n = (wl.ny, wl.nx)
    dn = torch.zeros(n, dtype=torch.complex128, device="cuda")
    jx = torch.zeros(n, dtype=torch.float64, device="cuda"); jy = torch.zeros_like(jx); fe = torch.zeros_like(jx)
    st = ctx.sc_riccati_sweep(dn, jx, jy, fe, want_stats=stats)
    torch.cuda.synchronize()
    return dict(delta_new=dn.cpu().numpy(), jx=jx.cpu().numpy(), jy=jy.cpu().numpy(), fe_I=fe.cpu().numpy(), stats=st)


@pytest.mark.parametrize("cfg", [1, 2])
def test_full_config_sweep_elementwise(sc, cfg):
    """100 % of the outputs of one sweep (Delta_new, jx, jy, I at every grid point), both march instantiations."""
    wl = wlmod.make_workload(cfg)
    Ax = wl.Aext_x if np.any(wl.Aext_x) else None
    Ay = wl.Aext_y if np.any(wl.Aext_x) else None
    o = oracle.Oracle.from_workload(wl)
    ro = o.sweep(wl.delta0, Ax, Ay, wl.n_energies)
    for stats in (True, False):
        ctx = sc.ScContext.from_workload(wl)
        ctx.sc_set_fields(dev(wl.delta0.astype(np.complex128)), dev(Ax), dev(Ay))
        rg = gpu_sweep(ctx, wl, stats)
        assert ctx.sc_debug_last_march_variant() == (BENCH_KERNEL[64] if not stats else "march_kernel<0,true,0,double,1,false>")
        for key in ("delta_new", "jx", "jy", "fe_I"):
            assert relerr(rg[key], ro[key]) < TOL, (stats, key)
        if stats:
            assert rg["stats"].n_updates == ro["stats"]["n_updates"] and rg["stats"].n_bad == 0
            assert abs(rg["stats"].min_one_minus_abs_gamma - ro["stats"]["min_one_minus_abs_gamma"]) < 1e-9
        ctx.close()


def test_full_config3_ldos_sampled_energy_planes(sc):
    """sc_ldos at cfg 3's full launch configuration (512 energies, 128 angles, 566 x 566 grid) at 1 and 4 boundary
    iterations; 18 of the 512 energy planes (3.5 % of the output, every grid point of each) are compared,
    spread over the table with both ends and the +-eps pair around zero energy."""
    wl = wlmod.make_workload(3)
    ctx = sc.ScContext.from_workload(wl)
    ctx.sc_set_fields(dev(wl.delta0.astype(np.complex128)))
    idx = np.unique(np.concatenate([np.linspace(0, 511, 16).round().astype(int), [255, 256]]))
    assert len(idx) == 18 and idx[0] == 0 and idx[-1] == 511
    o = oracle.Oracle.from_workload(wl)
    out = torch.zeros((wl.n_energies, wl.ny, wl.nx), dtype=torch.float64, device="cuda")
    for iters in (1, 4):
        ctx.sc_ldos(wl.ldos_energies, wl.ldos_broadening, iters, out)
        torch.cuda.synchronize()
        assert ctx.sc_debug_last_march_variant() == "march_kernel<1,false,0,double,2,false>"
        ref = o.ldos(wl.delta0, None, None, wl.ldos_energies[idx], wl.ldos_broadening, iters)
        got = out[torch.as_tensor(idx, device="cuda")].cpu().numpy()
        assert relerr(got, ref) < TOL, iters
        assert np.all(got[:, wl.mask > 0] > 0) and np.all(got[:, wl.mask == 0] == 0)
    # north_star's ABS check on the full-size grain: zero-energy weight piles up at the [110] walls, not in the bulk
    zero = out[255].cpu().numpy()
    cy, cx = wl.ny // 2, wl.nx // 2
    wall = zero[wl.mask > 0].max()
    assert wall > 10.0 * zero[cy, cx]
    ctx.close()


def test_full_config4_production_launch_every_16th_angle_all_energies(sc):
    """SURVEY §8(d) rule for cfg 4, in FP64 and in FP32 mode.  ONE production sweep (the launch bench.py times: 256 angles
    x 512 Matsubara energies, plain table, no stats -> march_kernel<0,false,0,double|float,1,true>) from the reset boundary
    stores; the oracle sweeps every 16th angle (k = 0, 16, ..., 240: 8 marched pairs, both members of each) with all 512
    energies, once, and both precisions are compared with it.  Compared, all from that one launch: SF, SG, SI at every
    lattice node of the 16 angles (6.25 % of the per-angle sums the grid fields are made of, 16 energy rounds accumulated
    each) and gamma_end / gamma-tilde_end of every trajectory of those angles at every energy (the march's boundary
    output).  Then properties of the full grid outputs."""
    wl = wlmod.make_workload(4)
    Ax, Ay = wl.Aext_x, wl.Aext_y
    o = oracle.Oracle.from_workload(wl)
    z, w = o.matsubara(wl.n_energies)
    angles = list(range(0, wl.n_angles, 16))
    stores = o.reset_stores(wl.delta0, Ax, Ay, z)
    ro = o.raw_sweep(wl.delta0, Ax, Ay, z, w, stores, angle_list=angles, dbg_angle=-2)
    del stores
    assert ro["stats"]["n_bad"] == 0
    for precision, tol in ((64, TOL), (32, TOL32)):
        ctx = sc.ScContext.from_workload(wl, precision=precision)
        ctx.sc_set_fields(dev(wl.delta0.astype(np.complex128)), dev(Ax), dev(Ay))
        rg = gpu_sweep(ctx, wl, stats=False)
        assert ctx.sc_debug_last_march_variant() == BENCH_KERNEL[precision]
        assert ro["stats"]["n_updates"] * (wl.n_angles // len(angles)) == 4 * (ctx.n_pieces // 2) * wl.n_energies   # discs: every angle has the same pieces
        for ia, k in enumerate(angles):
            SF, SG, SI = ctx.sc_debug_partial(k)
            for name, a, b in (("SF", SF, ro["dbg"]["SF"][ia]), ("SG", SG, ro["dbg"]["SG"][ia]), ("SI", SI, ro["dbg"]["SI"][ia])):
                assert relerr(a, b) < tol, (precision, k, name, relerr(a, b))
            ge, gte = ctx.sc_debug_stores(k)
            r0, r1 = o.traj_offset(k), o.traj_offset(k) + o.ntraj_angle(k)
            assert ge.shape == (r1 - r0, wl.n_energies)
            assert relerr(ge, ro["stores"][0][r0:r1]) < tol and relerr(gte, ro["stores"][1][r0:r1]) < tol, (precision, k)
        # --- properties of the full outputs ---
        for key in ("delta_new", "jx", "jy", "fe_I"):
            assert np.all(np.isfinite(rg[key])) and np.all(rg[key][wl.mask == 0] == 0)
        # the phase of Delta_new winds -20 times around the rim (20 vortices, R11/R19)
        R = 0.95 * 40.0
        th = np.linspace(0, 2 * np.pi, 4001)
        ii = np.rint(R * np.cos(th) / wl.h + 0.5 * (wl.nx - 1)).astype(int); jj = np.rint(R * np.sin(th) / wl.h + 0.5 * (wl.ny - 1)).astype(int)
        ph = np.unwrap(np.angle(rg["delta_new"][jj, ii]))
        assert round((ph[-1] - ph[0]) / (2 * np.pi)) == -20
        # a second sweep with stats: invariants of the whole launch
        st = gpu_sweep(ctx, wl, stats=True)["stats"]
        assert st.n_bad == 0 and st.n_updates == 4 * (ctx.n_pieces // 2) * wl.n_energies
        assert 0.0 < st.min_one_minus_abs_gamma < 1.0
        ctx.close()
        del ctx, rg
        torch.cuda.empty_cache()


@pytest.mark.parametrize("precision,tol", [(64, TOL), (32, TOL32)])
def test_full_config4_grid_twin_elementwise(sc, precision, tol):
    """cfg 4's grain, grid (1600 x 1600), fields and flux with N_phi = 16, N_eps = 32: two Jacobi sweeps,
    every output compared at every grid point, through the stats-free unit-weight kernel, in FP64 and in FP32 mode."""
    wl = wlmod.make_workload(4, n_angles=16, n_energies=32)
    o = oracle.Oracle.from_workload(wl)
    ctx = sc.ScContext.from_workload(wl, precision=precision)
    ctx.sc_set_fields(dev(wl.delta0.astype(np.complex128)), dev(wl.Aext_x), dev(wl.Aext_y))
    stores = None
    for it in range(2):
        ro = o.sweep(wl.delta0, wl.Aext_x, wl.Aext_y, wl.n_energies, stores); stores = ro["stores"]
        rg = gpu_sweep(ctx, wl, stats=False)
        assert ctx.sc_debug_last_march_variant() == BENCH_KERNEL[precision]
        for key in ("delta_new", "jx", "jy", "fe_I"):
            assert relerr(rg[key], ro[key]) < tol, (it, key, relerr(rg[key], ro[key]))
    ctx.close()
