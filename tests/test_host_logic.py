"""CPU tests of the CUDA library's host side: the .so loads, exports every declared symbol, and its
independently written trajectory generator produces the same tables as the oracle's (integers equal,
floats to 1e-12) on the shapes of the configs.  No compute call is made here (no GPU)."""
import ctypes

import numpy as np
import pytest

import oracle
import workloads as wlmod
import paper_2205_15000_b200 as sc
from paper_2205_15000_b200 import build as scbuild


@pytest.fixture(scope="module")
def lib():
    scbuild.build()
    return sc.load_library()


def test_library_exports_every_declared_symbol(lib):
    names = sc.declared_symbols()
    assert {"sc_create", "sc_destroy", "sc_set_fields", "sc_riccati_sweep", "sc_ldos",
            "sc_update_vector_potential", "sc_iterate", "sc_reset_boundary"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/sc_riccati.h but not exported"
    assert b"sm_100a" in lib.sc_version()


def test_no_cpu_fallback_without_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    wl = wlmod.make_workload(0)
    with pytest.raises(sc.ScError) as e:
        sc.ScContext.from_workload(wl)
    assert e.value.status == 4           # SC_ERR_CUDA: fails loudly, no CPU path


def test_argument_errors(lib):
    wl = wlmod.make_workload(0)
    with pytest.raises(sc.ScError) as e:     # odd number of angles
        sc.ScContext(wl.nx, wl.ny, wl.h, wl.mask, wl.shapes, wl.t, wl.kappa, wl.symmetry, 15, 8, tables_only=True)
    assert e.value.status == 2
    bad = wl.mask.copy(); bad[0, 0] = 0
    with pytest.raises(sc.ScError) as e:     # mask disagrees with the shapes
        sc.ScContext(wl.nx, wl.ny, wl.h, bad, wl.shapes, wl.t, wl.kappa, wl.symmetry, 16, 8, tables_only=True)
    assert e.value.status == 2
    with pytest.raises(sc.ScError) as e:
        sc.ScContext(wl.nx, wl.ny, wl.h, wl.mask, wl.shapes, -1.0, wl.kappa, wl.symmetry, 16, 8, tables_only=True)
    assert e.value.status == 1


CASES = [
    (0, {}),
    (1, dict(pts_per_xi=5, n_angles=16, n_energies=4)),
    (2, dict(pts_per_xi=4, n_angles=32, n_energies=4, size_scale=0.5)),
    (4, dict(pts_per_xi=4, n_angles=24, n_energies=4, size_scale=0.25)),
]


def _workload(cfg, kw):
    return wlmod.make_annulus_workload(**kw) if cfg == "annulus" else wlmod.make_workload(cfg, **kw)


CASES += [("annulus", {}), ("annulus", dict(hole_offset=0.9, n_angles=12, pts_per_xi=4.0))]   # two trajectories per line


@pytest.mark.parametrize("cfg,kw", CASES)
def test_trajectory_tables_match_oracle(lib, cfg, kw):
    wl = _workload(cfg, kw)
    o = oracle.Oracle.from_workload(wl)
    c = sc.ScContext.from_workload(wl, tables_only=True)
    assert c.n_rot == o.nrot and c.n_traj == o.ntraj
    for k in range(wl.n_angles):
        a, b = o.tables(k), c.sc_debug_tables(k)
        for key in ("t", "jf", "jl", "elem_in", "elem_out"):
            assert np.array_equal(a[key], b[key]), (k, key)
        assert np.max(np.abs(a["u_in"] - b["u_in"])) < 1e-12 and np.max(np.abs(a["u_out"] - b["u_out"])) < 1e-12
        # entry gather (start value of gamma): same trajectories, same weights (order-insensitive)
        for i in range(len(a["t"])):
            ga = {int(j): w for j, w in zip(a["g_idx"][i, 0], a["g_w"][i, 0]) if j >= 0}
            gb = {int(j): w for j, w in zip(b["g_idx"][i], b["g_w"][i]) if j >= 0}
            assert ga.keys() == gb.keys(), (k, i)
            assert all(abs(ga[j] - gb[j]) < 1e-10 for j in ga)
    c.close()


@pytest.mark.parametrize("annulus", [False, True])
def test_mirror_structure_of_tables(lib, annulus):
    """angle k+N/2 is the exact mirror (j,t)->(N_rot-1-j, N_rot-1-t) of angle k — what lets the kernel take
    gamma-tilde_k from gamma_{k+N/2} (Eq. 13 :95); with a hole, the intervals of a line come in reverse order."""
    wl = wlmod.make_annulus_workload(hole_offset=0.7) if annulus else wlmod.make_workload(1, pts_per_xi=5, n_angles=16, n_energies=4)
    c = sc.ScContext.from_workload(wl, tables_only=True)
    H = wl.n_angles // 2
    for k in range(H):
        a, b = c.sc_debug_tables(k), c.sc_debug_tables(k + H)
        assert np.array_equal(a["t"][::-1], c.n_rot - 1 - b["t"])
        assert np.array_equal(a["jf"][::-1], c.n_rot - 1 - b["jl"])
        assert np.array_equal(a["u_in"][::-1], -b["u_out"])
    c.close()


# ---- Ozaki pole table (ref. 77): an input generator, pinned against the exact Fermi function ---------
def test_ozaki_table_reproduces_the_fermi_function():
    from paper_2205_15000_b200.ozaki import ozaki_poles, ozaki_energy_table
    x = np.linspace(-25.0, 25.0, 1001)
    exact = 1.0 / (1.0 + np.exp(x))
    for n in (12, 24):
        xi, R = ozaki_poles(n)
        f = 0.5 - sum(r * (1.0 / (x - 1j * a) + 1.0 / (x + 1j * a)) for a, r in zip(xi, R))
        assert np.max(np.abs(f - exact)) < 1e-13 and np.max(np.abs(f.imag)) < 1e-14
        # the lowest poles are the Matsubara frequencies pi (2n+1) with unit residue; the last ones carry the tail
        assert np.max(np.abs(xi[:n // 3] / np.pi - (2 * np.arange(n // 3) + 1))) < 1e-9 and np.max(np.abs(R[:n // 3] - 1)) < 1e-9
        assert np.all(np.diff(xi) > 0) and R[-1] > 10.0
    z, w = ozaki_energy_table(0.3, 12)
    assert np.allclose(z[:4], 1j * 0.3 * (np.arange(4) + 0.5), rtol=1e-12) and np.all(z.real == 0) and np.all(w > 0)


def test_ozaki_sum_reaches_the_infinite_matsubara_limit_of_the_gap_equation():
    """Bulk s-wave gap equation (Eq. 20 :135): ln t + sum_n [1/(n+1/2) - t/sqrt(eps_n^2 + D^2)] = 0 in the library's units.
    The summand decays only like 1/eps^3, so the pole sum is not exact, but 24 Ozaki poles are 300 times closer to the
    infinite-sum value (200 000 Matsubara terms plus the analytic tail) than 24 plain Matsubara terms, and 48 poles
    reach 1e-7."""
    from paper_2205_15000_b200.ozaki import ozaki_energy_table
    t, D = 0.3, 0.27
    summand = lambda eps: t / eps - t / np.sqrt(eps * eps + D * D)
    n = np.arange(200000, dtype=np.float64)
    eps = t * (n + 0.5)
    full = float(np.sum(summand(eps))) + 0.5 * D * D / (t * t) / (2.0 * 200000.0 ** 2)    # tail ~ int D^2/(2 t^2 n^3)
    oz = {}
    for npole in (24, 48):
        z, w = ozaki_energy_table(t, npole)
        oz[npole] = float(np.sum(w * summand(z.imag)))
    plain = float(np.sum(summand(eps[:24])))
    assert abs(oz[24] - full) < 2e-6 and abs(oz[48] - full) < 1e-7 and abs(plain - full) > 3e-4
