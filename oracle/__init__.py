"""CPU oracle for the Riccati sweep — TEST INFRASTRUCTURE, not the product.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference` legs may
import this package.  It never imports `paper_2205_15000_b200` and shares no code with it.

The numerical core is `sc_oracle.cpp` (plain C++17 loops, fp64); this file is the ctypes binding plus
the few vector formulas that close a sweep (Eq. 22, 8, 17/19, 27) and the self-consistency
driver (Algorithm 1 :203-205, App. E Picard / Barzilai-Borwein), written out in numpy.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sc_oracle.cpp")
_LIB = os.path.join(_HERE, "libsc_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle (g++ -O2 -fopenmp).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c++17", _SRC, "-o", _LIB])
    return _LIB


class _Shape(C.Structure):
    _fields_ = [("kind", C.c_int), ("add", C.c_int), ("cx", C.c_double), ("cy", C.c_double), ("r", C.c_double),
                ("nvert", C.c_int), ("vx", C.POINTER(C.c_double)), ("vy", C.POINTER(C.c_double))]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        L = _lib
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, C.c_int, C.c_double, C.c_void_p, C.POINTER(_Shape), C.c_int, C.c_double,
                                 C.c_int, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_components.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.orc_error.restype = C.c_char_p
        L.orc_error.argtypes = [C.c_void_p]
        for f in ("orc_nrot", "orc_ntraj", "orc_n_gather_fallback"):
            getattr(L, f).argtypes = [C.c_void_p]
        L.orc_ntraj_angle.argtypes = [C.c_void_p, C.c_int]
        L.orc_traj_offset.argtypes = [C.c_void_p, C.c_int]
        L.orc_angle_info.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_tables.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 4
        L.orc_step.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p]
        L.orc_gamma_h.argtypes = [C.c_void_p] * 3
        L.orc_opcount.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]
        L.orc_march.argtypes = [C.c_int, C.c_int] + [C.c_void_p] * 9
        L.orc_reset_stores.argtypes = [C.c_void_p] * 4 + [C.c_int] + [C.c_void_p] * 4
        L.orc_sweep.argtypes = ([C.c_void_p] * 4 + [C.c_int] + [C.c_void_p] * 12 + [C.c_void_p, C.c_int] +
                                [C.c_int] + [C.c_void_p] * 4 + [C.c_void_p] * 3)
        L.orc_debug_trajectory.argtypes = ([C.c_void_p] * 4 + [C.c_int] * 4 + [C.c_void_p] * 7)
        L.orc_debug_nodes.argtypes = [C.c_void_p] * 4 + [C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.orc_G.restype = C.c_double
        L.orc_G.argtypes = [C.c_int, C.c_int, C.c_double]
        L.orc_vector_potential.argtypes = [C.c_int, C.c_int, C.c_double, C.c_void_p, C.c_double] + [C.c_void_p] * 4
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


# ------------------------------------------------------------------------------------------------
# scalar helpers for the pins
# ------------------------------------------------------------------------------------------------
def step(g: complex, De: complex, z: complex, l: float, stepper: int = 0) -> complex:
    out = np.zeros(2)
    lib().orc_step(stepper, _p(np.array([g.real, g.imag])), _p(np.array([De.real, De.imag])),
                   _p(np.array([z.real, z.imag])), l, _p(out))
    return complex(out[0], out[1])


def step_opcount(stepper: int = 0, g: complex = 0.2 - 0.3j, De: complex = 0.3 + 0.1j, z: complex = 0.04 + 0.25j, l: float = 0.05):
    """Real floating-point operations of one step as the oracle states it (textbook complex arithmetic), counted by
    running the same C++ statements on an operation-counting scalar: dict(mul, add, div, sqrt, exp, sincos, value)."""
    cnt = np.zeros(6, np.int64); out = np.zeros(2)
    lib().orc_opcount(stepper, _p(np.array([g.real, g.imag])), _p(np.array([De.real, De.imag])),
                      _p(np.array([z.real, z.imag])), l, _p(cnt), _p(out))
    d = dict(zip(("mul", "add", "div", "sqrt", "exp", "sincos"), (int(v) for v in cnt)))
    d["value"] = complex(out[0], out[1])
    return d


def gamma_h(De: complex, z: complex) -> complex:
    out = np.zeros(2)
    lib().orc_gamma_h(_p(np.array([De.real, De.imag])), _p(np.array([z.real, z.imag])), _p(out))
    return complex(out[0], out[1])


def march(lengths, De, a, z0: complex, g_start: complex, gt_start: complex, stepper: int = 0):
    """March gamma up and gamma-tilde down a synthetic list of pieces; returns (G, GT, g_end, gt_end)
    with G, GT at the M-1 interior nodes."""
    lengths = _f64(lengths); De = _c128(De); a = _f64(a)
    M = len(lengths)
    G = np.zeros(M - 1, np.complex128); GT = np.zeros(M - 1, np.complex128); ends = np.zeros(4)
    lib().orc_march(stepper, M, _p(lengths), _p(De), _p(a), _p(np.array([z0.real, z0.imag])),
                    _p(np.array([g_start.real, g_start.imag])), _p(np.array([gt_start.real, gt_start.imag])),
                    _p(G), _p(GT), _p(ends))
    return G, GT, complex(ends[0], ends[1]), complex(ends[2], ends[3])


def G_table_entry(m: int, n: int, h: float) -> float:
    return lib().orc_G(m, n, h)


def vector_potential(mask, h, kappa, jx, jy):
    """A_ind of PAPER.md D1 (:1009) by direct summation, mask-mean of j removed (:1040)."""
    mask = np.ascontiguousarray(mask, np.uint8)
    ny, nx = mask.shape
    Ax = np.zeros((ny, nx)); Ay = np.zeros((ny, nx))
    lib().orc_vector_potential(nx, ny, h, _p(mask), kappa, _p(_f64(jx)), _p(_f64(jy)), _p(Ax), _p(Ay))
    return Ax, Ay


def vector_potential_lowrank(mask, h, kappa, jx, jy, eps):
    """The paper's own evaluation of D1 (App. D :1023-1038): eigendecompose the N x N table G_{m,n} (D7), keep the N*
    eigenpairs of largest |lambda| with sqrt(1 - sum_{n<N*} lambda_n^2 / sum_n lambda_n^2) < eps (D9), and apply
    A = -(1/kappa^2) sum_k lambda_k sum_{m'} sum_{n'} V_{|m'-m|} V_{|n'-n|} j_{m'n'} (D8) as two 1-D cross-correlations
    per eigenpair; j has its mask-mean removed (:1040).  Returns (Ax, Ay, N*)."""
    mask = np.ascontiguousarray(mask, np.uint8)
    ny, nx = mask.shape
    N = max(nx, ny)
    G = np.array([[G_table_entry(m, n, h) for n in range(N)] for m in range(N)])
    lam, V = np.linalg.eigh(G)
    order = np.argsort(-np.abs(lam), kind="stable")
    tot = float(np.sum(lam ** 2))
    nstar = N
    kept = 0.0
    for c, k in enumerate(order):
        kept += float(lam[k]) ** 2
        if math.sqrt(max(0.0, 1.0 - kept / tot)) < eps:
            nstar = c + 1
            break
    m = mask.astype(bool)
    out = []
    for j in (np.asarray(jx, np.float64), np.asarray(jy, np.float64)):
        J = np.where(m, j - j[m].mean(), 0.0)                         # [n'][m']
        A = np.zeros((ny, nx))
        for k in order[:nstar]:
            v = V[:, k]
            Ty = v[np.abs(np.subtract.outer(np.arange(ny), np.arange(ny)))]   # (Ty)_{n,n'} = V_{|n'-n|}
            Tx = v[np.abs(np.subtract.outer(np.arange(nx), np.arange(nx)))]
            A += lam[k] * (Ty @ J @ Tx)
        out.append(-A / (kappa * kappa))
    return out[0], out[1], nstar


def matsubara_denominator(t: float, ne: int) -> float:
    """D = ln t + sum_{n<ne} 1/(n + 1/2): denominator of PAPER.md Eq. 22 (:144), same cutoff as the
    numerator (reading R-A5)."""
    return math.log(t) + float(np.sum(1.0 / (np.arange(ne) + 0.5)))


class Oracle:
    """One grain + discretisation (the arguments of the product's `sc_create`)."""

    def __init__(self, nx, ny, h, mask, shapes, t, symmetry, n_angles, *, crystal_rotation=0.0, quadrature=0,
                 charge_sign=-1, bc_mode=0, stepper=0, kappa=-1.0):
        L = lib()
        self.nx, self.ny, self.h, self.t = nx, ny, h, t
        self.kappa = kappa
        self.sigma = charge_sign
        self.n_angles = n_angles
        self.mask = np.ascontiguousarray(mask, np.uint8)
        arr = (_Shape * len(shapes))()
        self._keep = []
        for i, s in enumerate(shapes):
            vx = np.asarray(s.vx, np.float64); vy = np.asarray(s.vy, np.float64)
            self._keep += [vx, vy]
            arr[i] = _Shape(s.kind, int(s.add), s.cx, s.cy, s.r, len(vx),
                            vx.ctypes.data_as(C.POINTER(C.c_double)), vy.ctypes.data_as(C.POINTER(C.c_double)))
        self._h = L.orc_create(nx, ny, h, _p(self.mask), arr, len(shapes), t, symmetry, crystal_rotation,
                               n_angles, quadrature, charge_sign, bc_mode, stepper)
        err = L.orc_error(self._h).decode()
        if err:
            raise ValueError(err)
        self.nrot = L.orc_nrot(self._h)
        self.ntraj = L.orc_ntraj(self._h)
        self.n_gather_fallback = L.orc_n_gather_fallback(self._h)
        self.symmetries = [int(symmetry)]
        self.tc_ratio = [1.0]
        self.crystal_rotation = crystal_rotation

    def set_components(self, symmetries, tc_ratio):
        """Several order-parameter components (Eq. 1 :37, Listing 11 :909-926): Delta(p_F,R) = sum_G
        Delta_G(R) eta_G(p_F), each with its own T_c^G = tc_ratio[G] * T_c in the gap equation (Eq. 20-22 :135-144;
        T_c, the energy unit, is the largest).  Afterwards every Delta argument / Delta_new result is
        [ncomp][ny][nx]."""
        syms = np.ascontiguousarray(symmetries, np.int32)
        assert len(syms) == len(tc_ratio) >= 1
        lib().orc_set_components(self._h, len(syms), _p(syms))
        self.symmetries = [int(v) for v in syms]
        self.tc_ratio = [float(v) for v in tc_ratio]

    @property
    def ncomp(self):
        return len(self.symmetries)

    @classmethod
    def from_workload(cls, wl, **kw):
        return cls(wl.nx, wl.ny, wl.h, wl.mask, wl.shapes, wl.t, wl.symmetry, wl.n_angles,
                   crystal_rotation=wl.crystal_rotation, charge_sign=wl.charge_sign, kappa=wl.kappa, **kw)

    def __del__(self):
        try:
            lib().orc_destroy(self._h)
        except Exception:
            pass

    # -- tables ---------------------------------------------------------------------------------
    def angle_info(self, k):
        v = np.zeros(2); eta = np.zeros(1); W = np.zeros(1)
        lib().orc_angle_info(self._h, k, _p(v), _p(eta), _p(W))
        return v, float(eta[0]), float(W[0])

    def ntraj_angle(self, k):
        return lib().orc_ntraj_angle(self._h, k)

    def traj_offset(self, k):
        return lib().orc_traj_offset(self._h, k)

    def tables(self, k):
        n = self.ntraj_angle(k)
        it = np.zeros((n, 6), np.int32); dt = np.zeros((n, 6)); gi = np.zeros((n, 2, 4), np.int32); gw = np.zeros((n, 2, 4))
        lib().orc_tables(self._h, k, _p(it), _p(dt), _p(gi), _p(gw))
        return dict(t=it[:, 0], jf=it[:, 1], jl=it[:, 2], elem_in=it[:, 3], elem_out=it[:, 4], u_in=dt[:, 0],
                    u_out=dt[:, 1], n_in=dt[:, 2:4], n_out=dt[:, 4:6], g_idx=gi, g_w=gw)

    # -- sweep ----------------------------------------------------------------------------------
    def reset_stores(self, delta, Ax, Ay, z, ):
        z = _c128(z); ne = len(z)
        g = np.zeros((self.ntraj, ne), np.complex128); gt = np.zeros((self.ntraj, ne), np.complex128)
        lib().orc_reset_stores(self._h, _p(_c128(delta)), _p(_f64(Ax)), _p(_f64(Ay)), ne,
                               _p(_f64(z.real)), _p(_f64(z.imag)), _p(g), _p(gt))
        return g, gt

    def raw_sweep(self, delta, Ax, Ay, z, w, stores, angle_list=None, dbg_angle=-1):
        """One Jacobi sweep.  Returns dict(num, Jx, Jy, I, R, stores=(g_new, gt_new), stats, [dbg])."""
        z = _c128(z); ne = len(z); w = _f64(w)
        delta = _c128(delta); Ax = _f64(Ax); Ay = _f64(Ay)
        g_old, gt_old = stores
        g_new = np.array(g_old, copy=True); gt_new = np.array(gt_old, copy=True)
        ny, nx = self.ny, self.nx
        assert delta.size == self.ncomp * ny * nx
        num = np.zeros((ny, nx) if self.ncomp == 1 else (self.ncomp, ny, nx), np.complex128)
        Jx = np.zeros((ny, nx)); Jy = np.zeros((ny, nx)); Ia = np.zeros((ny, nx)); Ra = np.zeros((ny, nx))
        al = None if angle_list is None else np.ascontiguousarray(angle_list, np.int32)
        dbg = None
        if dbg_angle >= 0 or dbg_angle == -2:        # -2: the node sums of every angle of angle_list, [len(angle_list)][nrot][nrot]
            shp = (self.nrot, self.nrot) if dbg_angle >= 0 else (len(al), self.nrot, self.nrot)
            dbg = dict(SF=np.zeros(shp, np.complex128), SG=np.zeros(shp), SI=np.zeros(shp), SR=np.zeros(shp))
        gmin = np.zeros(1); nupd = np.zeros(1, np.int64); bad = np.zeros(1, np.int32)
        lib().orc_sweep(self._h, _p(delta), _p(Ax), _p(Ay), ne, _p(_f64(z.real)), _p(_f64(z.imag)), _p(w),
                        _p(g_old), _p(gt_old), _p(g_new), _p(gt_new), _p(num), _p(Jx), _p(Jy), _p(Ia), _p(Ra),
                        _p(al), 0 if al is None else len(al), dbg_angle,
                        _p(dbg["SF"]) if dbg else None, _p(dbg["SG"]) if dbg else None,
                        _p(dbg["SI"]) if dbg else None, _p(dbg["SR"]) if dbg else None,
                        _p(gmin), _p(nupd), _p(bad))
        return dict(num=num, Jx=Jx, Jy=Jy, I=Ia, R=Ra, stores=(g_new, gt_new),
                    stats=dict(min_one_minus_abs_gamma=float(gmin[0]), n_updates=int(nupd[0]), n_bad=int(bad[0])),
                    dbg=dbg)

    def matsubara(self, ne):
        n = np.arange(ne, dtype=np.float64)
        return 1j * self.t * (n + 0.5), np.ones(ne)

    def sweep(self, delta, Ax, Ay, ne, stores=None, angle_list=None, dbg_angle=-1):
        """`sc_riccati_sweep`: Delta_new (Eq. 22 :144), j (Eq. 8 :69), I (Eq. 19 :128) from one Jacobi sweep
        at the Matsubara energies eps_n = t(n+1/2), n < ne (n >= 0 only and doubled, reading R-c7)."""
        z, w = self.matsubara(ne)
        if stores is None:
            stores = self.reset_stores(delta, Ax, Ay, z)
        r = self.raw_sweep(delta, Ax, Ay, z, w, stores, angle_list, dbg_angle)
        t = self.t
        m = self.mask.astype(bool)
        # Eq. 22 (:144): each component divides by its own ln(T/T_c^G) + sum 1/(n+1/2)
        D = np.array([math.log(t / tc) + float(np.sum(1.0 / (np.arange(ne) + 0.5))) for tc in self.tc_ratio])
        if self.ncomp == 1:
            r["delta_new"] = np.where(m, -2j * t * r["num"] / D[0], 0.0)
        else:
            r["delta_new"] = np.where(m[None], -2j * t * r["num"] / D[:, None, None], 0.0)
        r["jx"] = np.where(m, 2.0 * self.sigma * t * r["Jx"], 0.0)
        r["jy"] = np.where(m, 2.0 * self.sigma * t * r["Jy"], 0.0)
        r["fe_I"] = np.where(m, t * r["I"], 0.0)
        return r

    def ldos(self, delta, Ax, Ay, energies, broadening, n_boundary_iters):
        """`sc_ldos`: N(eps_m, R)/N_F = <Re g_n> (Eq. 14 :100) at eps_m + i delta, after n_boundary_iters
        Jacobi sweeps with frozen Delta, A starting from the homogeneous stores."""
        energies = np.asarray(energies, np.float64)
        out = np.zeros((len(energies), self.ny, self.nx))
        for m, e in enumerate(energies):
            z = np.array([e + 1j * broadening]); w = np.ones(1)
            stores = self.reset_stores(delta, Ax, Ay, z)
            for _ in range(n_boundary_iters):
                r = self.raw_sweep(delta, Ax, Ay, z, w, stores)
                stores = r["stores"]
            out[m] = np.where(self.mask.astype(bool), r["R"], 0.0)
        return out

    def free_energy_density(self, delta, ne, fe_I):
        """omega(R) of PAPER.md Eq. 17 (:120) without the magnetic term, Eilenberger form Eq. 19;
        |Delta(R)|^2 = <|Delta(p_F,R)|^2>_pF (:122) with the same Fermi-surface quadrature as the sweep."""
        if self.ncomp == 1:
            eta2 = sum(self.angle_info(k)[2] * self.angle_info(k)[1] ** 2 for k in range(self.n_angles))
            d2 = eta2 * np.abs(delta) ** 2
            return d2 * math.log(self.t) + d2 * float(np.sum(1.0 / (np.arange(ne) + 0.5))) - fe_I
        # Eq. 17 (:120): sum_G |Delta_G|^2 ln(T/T_c^G) + <|Delta(p_F,R)|^2> sum 1/(n+1/2) - I
        delta = np.asarray(delta).reshape(self.ncomp, self.ny, self.nx)
        d2 = np.zeros((self.ny, self.nx))
        for k in range(self.n_angles):
            W = self.angle_info(k)[2]
            tot = sum(self.basis(s, k) * delta[c] for c, s in enumerate(self.symmetries))
            d2 += W * np.abs(tot) ** 2
        logs = sum(np.abs(delta[c]) ** 2 * math.log(self.t / tc) for c, tc in enumerate(self.tc_ratio))
        return logs + d2 * float(np.sum(1.0 / (np.arange(ne) + 0.5))) - fe_I

    def basis(self, sym, k):
        """eta_G(phi_k) of Table III (:1238-1246) with the crystal-axes rotation (:890)."""
        phi = 2.0 * math.pi * k / self.n_angles - 2.0 * math.pi * self.crystal_rotation
        return {0: 1.0, 1: math.sqrt(2.0) * math.cos(2 * phi), 2: math.sqrt(2.0) * math.sin(2 * phi),
                3: math.sqrt(2.0) * math.sin(4 * phi)}[sym]

    def debug_trajectory(self, delta, Ax, Ay, k, local, z, n, stores):
        z = _c128(z); ne = len(z)
        G = np.zeros(self.nrot, np.complex128); GT = np.zeros(self.nrot, np.complex128); ends = np.zeros(8)
        nn = lib().orc_debug_trajectory(self._h, _p(_c128(delta)), _p(_f64(Ax)), _p(_f64(Ay)), k, local, ne, n,
                                        _p(_f64(z.real)), _p(_f64(z.imag)), _p(stores[0]), _p(stores[1]),
                                        _p(G), _p(GT), _p(ends))
        return G[:nn], GT[:nn], ends

    def debug_nodes(self, delta, Ax, Ay, k, local):
        Dn = np.zeros(self.nrot, np.complex128); an = np.zeros(self.nrot)
        nn = lib().orc_debug_nodes(self._h, _p(_c128(delta)), _p(_f64(Ax)), _p(_f64(Ay)), k, local, _p(Dn), _p(an))
        return Dn[:nn], an[:nn]


# ------------------------------------------------------------------------------------------------
# self-consistency driver (Algorithm 1 :203-205, Eq. 27 :201, App. E :1044-1127)
# ------------------------------------------------------------------------------------------------
def residual(new, old, p=2):
    """eps_G = ||x_i - x_{i-1}||_p / ||x_{i-1}||_p (Eq. 27)."""
    a = np.ravel(new - old); b = np.ravel(old)
    if p == 0:
        na, nb = np.max(np.abs(a)), np.max(np.abs(b))
    else:
        na, nb = np.sum(np.abs(a) ** p) ** (1.0 / p), np.sum(np.abs(b) ** p) ** (1.0 / p)
    return float(na / nb) if nb > 0 else float(na)


class Accelerator:
    """Fixed-point accelerators of App. E (:1044-1151) acting on the concatenated iterate x with d = g(x) - x (E4):
    update(d) returns the increment x_{i+1} - x_i.  `ncomp` equal slices of x are the "components" of CongAcc.
      0  Picard: alpha d (E5 :1070);
      1  Barzilai-Borwein with alternating BB1/BB2 scaling (E8-E11 :1107-1115), alpha clipped to [1e-3, 100]
         (Listing 15 :1121-1127).  Reading R-BB: iteration index i starts at 0; the first update uses alpha = step;
         for i >= 1 alpha_{i+1} = alpha_i * (s^BB1 if i odd else s^BB2);
      2  Polyak "small heavy sphere" (E6-E7 :1087-1089): v <- (1 - drag) v + alpha d, increment v, v_0 = 0
         (Listing 14 :1093: step 2.0, drag 0.5);
      3  CongAcc (E12-E17 :1134-1151), per component c: s = cos(m_c, d_c) (taken as 0 while m_c = 0);
         alpha_c <- clip(alpha_c k^s); w_c <- w_c if s >= s_min else the root w* of E17 (bisection on [0, 1],
         60 halvings); m_c <- w_c m_c + (1 - w_c) d_c; increment alpha_c m_c; w_{0,c} = 0, m_{0,c} = 0
         (Listing 16 :1157: step 0.5, k = 1.234, s_min = 0.7, alpha in [1e-3, 100])."""

    def __init__(self, kind=0, step=1.0, drag=0.5, step_factor=1.234, cos_min=0.7, step_min=1e-3, step_max=100.0, ncomp=4):
        self.kind, self.alpha = kind, step
        self.drag, self.kfac, self.smin, self.amin, self.amax, self.ncomp = drag, step_factor, cos_min, step_min, step_max, ncomp
        self.i = 0
        self.d_prev = None
        self.vel = None
        self.m = None
        self.alpha_c = [step] * ncomp
        self.w_c = [0.0] * ncomp

    @staticmethod
    def cos_mix(w, mm, md, dd):
        """cos(w m + (1-w) d, d) from the three dot products m.m, m.d, d.d."""
        num = w * md + (1.0 - w) * dd
        n2 = w * w * mm + 2.0 * w * (1.0 - w) * md + (1.0 - w) * (1.0 - w) * dd
        return num / np.sqrt(n2 * dd) if n2 > 0 and dd > 0 else 1.0

    def update(self, d):
        d = np.asarray(d, np.float64)
        if self.kind == 1 and self.d_prev is not None:
            dd = d - self.d_prev
            dot = abs(float(np.dot(self.d_prev, dd)))
            if self.i % 2 == 1:
                s = float(np.dot(self.d_prev, self.d_prev)) / dot if dot > 0 else 1.0
            else:
                nd = float(np.dot(dd, dd))
                s = dot / nd if nd > 0 else 1.0
            self.alpha = min(max(self.alpha * s, self.amin), self.amax)
        if self.kind == 2:
            if self.vel is None:
                self.vel = np.zeros_like(d)
            self.vel = (1.0 - self.drag) * self.vel + self.alpha * d
            upd = self.vel.copy()
        elif self.kind == 3:
            if self.m is None:
                self.m = np.zeros_like(d)
            n = d.size // self.ncomp
            upd = np.zeros_like(d)
            for c in range(self.ncomp):
                sl = slice(c * n, (c + 1) * n)
                mc, dc = self.m[sl], d[sl]
                mm, md, dd_ = float(np.dot(mc, mc)), float(np.dot(mc, dc)), float(np.dot(dc, dc))
                s = md / np.sqrt(mm * dd_) if mm > 0 and dd_ > 0 else 0.0
                self.alpha_c[c] = min(max(self.alpha_c[c] * self.kfac ** s, self.amin), self.amax)
                if self.i == 0:
                    self.w_c[c] = 0.0
                elif s < self.smin:
                    lo, hi = 0.0, 1.0                      # cos = 1 at w = 0 and = s < s_min at w = 1
                    for _ in range(60):
                        mid = 0.5 * (lo + hi)
                        if self.cos_mix(mid, mm, md, dd_) >= self.smin:
                            lo = mid
                        else:
                            hi = mid
                    self.w_c[c] = 0.5 * (lo + hi)
                self.m[sl] = self.w_c[c] * mc + (1.0 - self.w_c[c]) * dc
                upd[sl] = self.alpha_c[c] * self.m[sl]
        else:
            upd = self.alpha * d
        self.d_prev = d.copy()
        self.i += 1
        return upd


class Driver:
    """Algorithm 1 (:203-205): sweep -> A-solve -> accelerator on x = (Re Delta, Im Delta, kappa^2 A_x^ind,
    kappa^2 A_y^ind) (E3 :1053) -> residual (Eq. 27 :201).  `accelerator` and the keyword parameters are Accelerator's."""

    def __init__(self, orc: Oracle, Aext_x, Aext_y, ne, accelerator=0, step=1.0, norm=2, **kw):
        self.o, self.ne, self.norm = orc, ne, norm            # norm: p of Eq. 27 (:201; :960 "norm"): 1, 2, or 0 = maximum norm
        self.accel = Accelerator(accelerator, step, ncomp=4, **kw)
        self.Aext = (np.asarray(Aext_x, np.float64), np.asarray(Aext_y, np.float64))
        self.stores = None

    def iterate(self, delta, Aind_x, Aind_y, burnin=False):
        o = self.o
        Ax = self.Aext[0] + Aind_x; Ay = self.Aext[1] + Aind_y
        if self.stores is None:
            self.stores = o.reset_stores(delta, Ax, Ay, o.matsubara(self.ne)[0])
        r = o.sweep(delta, Ax, Ay, self.ne, self.stores)
        self.stores = r["stores"]
        out = dict(delta_new=r["delta_new"], jx=r["jx"], jy=r["jy"], fe_I=r["fe_I"])
        if burnin:
            out.update(delta=delta, Aind_x=Aind_x, Aind_y=Aind_y)
            return out
        k2 = o.kappa * o.kappa if o.kappa > 0 else 0.0
        if o.kappa > 0:
            gAx, gAy = vector_potential(o.mask, o.h, o.kappa, r["jx"], r["jy"])
        else:
            gAx, gAy = np.zeros_like(Aind_x), np.zeros_like(Aind_y)
        # E3 (:1053): x = (Re Delta_G, Im Delta_G for every component G, kappa^2 A_x, kappa^2 A_y)
        nc = o.ncomp
        n = o.nx * o.ny
        dl = np.asarray(delta).reshape(nc, o.ny, o.nx); dn = np.asarray(r["delta_new"]).reshape(nc, o.ny, o.nx)
        parts = lambda d_, ax_, ay_: np.concatenate([v for c in range(nc) for v in (d_[c].real.ravel(), d_[c].imag.ravel())] +
                                                    [k2 * ax_.ravel(), k2 * ay_.ravel()])
        x = parts(dl, Aind_x, Aind_y)
        gx = parts(dn, gAx, gAy)
        if self.accel.ncomp != 2 * nc + 2:
            self.accel.ncomp = 2 * nc + 2
            self.accel.alpha_c = [self.accel.alpha] * (2 * nc + 2); self.accel.w_c = [0.0] * (2 * nc + 2)
        xn = x + self.accel.update(gx - x)
        shp = (o.ny, o.nx)
        dout = np.stack([(xn[2 * c * n:(2 * c + 1) * n] + 1j * xn[(2 * c + 1) * n:(2 * c + 2) * n]).reshape(shp) * o.mask for c in range(nc)])
        out["delta"] = dout[0] if nc == 1 else dout
        if o.kappa > 0:
            out["Aind_x"] = (xn[2 * nc * n:(2 * nc + 1) * n] / k2).reshape(shp); out["Aind_y"] = (xn[(2 * nc + 1) * n:] / k2).reshape(shp)
        else:
            out["Aind_x"], out["Aind_y"] = Aind_x, Aind_y
        out["res_delta"] = residual(out["delta"], delta, self.norm)
        if o.kappa > 0:       # one element of a vector field is the 2-vector at a grid point: |A| = |A_x + i A_y|
            out["res_A"] = residual(out["Aind_x"] + 1j * out["Aind_y"], Aind_x + 1j * Aind_y, self.norm)
        out["alpha"] = self.accel.alpha if self.accel.kind != 3 else list(self.accel.alpha_c)
        out["w"] = list(self.accel.w_c)
        return out
