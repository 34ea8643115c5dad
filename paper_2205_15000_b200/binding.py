"""ctypes binding of include/sc_riccati.h — same names, argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os
import re
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

SYM_S, SYM_DX2Y2, SYM_DXY, SYM_G = 0, 1, 2, 3

_HERE = os.path.dirname(os.path.abspath(__file__))
_HEADER = os.path.join(os.path.dirname(_HERE), "include", "sc_riccati.h")

_STATUS = {0: "SC_OK", 1: "SC_ERR_ARG", 2: "SC_ERR_GEOMETRY", 3: "SC_ERR_STATE", 4: "SC_ERR_CUDA",
           5: "SC_ERR_NOMEM", 6: "SC_ERR_NUMERIC"}


class ScError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


class _Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("h", C.c_double)]


class _Shape(C.Structure):
    _fields_ = [("kind", C.c_int), ("add", C.c_int), ("cx", C.c_double), ("cy", C.c_double), ("r", C.c_double),
                ("nvert", C.c_int), ("vx", C.POINTER(C.c_double)), ("vy", C.POINTER(C.c_double))]


class _Opts(C.Structure):
    _fields_ = [("n_angles", C.c_int), ("n_matsubara", C.c_int), ("precision", C.c_int), ("stepper", C.c_int),
                ("quadrature", C.c_int), ("charge_sign", C.c_int), ("bc_mode", C.c_int),
                ("crystal_rotation", C.c_double), ("device", C.c_int), ("cuda_stream", C.c_void_p),
                ("residual_norm", C.c_int)]


class _Stats(C.Structure):
    _fields_ = [("res_delta", C.c_double), ("res_j", C.c_double), ("res_A", C.c_double), ("res_fe", C.c_double),
                ("min_one_minus_abs_gamma", C.c_double), ("n_updates", C.c_longlong),
                ("n_updates_executed", C.c_longlong), ("ms", C.c_float), ("n_bad", C.c_int)]


@dataclass
class SweepStats:
    res_delta: float
    res_j: float
    res_A: float
    res_fe: float
    min_one_minus_abs_gamma: float
    n_updates: int
    n_updates_executed: int
    ms: float
    n_bad: int


def lib_path() -> str:
    """The in-tree library built by `paper_2205_15000_b200.build`."""
    return os.path.join(_HERE, "libsc_riccati.so")


def declared_symbols() -> list:
    """Names of the functions include/sc_riccati.h declares (used by the load/export test)."""
    src = open(_HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sc_[a-z0-9_]+)\s*\(", src)))


ALLREDUCE_FN = C.CFUNCTYPE(None, C.c_void_p)

_lib = None


def load_library():
    """Load the in-tree CUDA library.  Fails loudly when it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    p = lib_path()
    if not os.path.exists(p):
        raise ScError(4, f"{p} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                         "(the CUDA extension is required; there is no CPU path)")
    L = C.CDLL(p)
    vp, i, d = C.c_void_p, C.c_int, C.c_double
    L.sc_version.restype = C.c_char_p
    L.sc_last_error.restype = C.c_char_p
    L.sc_last_error.argtypes = [vp]
    L.sc_create.argtypes = [C.POINTER(_Grid), vp, C.POINTER(_Shape), i, d, d, i, C.POINTER(_Opts), C.POINTER(vp)]
    L.sc_destroy.argtypes = [vp]
    L.sc_set_fields.argtypes = [vp, vp, vp, vp]
    L.sc_reset_boundary.argtypes = [vp]
    L.sc_set_energies.argtypes = [vp, vp, vp, vp, i, d]
    L.sc_set_components.argtypes = [vp, i, vp, vp]
    L.sc_set_allreduce_hook.argtypes = [vp, vp, ALLREDUCE_FN, vp]
    L.sc_riccati_sweep.argtypes = [vp, vp, vp, vp, vp, C.POINTER(_Stats)]
    L.sc_ldos.argtypes = [vp, vp, i, d, i, vp, C.POINTER(_Stats)]
    L.sc_update_vector_potential.argtypes = [vp, vp, vp, vp, vp, C.POINTER(d)]
    L.sc_set_external_field.argtypes = [vp, vp, vp]
    L.sc_iterate.argtypes = [vp, i, d, i, vp, vp, vp, C.POINTER(_Stats)]
    L.sc_set_accelerator_params.argtypes = [vp, d, d, d, d, d]
    L.sc_set_vector_potential_error.argtypes = [vp, d, C.POINTER(i)]
    L.sc_debug_geometry.argtypes = [vp, C.POINTER(i), C.POINTER(i), C.POINTER(C.c_longlong)]
    L.sc_debug_tables.argtypes = [vp, i, C.POINTER(i), vp, vp, vp, vp]
    L.sc_debug_trajectory.argtypes = [vp, i, i, i, C.POINTER(i), vp, vp]
    L.sc_debug_partial.argtypes = [vp, i, vp, vp, vp]
    L.sc_debug_stores.argtypes = [vp, i, vp, vp]
    L.sc_debug_math.argtypes = [vp, i, vp]
    L.sc_debug_fp64_peak.argtypes = [vp, C.POINTER(d), C.POINTER(d)]
    L.sc_debug_last_march_ms.argtypes = [vp, C.POINTER(C.c_float)]
    L.sc_debug_fp64_peak_sustained.argtypes = [vp, d, C.POINTER(d)]
    L.sc_debug_pipe_peak.argtypes = [vp, i, d, C.POINTER(d)]
    L.sc_debug_march_time.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(i)]
    L.sc_debug_march_units.argtypes = [vp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
    L.sc_debug_last_march_variant.argtypes = [vp, C.c_char_p, i]
    L.sc_debug_launch_count.argtypes = [vp, C.POINTER(C.c_longlong)]
    L.sc_residual_norm_static.argtypes = [vp, vp, C.c_longlong, i, vp, i, vp, C.c_char_p, i]
    _lib = L
    return L


def _dev_ptr(t, dtype_name: str, numel: int):
    """Raw device pointer of a contiguous CUDA torch tensor (None passes through)."""
    if t is None:
        return None
    import torch
    want = {"f64": torch.float64, "c128": torch.complex128}[dtype_name]
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == want and t.numel() == numel):
        raise ScError(1, f"expected a contiguous CUDA {dtype_name} tensor with {numel} elements")
    return C.c_void_p(t.data_ptr())


RESIDUAL_STATIC_MAX_ELEMENTS = 8388608     # SC_RESIDUAL_STATIC_MAX_ELEMENTS of include/sc_riccati.h


def sc_residual_norm_static(x_new, x_old, out, norm_p: int = 2, stream: Optional[int] = None):
    """Eq. 27's residual of two complex128 CUDA tensors into `out` (CUDA float64, 3 values: ||x_new - x_old||_p,
    ||x_old||_p, ratio) without any allocation by the library: the scratch is a static device array (see the header).
    Enqueues on `stream` (default: torch's current stream of the tensors' device) and does not synchronise."""
    import torch
    L = load_library()
    n = x_new.numel() if isinstance(x_new, torch.Tensor) else 0
    a, b, o = _dev_ptr(x_new, "c128", n), _dev_ptr(x_old, "c128", n), _dev_ptr(out, "f64", 3)
    if a is None or b is None or o is None:
        raise ScError(1, "sc_residual_norm_static: x_new, x_old and out are required")
    if not (x_new.device == x_old.device == out.device):
        raise ScError(1, "sc_residual_norm_static: tensors live on different devices")
    if stream is None:
        stream = torch.cuda.current_stream(x_new.device).cuda_stream
    err = C.create_string_buffer(256)
    rc = L.sc_residual_norm_static(a, b, n, int(norm_p), o, x_new.device.index, C.c_void_p(stream), err, len(err))
    if rc:
        raise ScError(rc, err.value.decode())
    return out


def _stats(s: _Stats) -> SweepStats:
    return SweepStats(s.res_delta, s.res_j, s.res_A, s.res_fe, s.min_one_minus_abs_gamma, s.n_updates,
                      s.n_updates_executed, s.ms, s.n_bad)


class ScContext:
    """sc_ctx: one grain + discretisation on one GPU."""

    def __init__(self, nx: int, ny: int, h: float, mask: np.ndarray, shapes: Sequence, t: float, kappa: float,
                 symmetry: int, n_angles: int, n_matsubara: int, *, crystal_rotation: float = 0.0,
                 quadrature: int = 0, charge_sign: int = -1, bc_mode: int = 0, precision: int = 64,
                 stepper: int = 0, device: int = 0, stream: Optional[int] = None, tables_only: bool = False,
                 residual_norm: int = 2):
        """tables_only=True keeps a context whose sc_create stopped at SC_ERR_CUDA (no device) so that the host-built
        trajectory tables can still be read with sc_debug_tables; every compute call on it fails."""
        import torch
        L = load_library()
        if not torch.cuda.is_available() and not tables_only:
            raise ScError(4, "no CUDA device: this library has no CPU path")
        self._L = L
        self.nx, self.ny, self.h, self.t, self.kappa = nx, ny, h, t, kappa
        self.n_angles, self.n_matsubara = n_angles, n_matsubara
        self.n_components = 1
        self.device = torch.device("cuda", device)
        mask = np.ascontiguousarray(mask, np.uint8)
        arr = (_Shape * len(shapes))()
        keep = []
        for k, s in enumerate(shapes):
            vx = np.ascontiguousarray(s.vx, np.float64); vy = np.ascontiguousarray(s.vy, np.float64)
            keep += [vx, vy]
            arr[k] = _Shape(int(s.kind), int(s.add), s.cx, s.cy, s.r, len(vx),
                            vx.ctypes.data_as(C.POINTER(C.c_double)), vy.ctypes.data_as(C.POINTER(C.c_double)))
        if stream is None:
            stream = torch.cuda.current_stream(self.device).cuda_stream if torch.cuda.is_available() else 0
        opts = _Opts(n_angles, n_matsubara, precision, stepper, quadrature, charge_sign, bc_mode, crystal_rotation,
                     device, C.c_void_p(stream), residual_norm)
        grid = _Grid(nx, ny, h)
        h_ = C.c_void_p()
        rc = L.sc_create(C.byref(grid), mask.ctypes.data_as(C.c_void_p), arr, len(shapes), t, kappa, symmetry,
                         C.byref(opts), C.byref(h_))
        self._h = h_
        if rc == 4 and tables_only and h_:
            rc = 0
        if rc:
            msg = L.sc_last_error(h_).decode() if h_ else "sc_create failed"
            if h_:
                L.sc_destroy(h_)
            self._h = None
            raise ScError(rc, msg)
        nrot, ntraj, npieces = C.c_int(), C.c_int(), C.c_longlong()
        L.sc_debug_geometry(self._h, C.byref(nrot), C.byref(ntraj), C.byref(npieces))
        self.n_rot, self.n_traj, self.n_pieces = nrot.value, ntraj.value, npieces.value

    @classmethod
    def from_workload(cls, wl, **kw):
        return cls(wl.nx, wl.ny, wl.h, wl.mask, wl.shapes, wl.t, wl.kappa, wl.symmetry, wl.n_angles, wl.n_energies,
                   crystal_rotation=wl.crystal_rotation, charge_sign=wl.charge_sign, **kw)

    def close(self):
        if getattr(self, "_h", None):
            self._L.sc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc:
            raise ScError(rc, self._L.sc_last_error(self._h).decode())

    # ---- the calls of include/sc_riccati.h -------------------------------------------------------
    def sc_set_components(self, symmetries, tc_ratio):
        sy = np.ascontiguousarray(symmetries, np.int32); tc = np.ascontiguousarray(tc_ratio, np.float64)
        if len(sy) != len(tc):
            raise ScError(1, "symmetries and tc_ratio differ in length")
        self._check(self._L.sc_set_components(self._h, len(sy), sy.ctypes.data_as(C.c_void_p), tc.ctypes.data_as(C.c_void_p)))
        self.n_components = len(sy)

    def sc_set_fields(self, delta, Ax=None, Ay=None):
        n = self.nx * self.ny
        self._check(self._L.sc_set_fields(self._h, _dev_ptr(delta, "c128", self.n_components * n), _dev_ptr(Ax, "f64", n), _dev_ptr(Ay, "f64", n)))

    def sc_set_energies(self, z, w, denominator_sum=float("nan")):
        z = np.ascontiguousarray(z, np.complex128)
        zr = np.ascontiguousarray(z.real); zi = np.ascontiguousarray(z.imag); w = np.ascontiguousarray(w, np.float64)
        self._check(self._L.sc_set_energies(self._h, zr.ctypes.data_as(C.c_void_p), zi.ctypes.data_as(C.c_void_p),
                                            w.ctypes.data_as(C.c_void_p), len(zr), float(denominator_sum)))
        self.n_matsubara = len(zr)

    def sc_set_allreduce_hook(self, acc, fn):
        """acc: CUDA fp64 tensor [2 n_components + 3][ny][nx]; fn(): enqueues the all-reduce of acc on the context's stream."""
        if fn is None:
            self._hook = None
            self._check(self._L.sc_set_allreduce_hook(self._h, None, ALLREDUCE_FN(), None))
            return
        self._hook = (ALLREDUCE_FN(lambda user: fn()), acc)          # keep the callback and the buffer alive
        self._check(self._L.sc_set_allreduce_hook(self._h, _dev_ptr(acc, "f64", (2 * self.n_components + 3) * self.nx * self.ny), self._hook[0], None))

    def sc_reset_boundary(self):
        self._check(self._L.sc_reset_boundary(self._h))

    def sc_riccati_sweep(self, delta_new=None, jx=None, jy=None, fe_I=None, want_stats=False):
        n = self.nx * self.ny
        st = _Stats()
        self._check(self._L.sc_riccati_sweep(self._h, _dev_ptr(delta_new, "c128", self.n_components * n), _dev_ptr(jx, "f64", n),
                                             _dev_ptr(jy, "f64", n), _dev_ptr(fe_I, "f64", n),
                                             C.byref(st) if want_stats else None))
        return _stats(st) if want_stats else None

    def sc_ldos(self, energies, broadening, n_boundary_iters, ldos, want_stats=False):
        e = np.ascontiguousarray(energies, np.float64)
        st = _Stats()
        self._check(self._L.sc_ldos(self._h, e.ctypes.data_as(C.c_void_p), len(e), broadening, n_boundary_iters,
                                    _dev_ptr(ldos, "f64", len(e) * self.nx * self.ny), C.byref(st) if want_stats else None))
        return _stats(st) if want_stats else None

    def sc_update_vector_potential(self, jx, jy, Aind_x, Aind_y, want_energy=False):
        n = self.nx * self.ny
        fe = C.c_double()
        self._check(self._L.sc_update_vector_potential(self._h, _dev_ptr(jx, "f64", n), _dev_ptr(jy, "f64", n),
                                                       _dev_ptr(Aind_x, "f64", n), _dev_ptr(Aind_y, "f64", n),
                                                       C.byref(fe) if want_energy else None))
        return fe.value if want_energy else None

    def sc_set_external_field(self, Ax, Ay):
        n = self.nx * self.ny
        self._check(self._L.sc_set_external_field(self._h, _dev_ptr(Ax, "f64", n), _dev_ptr(Ay, "f64", n)))

    def sc_iterate(self, accelerator, step, burnin, delta, Aind_x=None, Aind_y=None, want_stats=False):
        n = self.nx * self.ny
        st = _Stats()
        self._check(self._L.sc_iterate(self._h, accelerator, step, int(burnin), _dev_ptr(delta, "c128", self.n_components * n),
                                       _dev_ptr(Aind_x, "f64", n), _dev_ptr(Aind_y, "f64", n),
                                       C.byref(st) if want_stats else None))
        return _stats(st) if want_stats else None

    def sc_set_vector_potential_error(self, eps):
        """Returns N*, the number of eigenpairs of G kept (0: exact FFT correlation)."""
        n = C.c_int()
        self._check(self._L.sc_set_vector_potential_error(self._h, float(eps), C.byref(n)))
        return n.value

    def sc_set_accelerator_params(self, drag=0.0, step_factor=0.0, cos_similarity_min=0.0, step_min=0.0, step_max=0.0):
        self._check(self._L.sc_set_accelerator_params(self._h, drag, step_factor, cos_similarity_min, step_min, step_max))

    # ---- debug taps --------------------------------------------------------------------------------
    def sc_debug_tables(self, k):
        n = C.c_int()
        self._check(self._L.sc_debug_tables(self._h, k, C.byref(n), None, None, None, None))
        it = np.zeros((n.value, 6), np.int32); dt = np.zeros((n.value, 2)); gi = np.zeros((n.value, 4), np.int32); gw = np.zeros((n.value, 4))
        self._check(self._L.sc_debug_tables(self._h, k, C.byref(n), it.ctypes.data_as(C.c_void_p), dt.ctypes.data_as(C.c_void_p),
                                            gi.ctypes.data_as(C.c_void_p), gw.ctypes.data_as(C.c_void_p)))
        return dict(t=it[:, 0], jf=it[:, 1], jl=it[:, 2], elem_in=it[:, 3], elem_out=it[:, 4], u_in=dt[:, 0], u_out=dt[:, 1],
                    g_idx=gi, g_w=gw)

    def sc_debug_trajectory(self, k, local, n_energy):
        G = np.zeros(self.n_rot, np.complex128); GT = np.zeros(self.n_rot, np.complex128)
        nn = C.c_int()
        self._check(self._L.sc_debug_trajectory(self._h, k, local, n_energy, C.byref(nn), G.ctypes.data_as(C.c_void_p),
                                                GT.ctypes.data_as(C.c_void_p)))
        return G[:nn.value], GT[:nn.value]

    def sc_debug_partial(self, k):
        nr = self.n_rot
        SF = np.zeros((nr, nr), np.complex128); SG = np.zeros((nr, nr)); SI = np.zeros((nr, nr))
        self._check(self._L.sc_debug_partial(self._h, k, SF.ctypes.data_as(C.c_void_p), SG.ctypes.data_as(C.c_void_p),
                                             SI.ctypes.data_as(C.c_void_p)))
        return SF, SG, SI

    def sc_debug_stores(self, k, n_energies=None):
        """(gamma_end, gamma_tilde_end) [n_traj(k)][n_energies] written by the last sweep's march launch."""
        n = C.c_int()
        self._check(self._L.sc_debug_tables(self._h, k, C.byref(n), None, None, None, None))
        ne = n_energies or self.n_matsubara
        G = np.zeros((n.value, ne), np.complex128); GT = np.zeros((n.value, ne), np.complex128)
        self._check(self._L.sc_debug_stores(self._h, k, G.ctypes.data_as(C.c_void_p), GT.ctypes.data_as(C.c_void_p)))
        return G, GT

    def sc_debug_math(self, n=2000):
        out = np.zeros(6)
        self._check(self._L.sc_debug_math(self._h, n, out.ctypes.data_as(C.c_void_p)))
        return dict(zip(["rcp", "rsqrt", "exp", "expm1", "sin", "cosm1"], out))

    def sc_debug_last_march_ms(self):
        ms = C.c_float()
        self._check(self._L.sc_debug_last_march_ms(self._h, C.byref(ms)))
        return ms.value

    last_march_ms = sc_debug_last_march_ms

    def sc_debug_march_time(self):
        """(total ms, launches) of the march kernel since the previous call; resets."""
        ms, n = C.c_float(), C.c_int()
        self._check(self._L.sc_debug_march_time(self._h, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def sc_debug_march_units(self):
        """(units marched, units in rounds that spilled T, units in rounds that recomputed T from the pole-subtracted
        table) since the previous call; resets."""
        a, b, c = C.c_longlong(), C.c_longlong(), C.c_longlong()
        self._check(self._L.sc_debug_march_units(self._h, C.byref(a), C.byref(b), C.byref(c)))
        return a.value, b.value, c.value

    def sc_debug_last_march_variant(self):
        buf = C.create_string_buffer(128)
        self._check(self._L.sc_debug_last_march_variant(self._h, buf, 128))
        return buf.value.decode()

    def sc_debug_launch_count(self):
        """Kernels of the library launched by this thread since the previous call; resets."""
        n = C.c_longlong()
        self._check(self._L.sc_debug_launch_count(self._h, C.byref(n)))
        return n.value

    def sc_debug_fp64_peak_sustained(self, seconds=2.0):
        a = C.c_double()
        self._check(self._L.sc_debug_fp64_peak_sustained(self._h, float(seconds), C.byref(a)))
        return a.value

    def sc_debug_pipe_peak(self, pipe, seconds=1.0):
        a = C.c_double()
        self._check(self._L.sc_debug_pipe_peak(self._h, int(pipe), float(seconds), C.byref(a)))
        return a.value

    def sc_debug_fp64_peak(self):
        a, b = C.c_double(), C.c_double()
        self._check(self._L.sc_debug_fp64_peak(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value
