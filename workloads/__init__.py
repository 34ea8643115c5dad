"""Seeded synthetic workloads for the Riccati sweep (inputs only — no method arithmetic).

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path
(`paper_2205_15000_b200/`).  It builds the five `BASELINE.json` configs (zero-based cfg 0..4) as plain
numpy arrays: grid, mask, shape list, initial order parameter, external vector potential, energy lists.
It contains none of the solver's arithmetic: no Riccati step, no gap equation, no interpolation.  The
bulk-gap amplitudes used to scale the initial guesses are literal input constants;
`tests/test_oracle_pins.py` checks that the oracle reproduces them, not the other way round.

The paper uses no dataset (Table I :1189-1202 describe its example grains);
these grains copy those shapes: disc with one vortex, Abrikosov lattice in a disc, [110] d-wave edges,
LDOS sweep.  All random numbers come from numpy PCG64(seed = 220515000 + cfg index).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

SEED_BASE = 220515000

# symmetry codes (Table III :1238-1246) — shared enum values of the C ABIs on both sides
SYM_S, SYM_DX2Y2, SYM_DXY, SYM_G = 0, 1, 2, 3

# Bulk gap amplitudes Delta_Gamma(t, N_eps) in units of 2 pi kB Tc at each config's own cutoff — literal
# inputs for the initial guess; pinned against the oracle's gap solver in the tests.
BULK_GAP = {
    ("s", 0.5, 16): 0.268717,
    ("s", 0.1, 128): 0.280764,
    ("s", 0.05, 512): 0.280738,
    ("d", 0.1, 256): 0.240795,
}


@dataclass
class Shape:
    """One CSG component: kind 0 = disc, 1 = convex polygon (CCW vertices)."""
    kind: int
    add: bool = True
    cx: float = 0.0
    cy: float = 0.0
    r: float = 0.0
    vx: List[float] = field(default_factory=list)
    vy: List[float] = field(default_factory=list)

    def area(self) -> float:
        if self.kind == 0:
            return math.pi * self.r * self.r
        x = np.asarray(self.vx)
        y = np.asarray(self.vy)
        return 0.5 * float(np.sum(x * np.roll(y, -1) - np.roll(x, -1) * y))

    def strictly_inside(self, x: np.ndarray, y: np.ndarray) -> np.ndarray:
        if self.kind == 0:
            return (x - self.cx) ** 2 + (y - self.cy) ** 2 < self.r ** 2
        ins = np.ones(np.broadcast(x, y).shape, dtype=bool)
        nv = len(self.vx)
        for e in range(nv):
            x0, y0 = self.vx[e], self.vy[e]
            x1, y1 = self.vx[(e + 1) % nv], self.vy[(e + 1) % nv]
            dx, dy = x1 - x0, y1 - y0
            ln = math.hypot(dx, dy)
            nxo, nyo = dy / ln, -dx / ln          # outward normal of a CCW polygon
            ins &= (nxo * (x - x0) + nyo * (y - y0)) < 0.0
        return ins


def square(side: float, rotation_turns: float = 0.0) -> Shape:
    """Square of given side centred at the origin, rotated by `rotation_turns` full turns (CCW vertices)."""
    hs = 0.5 * side
    base = [(-hs, -hs), (hs, -hs), (hs, hs), (-hs, hs)]
    c, s = math.cos(2 * math.pi * rotation_turns), math.sin(2 * math.pi * rotation_turns)
    vx = [c * x - s * y for x, y in base]
    vy = [s * x + c * y for x, y in base]
    return Shape(kind=1, vx=vx, vy=vy)


def disc(radius: float, cx: float = 0.0, cy: float = 0.0, add: bool = True) -> Shape:
    return Shape(kind=0, add=add, cx=cx, cy=cy, r=radius)


@dataclass
class Workload:
    name: str
    cfg: int
    nx: int
    ny: int
    h: float
    shapes: List[Shape]
    mask: np.ndarray              # uint8 [ny][nx]
    symmetry: int
    crystal_rotation: float       # turns
    n_angles: int
    n_energies: int
    t: float                      # T / Tc
    kappa: float                  # <= 0: infinite
    charge_sign: int
    delta0: np.ndarray            # complex128 [ny][nx], zero outside the mask
    Aext_x: np.ndarray            # float64 [ny][nx] on the whole grid
    Aext_y: np.ndarray
    bulk_gap: float
    ldos_energies: Optional[np.ndarray] = None   # real energies (cfg 3)
    ldos_broadening: float = 0.0
    accelerator: int = 0          # 0 Picard, 1 Barzilai-Borwein
    n_iterations: int = 1
    notes: str = ""

    @property
    def x(self) -> np.ndarray:
        return (np.arange(self.nx) - 0.5 * (self.nx - 1)) * self.h

    @property
    def y(self) -> np.ndarray:
        return (np.arange(self.ny) - 0.5 * (self.ny - 1)) * self.h

    @property
    def n_in(self) -> int:
        return int(self.mask.sum())

    def area(self) -> float:
        return sum((1 if s.add else -1) * s.area() for s in self.shapes)


def grid_xy(nx: int, ny: int, h: float):
    x = (np.arange(nx) - 0.5 * (nx - 1)) * h
    y = (np.arange(ny) - 0.5 * (ny - 1)) * h
    return np.meshgrid(x, y)      # [ny][nx] each


def make_mask(shapes: List[Shape], nx: int, ny: int, h: float) -> np.ndarray:
    """mask[j][i] = 1 iff grid point (x_i, y_j) is strictly inside the CSG (add = union, remove = subtract,
    in list order)."""
    X, Y = grid_xy(nx, ny, h)
    ins = np.zeros((ny, nx), dtype=bool)
    for s in shapes:
        si = s.strictly_inside(X, Y)
        if s.add:
            ins |= si
        else:
            # closed removed region: points on its boundary are not in the grain either
            if s.kind == 0:
                closed = (X - s.cx) ** 2 + (Y - s.cy) ** 2 <= s.r ** 2
            else:
                closed = si
            ins &= ~closed
    return ins.astype(np.uint8)


def _even_grid(extent: float, h: float) -> int:
    n = int(round(extent / h))
    return n


def _vortex_phase(X, Y, centres, winding=-1.0):
    chi = np.zeros_like(X)
    for (cx, cy) in centres:
        chi += winding * np.arctan2(Y - cy, X - cx)      # PAPER.md:896 (B2), winding -1
    return chi


def _seeded_vortex_positions(rng, n, rmax, min_sep):
    pts = []
    guard = 0
    while len(pts) < n:
        guard += 1
        if guard > 100000:
            raise RuntimeError("cannot place vortices")
        r = rmax * math.sqrt(rng.random())
        th = 2 * math.pi * rng.random()
        p = (r * math.cos(th), r * math.sin(th))
        if all(math.hypot(p[0] - q[0], p[1] - q[1]) >= min_sep for q in pts):
            pts.append(p)
    return pts


def make_workload(cfg: int, *, pts_per_xi: Optional[float] = None, n_angles: Optional[int] = None,
                  n_energies: Optional[int] = None, size_scale: float = 1.0) -> Workload:
    """Build config `cfg` (zero-based index into BASELINE.json `configs`).

    The keyword overrides give reduced twins of the same shape (coarser grid, fewer angles/energies,
    smaller grain) for parity tests that the oracle can finish in seconds.
    """
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + cfg))
    if cfg == 0:
        ppx = pts_per_xi or 10.0
        side = 5.0 * size_scale
        h = 1.0 / ppx
        n = _even_grid(side, h)
        shapes = [square(side)]
        sym, rot, na, ne, t, kappa = SYM_S, 0.0, n_angles or 16, n_energies or 16, 0.5, -1.0
        gap = BULK_GAP[("s", 0.5, 16)]
        mask = make_mask(shapes, n, n, h)
        u = rng.uniform(-1.0, 1.0, size=(n, n))
        nu = rng.uniform(-0.1, 0.1, size=(n, n))
        delta0 = gap * (1.0 + 0.1 * u) * np.exp(1j * nu)
        Ax = np.zeros((n, n)); Ay = np.zeros((n, n))
        wl = Workload("cfg0_swave_square", 0, n, n, h, shapes, mask, sym, rot, na, ne, t, kappa, -1,
                      delta0 * mask, Ax, Ay, gap, accelerator=0, n_iterations=20)
    elif cfg in (1, 4):
        ppx = pts_per_xi or 20.0
        R = (10.0 if cfg == 1 else 40.0) * size_scale
        h = 1.0 / ppx
        n = _even_grid(2 * R, h)
        shapes = [disc(R)]
        sym, rot = SYM_S, 0.0
        if cfg == 1:
            na, ne, t, kappa, flux = n_angles or 64, n_energies or 128, 0.1, 2.0, 1.0
            gap = BULK_GAP[("s", 0.1, 128)]
        else:
            na, ne, t, kappa, flux = n_angles or 256, n_energies or 512, 0.05, 2.0, 20.0
            gap = BULK_GAP[("s", 0.05, 512)]
        mask = make_mask(shapes, n, n, h)
        X, Y = grid_xy(n, n, h)
        area = math.pi * R * R
        Bext = math.pi * flux / area                                  # units B0 = Phi0/(pi xi0^2)
        Ax = -0.5 * Bext * Y; Ay = 0.5 * Bext * X                     # symmetric gauge
        if cfg == 1:
            amp = 1.0 + 0.05 * rng.uniform(-1.0, 1.0, size=(n, n))
            chi = _vortex_phase(X, Y, [(0.0, 0.0)])
        else:
            centres = _seeded_vortex_positions(rng, 20, 0.8 * R, 6.0 * size_scale)
            amp = np.ones((n, n))
            chi = _vortex_phase(X, Y, centres)
        delta0 = gap * amp * np.exp(1j * chi)
        wl = Workload(f"cfg{cfg}_swave_disc", cfg, n, n, h, shapes, mask, sym, rot, na, ne, t, kappa, -1,
                      delta0 * mask, Ax, Ay, gap, accelerator=1, n_iterations=10 if cfg == 1 else 3)
    elif cfg in (2, 3):
        ppx = pts_per_xi or 20.0
        side = 20.0 * size_scale
        h = 1.0 / ppx
        ext = side * math.sqrt(2.0)
        n = int(math.ceil(ext / h))
        n += n % 2                                                    # 566 at full size
        shapes = [square(side, 0.125)]
        sym, rot, t = SYM_DX2Y2, 0.0, 0.1
        gap = BULK_GAP[("d", 0.1, 256)]
        mask = make_mask(shapes, n, n, h)
        X, Y = grid_xy(n, n, h)
        Ax = np.zeros((n, n)); Ay = np.zeros((n, n))
        if cfg == 2:
            na, ne, kappa = n_angles or 128, n_energies or 256, 80.0
            u1 = rng.uniform(-1.0, 1.0, size=(n, n)); u2 = rng.uniform(-1.0, 1.0, size=(n, n))
            delta0 = gap + 0.05 * gap * (u1 + 1j * u2)
            wl = Workload("cfg2_dwave_110_square", 2, n, n, h, shapes, mask, sym, rot, na, ne, t, kappa, -1,
                          delta0 * mask, Ax, Ay, gap, accelerator=1, n_iterations=10)
        else:
            na, ne, kappa = n_angles or 128, n_energies or 512, -1.0
            dwall = (0.5 * side - (np.abs(X) + np.abs(Y)) / math.sqrt(2.0))   # distance to the nearest wall
            delta0 = gap * np.tanh(np.clip(dwall, 0.0, None)) + 0j
            eps = -2.0 * gap + 4.0 * gap * np.arange(ne) / (ne - 1)
            wl = Workload("cfg3_ldos_dwave_110_square", 3, n, n, h, shapes, mask, sym, rot, na, ne, t, kappa,
                          -1, delta0 * mask, Ax, Ay, gap, ldos_energies=eps, ldos_broadening=0.01 * gap)
    else:
        raise ValueError(f"unknown config {cfg}")
    return wl


def matsubara(t: float, n: int):
    """eps_n = t (n + 1/2), n = 0..n-1, unit weights (PAPER.md:98 in units of 2 pi kB Tc)."""
    nn = np.arange(n, dtype=np.float64)
    return np.zeros(n), t * (nn + 0.5), np.ones(n)


def make_annulus_workload(r_in: float = 1.53, r_out: float = 4.0, pts_per_xi: float = 5.0, n_angles: int = 16,
                          n_energies: int = 24, t: float = 0.3, kappa: float = 3.0, flux_in_hole: float = 1.0,
                          hole_offset: float = 0.0, seed: int = 7) -> Workload:
    """Multiply-connected grain: a disc with a disc removed ("remove"), threaded
    by `flux_in_hole` flux quanta in the solenoid gauge A = Phi/(2 r) phi-hat (units A0 = Phi0/(pi xi0); the
    paper's annulus benchmarks :563-569), order parameter with the matching winding plus seeded noise.  Lattice
    lines through the hole cross the grain twice: two trajectories per line."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 100 + seed))
    h = 1.0 / pts_per_xi
    n = _even_grid(2 * r_out, h)
    shapes = [disc(r_out), disc(r_in, cx=hole_offset, cy=0.0, add=False)]
    mask = make_mask(shapes, n, n, h)
    X, Y = grid_xy(n, n, h)
    Xc = X - hole_offset
    r2 = np.maximum(Xc * Xc + Y * Y, (0.5 * h) ** 2)
    Ax = -0.5 * flux_in_hole * Y / r2; Ay = 0.5 * flux_in_hole * Xc / r2
    gap = 0.25
    delta0 = gap * (1.0 + 0.05 * rng.uniform(-1, 1, (n, n))) * np.exp(-1j * round(flux_in_hole) * np.arctan2(Y, Xc)
                                                                      + 0.05j * rng.uniform(-1, 1, (n, n)))
    return Workload("annulus_swave_solenoid", -2, n, n, h, shapes, mask, SYM_S, 0.0, n_angles, n_energies, t, kappa, -1,
                    delta0 * mask, Ax, Ay, gap, accelerator=1, n_iterations=5)

