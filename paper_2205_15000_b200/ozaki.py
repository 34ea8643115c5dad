"""Ozaki's continued-fraction pole table for Fermi-function (Matsubara) sums — host-side input generator.

PAPER.md:207: "The frequency summations are not over the usual Matsubara frequencies, but instead a more efficient
summation due to Ozaki" (ref. 77, T. Ozaki, Phys. Rev. B 75, 035123 (2007)).  The paper prints no table; the poles
follow from the published construction: the continued fraction of tanh turns 1/(1 + e^x) into

    f(x) = 1/2 - sum_{p=1}^{N} R_p [ 1/(x - i/b_p) + 1/(x + i/b_p) ],

where +-b_p are the eigenvalues of the symmetric tridiagonal matrix B (size 2N, zero diagonal,
B_{n,n+1} = 1 / (2 sqrt((2n-1)(2n+1))), n = 1..2N-1) and R_p = |v_p[0]|^2 / (4 b_p^2) with v_p the normalised
eigenvector.  A Matsubara sum T sum_n F(i eps_n) over eps_n = pi T (2n+1) (poles of f at x = i pi (2n+1), residue -1)
becomes T sum_p R_p F(i T / b_p): the lowest poles coincide with Matsubara frequencies to machine precision
(R_p = 1), the last few spread out with large weights and stand in for the whole tail.

The library takes energies and weights as data (`sc_set_energies`), so this module only builds the arrays; it is
pinned against the exact Fermi function in tests/test_host_logic.py.
"""
from __future__ import annotations

import numpy as np


def ozaki_poles(n_poles: int):
    """(xi_p, R_p), p = 1..n_poles: f(x) ~ 1/2 - sum_p R_p [1/(x - i xi_p) + 1/(x + i xi_p)], xi_p = 1/b_p ascending."""
    if n_poles < 1:
        raise ValueError("n_poles < 1")
    m = 2 * n_poles
    n = np.arange(1, m, dtype=np.float64)
    off = 0.5 / np.sqrt((2.0 * n - 1.0) * (2.0 * n + 1.0))
    B = np.diag(off, 1) + np.diag(off, -1)
    lam, vec = np.linalg.eigh(B)
    pos = lam > 0
    b = lam[pos]; v0 = vec[0, pos]
    xi = 1.0 / b
    R = (v0 * v0) / (4.0 * b * b)
    order = np.argsort(xi)
    return xi[order], R[order]


def ozaki_energy_table(t: float, n_poles: int):
    """(z, w) for `sc_set_energies` in the library's units (energies in 2 pi k_B T_c, t = T/T_c): z_p = i t xi_p / (2 pi)
    — the Matsubara table is z_n = i t (n + 1/2) = i t pi (2n+1) / (2 pi) with unit weights — and w_p = R_p."""
    xi, R = ozaki_poles(n_poles)
    return 1j * t * xi / (2.0 * np.pi), R
