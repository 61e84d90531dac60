"""Gridding-convolution-function (GCF) tables used as *inputs* by the tests and the bench.

PAPER.md:179 (section 5) says only "a spheroidal function from [24]".  The reading taken
(R4): the zero-order prolate spheroidal wave function psi_0(c, eta) with
eta = 2 r / S on the support |r| <= S/2 cells and c = pi S / 2, normalised to psi_0(0) = 1.
It is computed here from its definition: the eigenfunction of the band-limiting integral operator
int_{-1}^{1} sin(c (x - y)) / (pi (x - y)) psi(y) dy = lambda psi(x)  with the largest lambda,
obtained through the commuting prolate differential operator in a Legendre basis (double
precision), and checked in tests against scipy.special.pro_ang1.  No coefficient tables from
any third party are used.  Parity never depends on these values (the table is an argument of
the gridder); only the imaging invariant P4 does, and it takes its correction from the table.
"""
from __future__ import annotations

import functools

import numpy as np


@functools.lru_cache(maxsize=None)
def _pswf_legendre_coeffs(c: float, n_terms: int = 96) -> np.ndarray:
    """Coefficients of psi_0(c, .) in the Legendre basis P_0, P_2, P_4, ...

    psi_0 is the eigenfunction with the smallest eigenvalue chi of the prolate operator
    L psi = -((1 - x^2) psi')' + c^2 x^2 psi  on [-1, 1], which commutes with the band-limiting
    integral operator; unlike the integral operator (whose leading ~2c/pi eigenvalues are all 1 to
    machine precision) its spectrum is well separated, so this stays accurate for c = 8 pi.
    L P_k = k (k + 1) P_k + c^2 x^2 P_k; the matrix of x^2 in the orthonormal Legendre basis is
    formed by Gauss-Legendre quadrature (exact for these polynomial degrees).
    """
    degs = 2 * np.arange(n_terms)
    t, wt = np.polynomial.legendre.leggauss(2 * n_terms + 8)
    basis = np.stack([np.polynomial.legendre.legval(t, np.eye(1, int(k) + 1, int(k))[0]) * np.sqrt(k + 0.5)
                      for k in degs])                       # orthonormal P_k at the nodes
    x2 = (basis * (wt * t * t)[None, :]) @ basis.T
    a = np.diag((degs * (degs + 1)).astype(np.float64)) + c * c * x2
    chi, vec = np.linalg.eigh(a)
    beta = vec[:, 0] * np.sqrt(degs + 0.5)                  # back to plain P_k coefficients
    full = np.zeros(2 * n_terms)
    full[degs] = beta
    return full


def pswf0(c: float, eta: np.ndarray) -> np.ndarray:
    """psi_0(c, eta) for |eta| <= 1, normalised so that psi_0(c, 0) = 1."""
    coef = _pswf_legendre_coeffs(float(c))
    eta = np.asarray(eta, dtype=np.float64)
    return np.polynomial.legendre.legval(eta, coef) / np.polynomial.legendre.legval(0.0, coef)


def spheroidal_1d(support: int, oversample: int) -> np.ndarray:
    """1-D oversampled table T1[j], j = 0..S*O-1, sample j at r = (j - S*O/2)/O cells (float64)."""
    s, o = int(support), int(oversample)
    j = np.arange(s * o, dtype=np.float64)
    r = (j - (s * o) / 2.0) / o
    return pswf0(np.pi * s / 2.0, 2.0 * r / s)


def spheroidal_table(support: int, oversample: int) -> np.ndarray:
    """Separable real table K[jy][jx] = T1[jy] * T1[jx], float32, shape [S*O, S*O]."""
    t1 = spheroidal_1d(support, oversample)
    return np.outer(t1, t1).astype(np.float32)


def wplane_supports(n_planes: int = 32) -> list[int]:
    """Config 3 reading (R13): S_p = 2*round(4 + 12 p / (P-1)) = 8, 8, 10, ..., 32, 32."""
    return [2 * int(np.floor(4.0 + 12.0 * p / (n_planes - 1) + 0.5)) for p in range(n_planes)]


def wplane_tables(supports: list[int], oversample: int) -> np.ndarray:
    """Plane-major complex64 tables, flattened to float32 pairs.

    Plane p is [S_p*O][S_p*O] samples of  psi(ry) psi(rx) * exp(i * pi * kappa_p * (rx^2 + ry^2))
    with kappa_p = p / (P * S_p): a spheroidal taper times a Fresnel chirp whose curvature grows
    with the plane index -- a smooth complex table of the right shapes.  BASELINE.json's config 3
    fixes the shapes only; parity is table-agnostic (input recipe).
    """
    out = []
    n_planes = len(supports)
    for p, s in enumerate(supports):
        t1 = spheroidal_1d(s, oversample)
        j = np.arange(s * oversample, dtype=np.float64)
        r = (j - (s * oversample) / 2.0) / oversample
        kappa = p / (n_planes * s)
        chirp = np.exp(1j * np.pi * kappa * (r[:, None] ** 2 + r[None, :] ** 2))
        plane = (np.outer(t1, t1) * chirp).astype(np.complex64)
        out.append(plane.view(np.float32).ravel())
    return np.concatenate(out)
