"""Seeded synthetic input generators (gauge links, spinors, sources).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path: it is the
only code the two sides share, and it holds none of the method's arithmetic
(no Dslash, no gamma matrices, no clover, no solver).  It only draws random
numbers and shapes them into the boundary (user-facing) layouts:

  gauge  : float64 array  [T][Z][Y][X][mu=0..3 (x,y,z,t)][row][col][re,im]
  spinor : float64 array  [T][Z][Y][X][spin=0..3][colour=0..2][re,im]

Recipe (BASELINE.json configs[0], SURVEY.md §8(c) readings S5, S6, S8; the paper
itself, /root/reference/PAPER.md, measures on production gauge configurations
 that are not available, so these random SU(3) fields stand in
for them -- see DESIGN.md "Input recipe"):

  * G  : 3x3 complex, Re and Im ~ N(0,1) i.i.d.  (numpy PCG64, default_rng)
  * H  = (G + G^dagger)/2, then H -= tr(H)/3       (traceless Hermitian)
  * U0 = exp(i*eps*H)                               (scaling-and-squaring Taylor)
  * U  = Gram-Schmidt(U0) on rows: r1/|r1|; r2 -= (r1^dag r2) r1, normalise;
         r3 = conj(r1 x r2)          => exactly unitary with det U = 1, and the
         third row is exactly what a 12-real reconstruction rebuilds.
  * spinors: every real component ~ N(0,1).

``dims`` is always (X, Y, Z, T).
"""
from __future__ import annotations

import numpy as np

__all__ = [
    "gauge_field", "tiled_gauge_field", "unit_gauge_field", "spinor_field", "su3_site_field",
    "as_complex", "as_real", "round_to_f32", "chebyshev_sign_coefficients",
]


def as_complex(a: np.ndarray) -> np.ndarray:
    """View a [..., 2] real array as complex [...]."""
    a = np.ascontiguousarray(a)
    if a.dtype == np.float64:
        return a.view(np.complex128)[..., 0]
    if a.dtype == np.float32:
        return a.view(np.complex64)[..., 0]
    raise TypeError(a.dtype)


def as_real(a: np.ndarray) -> np.ndarray:
    """View a complex [...] array as real [..., 2]."""
    a = np.ascontiguousarray(a)
    if a.dtype == np.complex128:
        return a.view(np.float64).reshape(a.shape + (2,))
    if a.dtype == np.complex64:
        return a.view(np.float32).reshape(a.shape + (2,))
    raise TypeError(a.dtype)


def round_to_f32(a: np.ndarray) -> np.ndarray:
    """Round an fp64 field to fp32 and return it again as fp64.

    Used so that an fp64 oracle and an fp32 CUDA run see bit-identical inputs
    (SURVEY.md §8(c) S20)."""
    return a.astype(np.float32).astype(np.float64)


def _expi_hermitian(H: np.ndarray, eps: float) -> np.ndarray:
    """exp(i*eps*H) for a stack of 3x3 matrices, scaling-and-squaring Taylor."""
    A = (1j * eps) * H
    # ||A|| <= eps * ||H||_F ; scale so the series argument is small everywhere
    nrm = float(np.sqrt((np.abs(A) ** 2).sum(axis=(-1, -2)).max())) if A.size else 0.0
    s = 0
    while nrm > 0.25:
        nrm *= 0.5
        s += 1
    A = A / (2.0 ** s)
    eye = np.eye(3, dtype=np.complex128)
    # Horner form of sum_{k<=12} A^k/k!
    E = eye + A / 12.0
    for k in range(11, 0, -1):
        E = eye + np.matmul(A, E) / k
    for _ in range(s):
        E = np.matmul(E, E)
    return E


def _gram_schmidt_rows(U: np.ndarray) -> np.ndarray:
    r1 = U[..., 0, :]
    r2 = U[..., 1, :]
    r1 = r1 / np.sqrt((np.abs(r1) ** 2).sum(-1, keepdims=True))
    r2 = r2 - (np.conj(r1) * r2).sum(-1, keepdims=True) * r1
    r2 = r2 / np.sqrt((np.abs(r2) ** 2).sum(-1, keepdims=True))
    r3 = np.conj(np.cross(r1, r2))
    return np.stack([r1, r2, r3], axis=-2)


def _su3_from_normals(G: np.ndarray, eps: float) -> np.ndarray:
    """G: [..., 3, 3, 2] N(0,1) reals -> SU(3) matrices [..., 3, 3] complex."""
    Gc = as_complex(G)
    H = 0.5 * (Gc + np.conj(np.swapaxes(Gc, -1, -2)))
    tr = np.trace(H, axis1=-2, axis2=-1) / 3.0
    H = H - tr[..., None, None] * np.eye(3)
    return _gram_schmidt_rows(_expi_hermitian(H, eps))


def gauge_field(dims, eps: float, seed: int = 0) -> np.ndarray:
    """Random SU(3) links U_mu(x) = GS(exp(i*eps*H)), boundary layout, fp64.

    Returns float64 [T][Z][Y][X][4][3][3][2].  One time-slice of normals is drawn
    at a time from a single PCG64 stream (so the result does not depend on any
    chunking choice)."""
    X, Y, Z, T = (int(d) for d in dims)
    rng = np.random.default_rng([int(seed), 0])
    out = np.empty((T, Z, Y, X, 4, 3, 3, 2), dtype=np.float64)
    for t in range(T):
        G = rng.standard_normal((Z, Y, X, 4, 3, 3, 2))
        out[t] = as_real(_su3_from_normals(G, eps))
    return out


def tiled_gauge_field(dims, eps: float, seed: int = 0, t_block: int = 16) -> np.ndarray:
    """gauge_field for a (X,Y,Z,t_block) lattice repeated T/t_block times along t.

    Used where the full-size field would take minutes to draw on the host (bench.py and
    the full-size sampled parity tests): every link is still an SU(3) matrix of the recipe
    above and the field is periodic, so it is a valid input of the same distribution; only
    its long-range structure in t repeats.  Falls back to gauge_field when t_block does
    not divide T."""
    X, Y, Z, T = (int(d) for d in dims)
    if t_block >= T or T % t_block:
        return gauge_field(dims, eps, seed)
    blk = gauge_field((X, Y, Z, t_block), eps, seed)
    return np.ascontiguousarray(np.concatenate([blk] * (T // t_block), axis=0))


def unit_gauge_field(dims) -> np.ndarray:
    """U_mu(x) = 1 everywhere (free field), boundary layout."""
    X, Y, Z, T = (int(d) for d in dims)
    out = np.zeros((T, Z, Y, X, 4, 3, 3, 2), dtype=np.float64)
    for a in range(3):
        out[..., a, a, 0] = 1.0
    return out


def su3_site_field(dims, eps: float, seed: int) -> np.ndarray:
    """One random SU(3) matrix per site, complex [T][Z][Y][X][3][3] (gauge
    transformations g(x) for covariance tests)."""
    X, Y, Z, T = (int(d) for d in dims)
    rng = np.random.default_rng([int(seed), 7])
    G = rng.standard_normal((T, Z, Y, X, 3, 3, 2))
    return _su3_from_normals(G, eps)


def spinor_field(dims, seed: int = 0, index: int = 0) -> np.ndarray:
    """Gaussian spinor, every real component ~ N(0,1); float64
    [T][Z][Y][X][4][3][2].  ``index`` selects an independent stream (source,
    second test vector, k-th right-hand side ...)."""
    X, Y, Z, T = (int(d) for d in dims)
    rng = np.random.default_rng([int(seed), 1 + int(index)])
    return rng.standard_normal((T, Z, Y, X, 4, 3, 2))


def chebyshev_sign_coefficients(degree: int = 100, eps2: float = 0.01) -> np.ndarray:
    """Workload parameter for the overlap-kernel configuration (BASELINE.json
    configs[4], reading S16/O8): Chebyshev-Gauss interpolation coefficients of the
    smoothed sign function f(x) = x/sqrt(x^2 + eps2) on [-1, 1],
      N = degree+1, x_j = cos(pi (j+1/2)/N),
      c_k = (2/N) sum_j f(x_j) cos(k pi (j+1/2)/N),  c_0 halved.
    The coefficients are an INPUT of the polynomial driver (both the oracle and the
    CUDA path receive this same array); bandwidth does not depend on them."""
    N = int(degree) + 1
    j = np.arange(N)
    th = np.pi * (j + 0.5) / N
    x = np.cos(th)
    f = x / np.sqrt(x * x + eps2)
    k = np.arange(N)[:, None]
    c = (2.0 / N) * (f[None, :] * np.cos(k * th[None, :])).sum(axis=1)
    c[0] *= 0.5
    return c
