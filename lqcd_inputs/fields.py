"""Synthetic lattice fields in the canonical layout ("Canonical data").

Canonical layout (interchange format of the C ABI, the oracle and the tests):
  * site order   lex = x0 + N0*(x1 + N1*(x2 + N2*x3))      (numerator of PAPER.md:261, Eq. 9)
  * links        U[lex][mu][row][col]  complex128, rows are the paper's r0,r1,r2
  * full spinor  psi[lex][c]           complex128
  * half spinor  of parity p: phi[idxh][c], idxh = lex // 2 over sites with
                 (x0+x1+x2+x3) % 2 == p   (Eq. 9; valid for both
                 parities because N0 is even)

Recipes follow SURVEY.md section 8(c) reading #18 (restated in DESIGN.md):
  * "Haar-like" links (BASELINE.json config 1): complex Gaussian 3x3, Gram-Schmidt,
    determinant fixed to 1.
  * "smooth" links (configs 2-5): U = exp(i*eps*H), H = sum_a w_a lambda_a / sqrt(2),
    w_a ~ N(0,1) -- the paper's momentum distribution exp(-Tr H^2 / 2) --
    then re-unitarised the same way.
  * spinors: Re, Im ~ N(0,1) independently.
All randomness comes from numpy.random.Generator(PCG64) seeded by the caller; draw order is
the canonical array order, links first, spinors after, from the same generator.

The determinant is fixed by rotating the third Gram-Schmidt row by conj(det) -- deliberately
NOT by the wedge-product formula r2 = (r0 ^ r1)* of PAPER.md:272, so that the generator does
not contain (and therefore independently pins) the row-3 reconstruction used by the method.
"""
from __future__ import annotations

import numpy as np

_CHUNK = 1 << 18  # matrices per chunk; bounds temporary memory for the big lattices


def volume(dims) -> int:
    n0, n1, n2, n3 = (int(d) for d in dims)
    return n0 * n1 * n2 * n3


def _check_dims(dims):
    dims = tuple(int(d) for d in dims)
    if len(dims) != 4 or any(d < 2 or d % 2 for d in dims):
        raise ValueError("dims must be four even extents >= 2 (PAPER.md:249, footnote d)")
    return dims


def _as_rng(seed_or_rng):
    if isinstance(seed_or_rng, np.random.Generator):
        return seed_or_rng
    return np.random.default_rng(int(seed_or_rng))


def _inner(a, b):
    """<a,b> = sum_c conj(a_c) b_c over the last axis, keepdims."""
    return np.sum(np.conj(a) * b, axis=-1, keepdims=True)


def _reunitarise(m: np.ndarray) -> np.ndarray:
    """Gram-Schmidt on the rows of m[...,3,3], then det -> 1 by a phase on row 2."""
    r0 = m[..., 0, :]
    r0 = r0 / np.sqrt(_inner(r0, r0).real)
    r1 = m[..., 1, :]
    r1 = r1 - _inner(r0, r1) * r0
    r1 = r1 / np.sqrt(_inner(r1, r1).real)
    r2 = m[..., 2, :]
    r2 = r2 - _inner(r0, r2) * r0 - _inner(r1, r2) * r1
    r2 = r2 / np.sqrt(_inner(r2, r2).real)
    u = np.stack([r0, r1, r2], axis=-2)
    det = np.linalg.det(u)
    u[..., 2, :] *= np.conj(det)[..., None]
    return u


def haar_like_links(dims, seed_or_rng) -> np.ndarray:
    """BASELINE.json config 1 links: Gaussian complex 3x3 -> Gram-Schmidt -> det = 1."""
    dims = _check_dims(dims)
    rng = _as_rng(seed_or_rng)
    n = 4 * volume(dims)
    out = np.empty((n, 3, 3), dtype=np.complex128)
    for lo in range(0, n, _CHUNK):
        hi = min(n, lo + _CHUNK)
        g = rng.standard_normal((hi - lo, 3, 3, 2))
        out[lo:hi] = _reunitarise(g[..., 0] + 1j * g[..., 1])
    return out.reshape(volume(dims), 4, 3, 3)


def _hermitian_from_omega(w: np.ndarray) -> np.ndarray:
    """H = sum_{a=1..8} w_a lambda_a / sqrt(2) with the Gell-Mann matrices lambda_a."""
    h = np.zeros(w.shape[:-1] + (3, 3), dtype=np.complex128)
    s3 = 1.0 / np.sqrt(3.0)
    h[..., 0, 1] = w[..., 0] - 1j * w[..., 1]
    h[..., 1, 0] = w[..., 0] + 1j * w[..., 1]
    h[..., 0, 2] = w[..., 3] - 1j * w[..., 4]
    h[..., 2, 0] = w[..., 3] + 1j * w[..., 4]
    h[..., 1, 2] = w[..., 5] - 1j * w[..., 6]
    h[..., 2, 1] = w[..., 5] + 1j * w[..., 6]
    h[..., 0, 0] = w[..., 2] + s3 * w[..., 7]
    h[..., 1, 1] = -w[..., 2] + s3 * w[..., 7]
    h[..., 2, 2] = -2.0 * s3 * w[..., 7]
    return h / np.sqrt(2.0)


def _expm_small(a: np.ndarray) -> np.ndarray:
    """exp(a) for a batch of 3x3 matrices of modest norm: scaling (2^-4) + Taylor(14) + squaring."""
    a = a / 16.0
    eye = np.broadcast_to(np.eye(3, dtype=np.complex128), a.shape)
    term = eye.copy()
    acc = eye.copy()
    for k in range(1, 15):
        term = np.matmul(term, a) / k
        acc = acc + term
    for _ in range(4):
        acc = np.matmul(acc, acc)
    return acc


def smooth_links(dims, eps: float, seed_or_rng) -> np.ndarray:
    """BASELINE.json configs 2-5 links: U = exp(i*eps*H), re-unitarised."""
    dims = _check_dims(dims)
    rng = _as_rng(seed_or_rng)
    n = 4 * volume(dims)
    out = np.empty((n, 3, 3), dtype=np.complex128)
    for lo in range(0, n, _CHUNK):
        hi = min(n, lo + _CHUNK)
        w = rng.standard_normal((hi - lo, 8))
        out[lo:hi] = _reunitarise(_expm_small(1j * eps * _hermitian_from_omega(w)))
    return out.reshape(volume(dims), 4, 3, 3)


def unit_links(dims) -> np.ndarray:
    """Free field, U = 1 everywhere."""
    dims = _check_dims(dims)
    u = np.zeros((volume(dims), 4, 3, 3), dtype=np.complex128)
    u[..., 0, 0] = u[..., 1, 1] = u[..., 2, 2] = 1.0
    return u


def gaussian_spinor(dims, seed_or_rng) -> np.ndarray:
    """Full-lattice colour vector psi[lex][c], Re and Im ~ N(0,1)."""
    dims = _check_dims(dims)
    rng = _as_rng(seed_or_rng)
    g = rng.standard_normal((volume(dims), 3, 2))
    return np.ascontiguousarray(g[..., 0] + 1j * g[..., 1])


def gaussian_half_spinor(dims, seed_or_rng) -> np.ndarray:
    """Half-lattice colour vector phi[idxh][c] (either parity), Re and Im ~ N(0,1)."""
    dims = _check_dims(dims)
    rng = _as_rng(seed_or_rng)
    g = rng.standard_normal((volume(dims) // 2, 3, 2))
    return np.ascontiguousarray(g[..., 0] + 1j * g[..., 1])


def uniform_backfield(dims, seed_or_rng) -> np.ndarray:
    """Backfield theta[lex][mu] (the paper's unexplained `backfield` argument of acc_Deo, PAPER.md:320-326;
    reading R6 of DESIGN.md: a U(1) phase per link): theta ~ U(-pi, pi) independently -- the phase
    equivalent of Haar-like links; every value of e^{i theta} occurs."""
    dims = _check_dims(dims)
    rng = _as_rng(seed_or_rng)
    return rng.uniform(-np.pi, np.pi, size=(volume(dims), 4))


def rhmc_shifts(n: int = 8, lo_exp: float = -4.0, hi_exp: float = 0.0) -> np.ndarray:
    """BASELINE.json config 4: n shifts log-spaced in [10^lo_exp, 10^hi_exp]."""
    if n == 1:
        return np.array([10.0 ** lo_exp])
    return 10.0 ** (lo_exp + (hi_exp - lo_exp) * np.arange(n) / (n - 1))


def site_coords(dims) -> np.ndarray:
    """coords[lex] = (x0,x1,x2,x3) for the canonical site order."""
    n0, n1, n2, n3 = _check_dims(dims)
    lex = np.arange(n0 * n1 * n2 * n3)
    x0 = lex % n0
    x1 = (lex // n0) % n1
    x2 = (lex // (n0 * n1)) % n2
    x3 = lex // (n0 * n1 * n2)
    return np.stack([x0, x1, x2, x3], axis=1)


def half_index_of_parity(dims, parity: int) -> np.ndarray:
    """lex indices of the sites of the given parity, in idxh = lex//2 order (Eq. 9)."""
    c = site_coords(dims)
    lex = np.nonzero(c.sum(axis=1) % 2 == parity)[0]
    assert np.array_equal(lex // 2, np.arange(lex.size))
    return lex
