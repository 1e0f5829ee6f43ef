"""ctypes wrapper around oracle/staggered_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Argument marshalling only; every number is computed in staggered_oracle.c (plain C99, fp64),
whose header lists the paper passages it follows and the pins that check it.
All arrays are numpy complex128 / float64 in the canonical layout of lqcd_inputs/fields.py.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = C.CDLL(_build.build())

_c128 = np.ctypeslib.ndpointer(dtype=np.complex128, flags="C_CONTIGUOUS")
_i4 = C.c_int * 4
_pd = C.POINTER(C.c_double)
_pi = C.POINTER(C.c_int)

_lib.oracle_dirac_full.argtypes = [_i4, C.c_int, _c128, _c128, _c128, C.c_int]
_lib.oracle_dirac_full.restype = None
_lib.oracle_dirac_range.argtypes = [_i4, C.c_int, _c128, _c128, _c128, C.c_longlong, C.c_longlong]
_lib.oracle_dirac_range.restype = None
_lib.oracle_dirac_site.argtypes = [_i4, C.c_int, _c128, _c128, _i4, _c128]
_lib.oracle_dirac_site.restype = None
_lib.oracle_half_to_full.argtypes = [_i4, C.c_int, _c128, _c128]
_lib.oracle_half_to_full.restype = None
_lib.oracle_full_to_half.argtypes = [_i4, C.c_int, _c128, _c128]
_lib.oracle_full_to_half.restype = None
_lib.oracle_dslash_half.argtypes = [_i4, C.c_int, _c128, C.c_int, _c128, _c128]
_lib.oracle_dslash_half.restype = C.c_int
_lib.oracle_mdagm.argtypes = [_i4, C.c_int, _c128, C.c_double, C.c_double, _c128, _c128]
_lib.oracle_mdagm.restype = C.c_int
_lib.oracle_reconstruct_row3_field.argtypes = [_c128, C.c_size_t]
_lib.oracle_reconstruct_row3_field.restype = None
_lib.oracle_cg.argtypes = [_i4, C.c_int, _c128, C.c_double, _c128, _c128, C.c_double, C.c_int,
                           _pi, _pd, _pd, _pd, _pd, C.c_int]
_lib.oracle_cg.restype = C.c_int
_lib.oracle_cg_multishift.argtypes = [_i4, C.c_int, _c128, C.c_double, C.c_int, _pd, _c128, _c128,
                                      C.c_double, C.c_int, _pi, _pi, _pd, _pd, C.c_void_p,
                                      _pd, _pd, _pd, C.c_int]
_lib.oracle_cg_multishift.restype = C.c_int
_lib.oracle_rational_apply.argtypes = [_i4, C.c_int, _c128, C.c_double, C.c_int, _pd, C.c_double, _pd, _c128, _c128,
                                       C.c_double, C.c_int, _pi, _pi]
_lib.oracle_rational_apply.restype = C.c_int
_lib.oracle_fermion_force.argtypes = [_i4, C.c_int, _c128, C.c_int, _pd, _c128, _c128]
_lib.oracle_fermion_force.restype = C.c_int
_lib.oracle_gauge_staples.argtypes = [_i4, _c128, C.c_double, C.c_double, _c128]
_lib.oracle_gauge_staples.restype = None
# *_bf: the same functions with the optional backfield theta[V][4] (float64; NULL = none) after U
_lib.oracle_dirac_full_bf.argtypes = [_i4, C.c_int, _c128, C.c_void_p, _c128, _c128, C.c_int]
_lib.oracle_dirac_full_bf.restype = None
_lib.oracle_dirac_site_bf.argtypes = [_i4, C.c_int, _c128, C.c_void_p, _c128, _i4, _c128]
_lib.oracle_dirac_site_bf.restype = None
_lib.oracle_dslash_half_bf.argtypes = [_i4, C.c_int, _c128, C.c_void_p, C.c_int, _c128, _c128]
_lib.oracle_dslash_half_bf.restype = C.c_int
_lib.oracle_mdagm_bf.argtypes = [_i4, C.c_int, _c128, C.c_void_p, C.c_double, C.c_double, _c128, _c128]
_lib.oracle_mdagm_bf.restype = C.c_int
_lib.oracle_cg_bf.argtypes = [_i4, C.c_int, _c128, C.c_void_p, C.c_double, _c128, _c128, C.c_double, C.c_int,
                              _pi, _pd, _pd, _pd, _pd, C.c_int]
_lib.oracle_cg_bf.restype = C.c_int
_lib.oracle_cg_multishift_bf.argtypes = [_i4, C.c_int, _c128, C.c_void_p, C.c_double, C.c_int, _pd, _c128, _c128,
                                         C.c_double, C.c_int, _pi, _pi, _pd, _pd, C.c_void_p,
                                         _pd, _pd, _pd, C.c_int]
_lib.oracle_cg_multishift_bf.restype = C.c_int
_lib.oracle_fermion_force_bf.argtypes = [_i4, C.c_int, _c128, C.c_void_p, C.c_int, _pd, _c128, _c128]
_lib.oracle_fermion_force_bf.restype = C.c_int
_lib.oracle_num_threads.restype = C.c_int
_lib.oracle_set_num_threads.argtypes = [C.c_int]


def _dims(dims):
    dims = [int(d) for d in dims]
    if len(dims) != 4 or any(d < 2 or d % 2 for d in dims):
        raise ValueError("dims must be four even extents >= 2")
    return _i4(*dims), dims[0] * dims[1] * dims[2] * dims[3]


def _arr(a, shape):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    if a.shape != shape:
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


def _dptr(a):
    return a.ctypes.data_as(_pd)


class _Theta:
    """The optional backfield theta[V][4] (float64) as a void* argument; keeps the array alive."""

    def __init__(self, theta, V):
        self.a = None
        if theta is not None:
            self.a = np.ascontiguousarray(theta, dtype=np.float64)
            if self.a.shape != (V, 4):
                raise ValueError(f"backfield must have shape ({V}, 4), got {self.a.shape}")

    @property
    def ptr(self):
        return None if self.a is None else C.c_void_p(self.a.ctypes.data)


def num_threads() -> int:
    return int(_lib.oracle_num_threads())


def set_num_threads(n: int) -> None:
    _lib.oracle_set_num_threads(int(n))


def dirac_full(dims, U, psi, antiperiodic_t=True, which=2, theta=None):
    """(D psi)(x) on the whole lattice (which=2) or on one parity (0 even, 1 odd; rest zero).
    theta: optional backfield [V][4] (every link enters as e^{i theta} U); None calls the plain entry point."""
    n4, V = _dims(dims)
    out = np.zeros((V, 3), dtype=np.complex128)
    if theta is None:
        _lib.oracle_dirac_full(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), _arr(psi, (V, 3)), out, which)
    else:
        th = _Theta(theta, V)
        _lib.oracle_dirac_full_bf(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), th.ptr, _arr(psi, (V, 3)), out, which)
    return out


def dirac_range(dims, U, psi, out, lo, hi, antiperiodic_t=True):
    """out[lo:hi] = (D psi)(lex) for lex in [lo, hi); `out` is a caller-provided (V,3) array."""
    n4, V = _dims(dims)
    assert out.shape == (V, 3) and out.dtype == np.complex128 and 0 <= lo <= hi <= V
    _lib.oracle_dirac_range(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), _arr(psi, (V, 3)), out, lo, hi)
    return out


def dirac_site(dims, U, psi, x, antiperiodic_t=True, theta=None):
    n4, V = _dims(dims)
    out = np.zeros(3, dtype=np.complex128)
    if theta is None:
        _lib.oracle_dirac_site(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), _arr(psi, (V, 3)),
                               _i4(*[int(c) for c in x]), out)
    else:
        th = _Theta(theta, V)
        _lib.oracle_dirac_site_bf(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), th.ptr, _arr(psi, (V, 3)),
                                  _i4(*[int(c) for c in x]), out)
    return out


def half_to_full(dims, parity, half):
    n4, V = _dims(dims)
    full = np.empty((V, 3), dtype=np.complex128)
    _lib.oracle_half_to_full(n4, parity, _arr(half, (V // 2, 3)), full)
    return full


def full_to_half(dims, parity, full):
    n4, V = _dims(dims)
    half = np.empty((V // 2, 3), dtype=np.complex128)
    _lib.oracle_full_to_half(n4, parity, _arr(full, (V, 3)), half)
    return half


def dslash_half(dims, U, out_parity, in_half, antiperiodic_t=True, theta=None):
    """out_parity=0: D_eo in_o (even output); out_parity=1: D_oe in_e (odd output)."""
    n4, V = _dims(dims)
    out = np.empty((V // 2, 3), dtype=np.complex128)
    if theta is None:
        rc = _lib.oracle_dslash_half(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), out_parity,
                                     _arr(in_half, (V // 2, 3)), out)
    else:
        th = _Theta(theta, V)
        rc = _lib.oracle_dslash_half_bf(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), th.ptr, out_parity,
                                        _arr(in_half, (V // 2, 3)), out)
    if rc:
        raise MemoryError("oracle_dslash_half")
    return out


def mdagm(dims, U, mass, in_e, sigma=0.0, antiperiodic_t=True, theta=None):
    """(m^2 + sigma) in_e - D_eo D_oe in_e."""
    n4, V = _dims(dims)
    out = np.empty((V // 2, 3), dtype=np.complex128)
    if theta is None:
        rc = _lib.oracle_mdagm(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), mass, sigma,
                               _arr(in_e, (V // 2, 3)), out)
    else:
        th = _Theta(theta, V)
        rc = _lib.oracle_mdagm_bf(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), th.ptr, mass, sigma,
                                  _arr(in_e, (V // 2, 3)), out)
    if rc:
        raise MemoryError("oracle_mdagm")
    return out


def reconstruct_row3(U):
    """Copy of U with row 2 of every matrix replaced by (r0 ^ r1)^*."""
    out = np.array(U, dtype=np.complex128, order="C", copy=True)
    _lib.oracle_reconstruct_row3_field(out.reshape(-1), out.size // 9)
    return out


def cg(dims, U, mass, b, tol, max_iter, antiperiodic_t=True, hist_len=0, theta=None):
    """Returns dict(x, iters, converged, true_relres, alpha, beta, rnorm)."""
    n4, V = _dims(dims)
    x = np.empty((V // 2, 3), dtype=np.complex128)
    iters = C.c_int(0)
    relres = C.c_double(0.0)
    ha = np.zeros(max(hist_len, 1))
    hb = np.zeros(max(hist_len, 1))
    hr = np.zeros(max(hist_len, 1))
    if theta is None:
        rc = _lib.oracle_cg(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), mass, _arr(b, (V // 2, 3)), x,
                            tol, max_iter, C.byref(iters), C.byref(relres),
                            _dptr(ha), _dptr(hb), _dptr(hr), hist_len)
    else:
        th = _Theta(theta, V)
        rc = _lib.oracle_cg_bf(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), th.ptr, mass, _arr(b, (V // 2, 3)), x,
                               tol, max_iter, C.byref(iters), C.byref(relres),
                               _dptr(ha), _dptr(hb), _dptr(hr), hist_len)
    if rc < 0:
        raise MemoryError("oracle_cg")
    return dict(x=x, iters=iters.value, converged=(rc == 0), true_relres=relres.value,
                alpha=ha[:hist_len], beta=hb[:hist_len], rnorm=hr[:hist_len])


def cg_multishift(dims, U, mass, shifts, b, tol, max_iter, antiperiodic_t=True, hist_len=0, theta=None):
    """Returns dict(x[nshift], iters, converged, conv_iter, true_relres, zeta, r, alpha, beta, rnorm)."""
    n4, V = _dims(dims)
    shifts = np.ascontiguousarray(shifts, dtype=np.float64)
    ns = shifts.size
    x = np.empty((ns, V // 2, 3), dtype=np.complex128)
    r = np.empty((V // 2, 3), dtype=np.complex128)
    iters = C.c_int(0)
    conv = (C.c_int * ns)()
    relres = np.zeros(ns)
    zeta = np.zeros(ns)
    ha = np.zeros(max(hist_len, 1))
    hb = np.zeros(max(hist_len, 1))
    hr = np.zeros(max(hist_len, 1))
    if theta is None:
        rc = _lib.oracle_cg_multishift(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), mass, ns, _dptr(shifts),
                                       _arr(b, (V // 2, 3)), x.reshape(-1), tol, max_iter,
                                       C.byref(iters), conv, _dptr(relres), _dptr(zeta),
                                       r.ctypes.data_as(C.c_void_p),
                                       _dptr(ha), _dptr(hb), _dptr(hr), hist_len)
    else:
        th = _Theta(theta, V)
        rc = _lib.oracle_cg_multishift_bf(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), th.ptr, mass, ns, _dptr(shifts),
                                          _arr(b, (V // 2, 3)), x.reshape(-1), tol, max_iter,
                                          C.byref(iters), conv, _dptr(relres), _dptr(zeta),
                                          r.ctypes.data_as(C.c_void_p),
                                          _dptr(ha), _dptr(hb), _dptr(hr), hist_len)
    if rc == -1:
        raise MemoryError("oracle_cg_multishift")
    if rc == -2:
        raise ValueError("shifts must be >= 0 and nshift >= 1")
    return dict(x=x, iters=iters.value, converged=(rc == 0), conv_iter=np.array(list(conv)),
                true_relres=relres, zeta=zeta, r=r,
                alpha=ha[:hist_len], beta=hb[:hist_len], rnorm=hr[:hist_len])


def rational_apply(dims, U, mass, shifts, c0, coeffs, b, tol, max_iter, antiperiodic_t=True):
    """y = c0 b + sum_i coeffs[i] (A + shifts[i])^-1 b.  Returns dict(y, iters, converged, conv_iter)."""
    n4, V = _dims(dims)
    shifts = np.ascontiguousarray(shifts, dtype=np.float64)
    coeffs = np.ascontiguousarray(coeffs, dtype=np.float64)
    ns = shifts.size
    if coeffs.size != ns:
        raise ValueError("one coefficient per shift")
    y = np.empty((V // 2, 3), dtype=np.complex128)
    iters = C.c_int(0)
    conv = (C.c_int * ns)()
    rc = _lib.oracle_rational_apply(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), mass, ns, _dptr(shifts),
                                    float(c0), _dptr(coeffs), _arr(b, (V // 2, 3)), y, tol, max_iter,
                                    C.byref(iters), conv)
    if rc == -1:
        raise MemoryError("oracle_rational_apply")
    if rc == -2:
        raise ValueError("shifts must be >= 0 and nshift >= 1")
    return dict(y=y, iters=iters.value, converged=(rc == 0), conv_iter=np.array(list(conv)))


def fermion_force(dims, U, coeffs, xs, antiperiodic_t=True, theta=None):
    """F[V,4,3,3] = TA[U_mu(x) Q_mu(x)] from the solutions xs[nshift, V/2, 3] (even sites) and c_i.
    theta: optional backfield [V][4] (links e^{i theta} U in D and in the force)."""
    n4, V = _dims(dims)
    coeffs = np.ascontiguousarray(coeffs, dtype=np.float64)
    xs = np.ascontiguousarray(xs, dtype=np.complex128)
    if xs.shape != (coeffs.size, V // 2, 3):
        raise ValueError(f"xs must be ({coeffs.size}, {V // 2}, 3)")
    F = np.empty((V, 4, 3, 3), dtype=np.complex128)
    if theta is None:
        rc = _lib.oracle_fermion_force(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), coeffs.size, _dptr(coeffs),
                                       xs.reshape(-1), F.reshape(-1))
    else:
        th = _Theta(theta, V)
        rc = _lib.oracle_fermion_force_bf(n4, int(antiperiodic_t), _arr(U, (V, 4, 3, 3)), th.ptr, coeffs.size,
                                          _dptr(coeffs), xs.reshape(-1), F.reshape(-1))
    if rc:
        raise MemoryError("oracle_fermion_force")
    return F


SYMANZIK_C0, SYMANZIK_C1 = 5.0 / 3.0, -1.0 / 12.0


def gauge_staples(dims, U, c0=SYMANZIK_C0, c1=SYMANZIK_C1):
    """S[V,4,3,3]: staples of the tree-level Symanzik action (plaquette x c0 + 2x1 rectangles x c1)."""
    n4, V = _dims(dims)
    S = np.empty((V, 4, 3, 3), dtype=np.complex128)
    _lib.oracle_gauge_staples(n4, _arr(U, (V, 4, 3, 3)), float(c0), float(c1), S.reshape(-1))
    return S
