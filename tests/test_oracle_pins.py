"""Pins for the CPU oracle (-m "not gpu").

The paper prints no worked numerical example for this path, so each
pin is something the mathematics fixes independently of oracle/staggered_oracle.c:
a dense matrix built from the definition in numpy, closed forms, invariants and dense solves.
Each test names the mistake it would catch.
"""
import numpy as np
import pytest

import lqcd_inputs as gen
import oracle
from dense_reference import dense_dirac, dense_normal_operator, parity_mask


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


# ----------------------------------------------------------------------------------------------
# Operator: dense brute force (stencil, phases, BC, N=2 wrap, dagger, 1/2)
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 4, 4, 4), (4, 2, 6, 2)])
@pytest.mark.parametrize("ap", [True, False])
def test_dirac_matches_dense_matrix(dims, ap):
    rng = np.random.default_rng(1)
    U = gen.haar_like_links(dims, rng)
    psi = gen.gaussian_spinor(dims, rng)
    D = dense_dirac(dims, U, ap)
    want = (D @ psi.reshape(-1)).reshape(-1, 3)
    got = oracle.dirac_full(dims, U, psi, antiperiodic_t=ap)
    assert rel(got, want) < 1e-14
    # structure of the dense matrix itself: anti-Hermitian, no even-even / odd-odd block (Eq. 7)
    assert np.abs(D + D.conj().T).max() == 0.0
    par = np.repeat(parity_mask(dims), 3)
    assert np.abs(D[np.ix_(par == 0, par == 0)]).max() == 0.0
    assert np.abs(D[np.ix_(par == 1, par == 1)]).max() == 0.0


def test_dirac_columns_at_2x4():
    """oracle . e_j = column j of the dense matrix, every j (BASELINE.json config 1, 2^4)."""
    dims = (2, 2, 2, 2)
    U = gen.haar_like_links(dims, 1)
    D = dense_dirac(dims, U, True)
    V = gen.volume(dims)
    for j in range(3 * V):
        e = np.zeros(3 * V, dtype=np.complex128)
        e[j] = 1.0
        col = oracle.dirac_full(dims, U, e.reshape(V, 3)).reshape(-1)
        assert np.abs(col - D[:, j]).max() < 1e-15


@pytest.mark.parametrize("ap", [True, False])
def test_dirac_site_is_the_dense_row_at_every_site(ap):
    """oracle.dirac_site(x) (the checker of the large-volume sampled GPU parity tests) = rows
    3*lex(x)..3*lex(x)+2 of the dense matrix applied to psi, for EVERY site of 4x2x6x2 (N_mu = 2 wraps in
    two directions), both boundary conditions.  Catches a coordinate-order slip in the wrapper."""
    dims = (4, 2, 6, 2)
    rng = np.random.default_rng(21)
    U = gen.haar_like_links(dims, rng)
    psi = gen.gaussian_spinor(dims, rng)
    want = (dense_dirac(dims, U, ap) @ psi.reshape(-1)).reshape(-1, 3)
    coords = gen.site_coords(dims)
    for lex in range(gen.volume(dims)):
        got = oracle.dirac_site(dims, U, psi, coords[lex], antiperiodic_t=ap)
        assert np.abs(got - want[lex]).max() < 1e-14, (lex, coords[lex])


@pytest.mark.parametrize("ap", [True, False])
def test_dirac_range_fills_exactly_lo_hi(ap):
    """oracle.dirac_range(lo, hi) (what bench.py's CPU legs time) writes the dense-matrix values to
    exactly [lo, hi) and leaves a NaN-prefilled remainder untouched: an off-by-one at either end, or a
    loop over the wrong range, fails here."""
    dims = (4, 2, 6, 2)
    rng = np.random.default_rng(22)
    U = gen.haar_like_links(dims, rng)
    psi = gen.gaussian_spinor(dims, rng)
    V = gen.volume(dims)
    want = (dense_dirac(dims, U, ap) @ psi.reshape(-1)).reshape(-1, 3)
    for lo, hi in [(0, V), (0, 1), (V - 1, V), (5, 5), (7, 40), (1, V - 1), (48, 49)]:
        out = np.full((V, 3), np.nan + 1j * np.nan)
        oracle.dirac_range(dims, U, psi, out, lo, hi, antiperiodic_t=ap)
        assert np.isnan(out[:lo]).all() and np.isnan(out[hi:]).all(), (lo, hi)
        if hi > lo:
            assert np.abs(out[lo:hi] - want[lo:hi]).max() < 1e-14, (lo, hi)
    # and the three entry points agree bit for bit (same static function underneath)
    full = oracle.dirac_full(dims, U, psi, antiperiodic_t=ap)
    out = np.zeros((V, 3), dtype=np.complex128)
    oracle.dirac_range(dims, U, psi, out, 0, V, antiperiodic_t=ap)
    assert np.array_equal(out, full)


# ----------------------------------------------------------------------------------------------
# Backfield (the fourth argument of the paper's acc_Deo; reading R6: a U(1) phase
# per link, every link enters D as e^{i theta_mu(x)} U_mu(x))
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 6, 2), (4, 4, 4, 4)])
@pytest.mark.parametrize("ap", [True, False])
def test_backfield_dense_matrix_zero_field_and_absorbed_phases(dims, ap):
    """(i) theta = 0 reproduces D bit for bit; (ii) random theta = the dense matrix built from phased links
    (wrong sign of the backward phase, phase taken at x instead of x-mu, or a phase on psi instead of on the
    link all fail here; N_mu = 2 included); (iii) the phases absorbed into the links, U -> e^{i theta} U, give
    the same result through the PLAIN (already pinned) entry point; (iv) D stays anti-Hermitian."""
    rng = np.random.default_rng(31)
    U = gen.haar_like_links(dims, rng)
    psi = gen.gaussian_spinor(dims, rng)
    theta = gen.uniform_backfield(dims, rng)
    V = gen.volume(dims)
    plain = oracle.dirac_full(dims, U, psi, antiperiodic_t=ap)
    assert np.array_equal(oracle.dirac_full(dims, U, psi, antiperiodic_t=ap, theta=np.zeros((V, 4))), plain)
    D = dense_dirac(dims, U, ap, theta)
    assert np.abs(D + D.conj().T).max() < 1e-16
    got = oracle.dirac_full(dims, U, psi, antiperiodic_t=ap, theta=theta)
    assert rel(got, (D @ psi.reshape(-1)).reshape(-1, 3)) < 1e-14
    assert rel(got, plain) > 0.1                                   # the field does something
    absorbed = U * np.exp(1j * theta)[:, :, None, None]
    assert rel(got, oracle.dirac_full(dims, absorbed, psi, antiperiodic_t=ap)) < 1e-14
    # the single-site and half-lattice entry points see the same field
    coords = gen.site_coords(dims)
    for lex in (0, 1, V // 2 + 1, V - 1):
        assert np.abs(oracle.dirac_site(dims, U, psi, coords[lex], antiperiodic_t=ap, theta=theta) - got[lex]).max() < 1e-15
    for par in (0, 1):
        half_in = oracle.full_to_half(dims, 1 - par, psi)
        want = oracle.full_to_half(dims, par, got)
        assert rel(oracle.dslash_half(dims, U, par, half_in, antiperiodic_t=ap, theta=theta), want) < 1e-14


def test_backfield_constant_phase_shifts_the_free_momenta():
    """U = 1, theta_mu(x) = t_mu constant: plane waves on even sites are eigenvectors of A with eigenvalue
    m^2 + sum_mu sin^2(p_mu + t_mu) -- a momentum shift p -> p + t.  Catches a phase applied with the same
    sign to both hops (which would give sin^2 p scaled, not shifted) and a factor 2 in the phase."""
    dims = (4, 4, 6, 4)
    U = gen.unit_links(dims)
    m = 0.37
    t = np.array([0.3, -0.45, 1.1, 0.2])
    theta = np.tile(t, (gen.volume(dims), 1))
    xe = gen.site_coords(dims)[gen.half_index_of_parity(dims, 0)]
    colour = np.array([0.3 - 0.2j, 1.0 + 0.5j, -0.7j])
    for n in [(0, 0, 0, 0), (1, 0, 0, 0), (0, 1, 2, 1), (3, 2, 5, 3)]:
        p = np.array([2 * np.pi * n[0] / dims[0], 2 * np.pi * n[1] / dims[1],
                      2 * np.pi * n[2] / dims[2], (2 * n[3] + 1) * np.pi / dims[3]])
        phi = np.exp(1j * (xe @ p))[:, None] * colour[None, :]
        lam = m * m + np.sum(np.sin(p + t) ** 2)
        assert rel(oracle.mdagm(dims, U, m, phi, theta=theta), lam * phi) < 1e-13


def test_backfield_pure_gauge_is_removed_by_a_u1_transformation():
    """theta_mu(x) = a(x) - a(x+mu) (periodic a): D[U, theta] (g psi) = g D[U, 0] psi with g(x) = e^{i a(x)}.
    Catches a phase attached to the wrong end of the link."""
    dims = (4, 6, 2, 4)
    rng = np.random.default_rng(33)
    U = gen.smooth_links(dims, 0.5, rng)
    psi = gen.gaussian_spinor(dims, rng)
    V = gen.volume(dims)
    a = rng.uniform(-np.pi, np.pi, size=V)
    coords = gen.site_coords(dims)
    theta = np.empty((V, 4))
    for mu in range(4):
        c = coords.copy()
        c[:, mu] = (c[:, mu] + 1) % dims[mu]
        fwd = c[:, 0] + dims[0] * (c[:, 1] + dims[1] * (c[:, 2] + dims[2] * c[:, 3]))
        theta[:, mu] = a - a[fwd]
    g = np.exp(1j * a)[:, None]
    for ap in (True, False):
        lhs = oracle.dirac_full(dims, U, g * psi, antiperiodic_t=ap, theta=theta)
        assert rel(lhs, g * oracle.dirac_full(dims, U, psi, antiperiodic_t=ap)) < 1e-14


def test_backfield_normal_operator_and_solvers():
    """mdagm / CG / multi-shift CG with a backfield: the dense A built from phased links (Hermitian, spectrum
    >= m^2), dense solves, and the absorbed-phase equivalence with the plain (pinned) solvers iteration by
    iteration."""
    dims = (4, 4, 2, 4)
    rng = np.random.default_rng(34)
    U = gen.smooth_links(dims, 0.4, rng)
    theta = gen.uniform_backfield(dims, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m = 0.2
    A, _, _ = dense_normal_operator(dims, U, m, True, theta)
    assert np.abs(A - A.conj().T).max() < 1e-15 and np.linalg.eigvalsh(A).min() >= m * m - 1e-12
    assert rel(oracle.mdagm(dims, U, m, b, sigma=0.3, theta=theta).reshape(-1),
               (A + 0.3 * np.eye(A.shape[0])) @ b.reshape(-1)) < 1e-13
    r = oracle.cg(dims, U, m, b, 1e-12, 2000, theta=theta, hist_len=8)
    assert r["converged"] and rel(r["x"].reshape(-1), np.linalg.solve(A, b.reshape(-1))) < 1e-10
    absorbed = U * np.exp(1j * theta)[:, :, None, None]
    r0 = oracle.cg(dims, absorbed, m, b, 1e-12, 2000, hist_len=8)
    assert abs(r0["iters"] - r["iters"]) <= 2 and np.allclose(r0["alpha"], r["alpha"], rtol=1e-11)
    assert np.allclose(r0["rnorm"], r["rnorm"], rtol=1e-11) and rel(r0["x"], r["x"]) < 1e-9
    shifts = np.array([0.7, 0.0, 0.05])
    ms = oracle.cg_multishift(dims, U, m, shifts, b, 1e-12, 2000, theta=theta)
    assert ms["converged"]
    for i, s in enumerate(shifts):
        assert rel(ms["x"][i].reshape(-1), np.linalg.solve(A + s * np.eye(A.shape[0]), b.reshape(-1))) < 1e-10
    assert rel(oracle.cg(dims, U, m, b, 1e-12, 2000).get("x"), r["x"]) > 1e-2       # and it is not the plain solve


def test_half_lattice_views_and_parity_naming():
    """dslash_half(out_parity) = the (out, in) block of the dense matrix (reading R5)."""
    dims = (4, 4, 2, 4)
    rng = np.random.default_rng(7)
    U = gen.haar_like_links(dims, rng)
    _, D_eo, D_oe = dense_normal_operator(dims, U, 0.1)
    in_e = gen.gaussian_half_spinor(dims, rng)
    in_o = gen.gaussian_half_spinor(dims, rng)
    out_o = oracle.dslash_half(dims, U, 1, in_e)
    out_e = oracle.dslash_half(dims, U, 0, in_o)
    assert rel(out_o.reshape(-1), D_oe @ in_e.reshape(-1)) < 1e-14
    assert rel(out_e.reshape(-1), D_eo @ in_o.reshape(-1)) < 1e-14
    # half <-> full round trip uses idxh = lex // 2 (Eq. 9)
    lex_e = gen.half_index_of_parity(dims, 0)
    full = oracle.half_to_full(dims, 0, in_e)
    assert np.array_equal(full[lex_e], in_e)
    assert np.abs(np.delete(full, lex_e, axis=0)).max() == 0.0
    assert np.array_equal(oracle.full_to_half(dims, 0, full), in_e)


# ----------------------------------------------------------------------------------------------
# Closed forms
# ----------------------------------------------------------------------------------------------
def test_free_field_plane_wave_spectrum():
    """U=1: every plane wave on even sites is an eigenvector of A with eigenvalue
    m^2 + sum_mu sin^2 p_mu, p_{0,1,2} = 2 pi n/N, p_3 = (2n+1) pi/N3 (antiperiodic).
    Catches a missing 1/2 (x4), a wrong phase convention, a wrong BC."""
    dims = (4, 4, 6, 4)
    U = gen.unit_links(dims)
    m = 0.37
    coords = gen.site_coords(dims)
    lex_e = gen.half_index_of_parity(dims, 0)
    xe = coords[lex_e]
    colour = np.array([0.3 - 0.2j, 1.0 + 0.5j, -0.7j])
    worst = 0.0
    for n in [(0, 0, 0, 0), (1, 0, 0, 0), (0, 1, 2, 1), (3, 2, 5, 3), (2, 3, 1, 2), (1, 1, 1, 0)]:
        p = np.array([2 * np.pi * n[0] / dims[0], 2 * np.pi * n[1] / dims[1],
                      2 * np.pi * n[2] / dims[2], (2 * n[3] + 1) * np.pi / dims[3]])
        phi = np.exp(1j * (xe @ p))[:, None] * colour[None, :]
        lam = m * m + np.sum(np.sin(p) ** 2)
        out = oracle.mdagm(dims, U, m, phi)
        worst = max(worst, rel(out, lam * phi))
    assert worst < 1e-13
    # periodic variant: p_3 = 2 pi n / N3
    p = np.array([2 * np.pi / 4, 0.0, 2 * np.pi * 2 / 6, 2 * np.pi * 3 / 4])
    phi = np.exp(1j * (xe @ p))[:, None] * colour[None, :]
    out = oracle.mdagm(dims, U, m, phi, antiperiodic_t=False)
    assert rel(out, (m * m + np.sum(np.sin(p) ** 2)) * phi) < 1e-13


def test_constant_spinor_boundary_closed_form():
    """U=1, psi = constant c: (D psi)(x) = +eta_3(x) c at x3=0, -eta_3(x) c at x3=N3-1,
    0 elsewhere; identically 0 with periodic BC.  Catches a sign or slice error in the BC."""
    dims = (4, 2, 4, 6)
    U = gen.unit_links(dims)
    c = np.array([1.0 + 2.0j, -0.5j, 0.25])
    V = gen.volume(dims)
    psi = np.tile(c, (V, 1))
    coords = gen.site_coords(dims)
    eta3 = (-1.0) ** (coords[:, 0] + coords[:, 1] + coords[:, 2])
    want = np.zeros((V, 3), dtype=np.complex128)
    want[coords[:, 3] == 0] = (eta3[coords[:, 3] == 0])[:, None] * c
    want[coords[:, 3] == dims[3] - 1] = -(eta3[coords[:, 3] == dims[3] - 1])[:, None] * c
    got = oracle.dirac_full(dims, U, psi, antiperiodic_t=True)
    assert np.abs(got - want).max() == 0.0
    assert np.abs(oracle.dirac_full(dims, U, psi, antiperiodic_t=False)).max() == 0.0


# ----------------------------------------------------------------------------------------------
# Invariants
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 2, 8)])
def test_antihermiticity_D_oe_dagger_is_minus_D_eo(dims):
    """<phi, D_eo psi> + <D_oe phi, psi> = 0 (Eq. 7), real and imaginary parts."""
    rng = np.random.default_rng(11)
    U = gen.smooth_links(dims, 0.5, rng)
    phi_e = gen.gaussian_half_spinor(dims, rng)
    psi_o = gen.gaussian_half_spinor(dims, rng)
    lhs = np.vdot(phi_e, oracle.dslash_half(dims, U, 0, psi_o))
    rhs = np.vdot(oracle.dslash_half(dims, U, 1, phi_e), psi_o)
    scale = np.linalg.norm(phi_e) * np.linalg.norm(psi_o)
    assert abs(lhs + rhs) / scale < 1e-13
    assert abs(lhs) / scale > 1e-4  # the identity is not vacuous


def test_gauge_covariance():
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dagger, psi' = g psi  =>  D[U'] psi' = g D[U] psi."""
    dims = (4, 4, 4, 6)
    rng = np.random.default_rng(5)
    U = gen.smooth_links(dims, 0.3, rng)
    psi = gen.gaussian_spinor(dims, rng)
    V = gen.volume(dims)
    g = gen.haar_like_links(dims, rng)[:, 0]           # one SU(3) per site
    coords = gen.site_coords(dims)
    Up = np.empty_like(U)
    for mu in range(4):
        fwd = coords.copy()
        fwd[:, mu] = (fwd[:, mu] + 1) % dims[mu]
        lex_f = fwd[:, 0] + dims[0] * (fwd[:, 1] + dims[1] * (fwd[:, 2] + dims[2] * fwd[:, 3]))
        Up[:, mu] = np.einsum("nab,nbc,ndc->nad", g, U[:, mu], g[lex_f].conj())
    psip = np.einsum("nab,nb->na", g, psi)
    lhs = oracle.dirac_full(dims, Up, psip)
    rhs = np.einsum("nab,nb->na", g, oracle.dirac_full(dims, U, psi))
    assert rel(lhs, rhs) < 1e-13
    assert V == psi.shape[0]


def test_normal_operator_positive_definite_and_matches_dense():
    """A = m^2 - D_eo D_oe: Hermitian, eigenvalues >= m^2; oracle.mdagm = dense A."""
    dims = (4, 4, 4, 4)
    rng = np.random.default_rng(3)
    U = gen.haar_like_links(dims, rng)
    m = 0.05
    A, _, _ = dense_normal_operator(dims, U, m)
    assert np.abs(A - A.conj().T).max() < 1e-14
    ev = np.linalg.eigvalsh(A)
    assert ev.min() >= m * m * (1 - 1e-9)
    v = gen.gaussian_half_spinor(dims, rng)
    assert rel(oracle.mdagm(dims, U, m, v).reshape(-1), A @ v.reshape(-1)) < 1e-13
    assert rel(oracle.mdagm(dims, U, m, v, sigma=0.7).reshape(-1), (A + 0.7 * np.eye(A.shape[0])) @ v.reshape(-1)) < 1e-13


def test_norm_ratio_statistical_sanity():
    """Gaussian psi: ||D psi||^2 / ||psi||^2 ~ 2 (8 hops x (1/2)^2) -- sanity, loose."""
    dims = (4, 4, 4, 4)
    rng = np.random.default_rng(9)
    U = gen.haar_like_links(dims, rng)
    psi = gen.gaussian_spinor(dims, rng)
    ratio = np.linalg.norm(oracle.dirac_full(dims, U, psi)) ** 2 / np.linalg.norm(psi) ** 2
    assert 1.7 < ratio < 2.3


# ----------------------------------------------------------------------------------------------
# Row-3 reconstruction
# ----------------------------------------------------------------------------------------------
def test_row3_reconstruction_against_generator():
    """The generators fix det=1 by a phase on the Gram-Schmidt row 2 (no wedge product), so
    r2 = (r0 ^ r1)^* must reproduce their row 2 to round-off."""
    dims = (4, 4, 2, 2)
    for U in (gen.haar_like_links(dims, 21), gen.smooth_links(dims, 0.5, 22)):
        R = oracle.reconstruct_row3(U)
        assert np.array_equal(R[..., :2, :], U[..., :2, :])
        assert np.abs(R[..., 2, :] - U[..., 2, :]).max() < 5e-15
        eye = np.einsum("nmab,nmcb->nmac", R, R.conj())
        assert np.abs(eye - np.eye(3)).max() < 5e-15
        assert np.abs(np.linalg.det(R) - 1.0).max() < 5e-15
    # and a hand example: rows e0, e1 -> e2 ; rows (i e0), e1 -> conj(i) e2 = -i e2
    M = np.zeros((1, 3, 3), dtype=np.complex128)
    M[0, 0, 0] = 1j
    M[0, 1, 1] = 1.0
    assert np.allclose(oracle.reconstruct_row3(M)[0, 2], [0, 0, -1j])


# ----------------------------------------------------------------------------------------------
# CG (reading R10) and multi-shift CG (reading R11)
# ----------------------------------------------------------------------------------------------
def test_cg_against_dense_solve():
    dims = (4, 4, 4, 4)
    rng = np.random.default_rng(2)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m = 0.1
    A, _, _ = dense_normal_operator(dims, U, m)
    x_dense = np.linalg.solve(A, b.reshape(-1))
    res = oracle.cg(dims, U, m, b, 1e-12, 2000, hist_len=2000)
    assert res["converged"]
    assert res["true_relres"] < 5e-12
    assert rel(res["x"].reshape(-1), x_dense) < 1e-9
    # the recursive residual history is what the stopping rule saw
    k = res["iters"]
    assert res["rnorm"][k - 1] <= 1e-12 * np.linalg.norm(b)
    assert res["rnorm"][k - 2] > 1e-12 * np.linalg.norm(b)
    # A-norm of the error decreases monotonically (textbook CG property): replay with max_iter
    errs = []
    for it in (1, 2, 3, 5, 8, 13):
        xi = oracle.cg(dims, U, m, b, 1e-30, it)["x"].reshape(-1)
        e = xi - x_dense
        errs.append(np.real(np.vdot(e, A @ e)))
    assert all(errs[i + 1] < errs[i] for i in range(len(errs) - 1))


def test_cg_first_step_closed_form():
    """alpha_0 = <b,b>/<b,Ab>, x_1 = alpha_0 b, beta_0 = |r_1|^2/|b|^2 -- against the dense A."""
    dims = (2, 2, 2, 2)
    rng = np.random.default_rng(4)
    U = gen.haar_like_links(dims, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m = 0.3
    A, _, _ = dense_normal_operator(dims, U, m)
    bv = b.reshape(-1)
    a0 = np.real(np.vdot(bv, bv)) / np.real(np.vdot(bv, A @ bv))
    r1 = bv - a0 * (A @ bv)
    res = oracle.cg(dims, U, m, b, 1e-30, 2, hist_len=2)
    assert abs(res["alpha"][0] - a0) < 1e-14 * abs(a0)
    assert abs(res["rnorm"][0] - np.linalg.norm(r1)) < 1e-13 * np.linalg.norm(r1)
    assert abs(res["beta"][0] - np.vdot(r1, r1).real / np.vdot(bv, bv).real) < 1e-13
    x1 = oracle.cg(dims, U, m, b, 1e-30, 1)["x"].reshape(-1)
    assert rel(x1, a0 * bv) < 1e-15


def test_cg_exact_termination_and_special_cases():
    # 2^4: dim = 24; in exact arithmetic CG terminates within 24 iterations, in fp64 loss of
    # orthogonality costs a few more at tol 1e-10
    dims = (2, 2, 2, 2)
    rng = np.random.default_rng(6)
    U = gen.haar_like_links(dims, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    res = oracle.cg(dims, U, 0.5, b, 1e-10, 100)
    assert res["converged"] and res["iters"] <= 24 + 4
    # free field + plane-wave rhs: an eigenvector -> exactly 1 iteration, x = b / lambda
    dims = (4, 4, 4, 4)
    Uf = gen.unit_links(dims)
    xe = gen.site_coords(dims)[gen.half_index_of_parity(dims, 0)]
    p = np.array([2 * np.pi / 4, 0.0, 2 * np.pi * 2 / 4, 3 * np.pi / 4])
    bw = np.exp(1j * (xe @ p))[:, None] * np.array([1.0, 2.0j, -0.5])[None, :]
    m = 0.2
    res = oracle.cg(dims, Uf, m, bw, 1e-12, 50)
    assert res["iters"] == 1
    assert rel(res["x"], bw / (m * m + np.sum(np.sin(p) ** 2))) < 1e-13
    # m -> infinity: x -> b / m^2
    b2 = gen.gaussian_half_spinor(dims, rng)
    res = oracle.cg(dims, Uf, 1e4, b2, 1e-12, 50)
    assert rel(res["x"], b2 / 1e8) < 1e-7
    # zero rhs
    res = oracle.cg(dims, Uf, m, np.zeros_like(b2), 1e-12, 50)
    assert res["iters"] == 0 and np.abs(res["x"]).max() == 0.0
    # max_iter reached is reported, not hidden
    res = oracle.cg(dims, gen.smooth_links(dims, 0.5, 8), 0.01, b2, 1e-14, 3)
    assert not res["converged"] and res["iters"] == 3


def test_multishift_against_dense_and_single_shift():
    dims = (4, 4, 4, 4)
    rng = np.random.default_rng(4)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m = 0.05
    shifts = np.array([0.3, 1e-3, 1.0, 0.02])        # unsorted on purpose: base = the minimum
    A, _, _ = dense_normal_operator(dims, U, m)
    res = oracle.cg_multishift(dims, U, m, shifts, b, 1e-11, 5000)
    assert res["converged"]
    eye = np.eye(A.shape[0])
    for i, s in enumerate(shifts):
        xd = np.linalg.solve(A + s * eye, b.reshape(-1))
        assert rel(res["x"][i].reshape(-1), xd) < 1e-8
        assert res["true_relres"][i] < 3e-11
    # larger shifts freeze earlier (zeta_i decreases faster for larger delta_i)
    order = np.argsort(shifts)
    assert all(res["conv_iter"][order[j]] >= res["conv_iter"][order[j + 1]] for j in range(3))
    assert res["conv_iter"].max() == res["iters"]
    # single-shift CG on A + sigma == CG with mass^2 -> m^2 + sigma
    s = shifts[0]
    single = oracle.cg(dims, U, np.sqrt(m * m + s), b, 1e-11, 5000)
    assert rel(res["x"][0], single["x"]) < 1e-8
    assert abs(single["iters"] - res["conv_iter"][0]) <= 2


def test_multishift_residual_identity_and_first_zeta():
    """b - (A + sigma_i) x_i = zeta_i r while shift i is active; zeta_i after step 0 =
    1/(1 + delta_i alpha_0).  Catches any slip in the zeta/alpha_i/beta_i recurrences."""
    dims = (4, 4, 2, 4)
    rng = np.random.default_rng(12)
    U = gen.smooth_links(dims, 0.4, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m = 0.03
    shifts = gen.rhmc_shifts(8)
    assert np.allclose(shifts[[0, 1, 7]], [1e-4, 3.72759372e-4, 1.0])
    bn = np.linalg.norm(b)
    for it in (1, 2, 3, 7, 20):
        res = oracle.cg_multishift(dims, U, m, shifts, b, 1e-30, it, hist_len=it)
        assert res["iters"] == it and not res["converged"]
        for i, s in enumerate(shifts):
            true_r = b - oracle.mdagm(dims, U, m, res["x"][i], sigma=s)
            assert np.linalg.norm(true_r - res["zeta"][i] * res["r"]) < 1e-12 * bn
        if it == 1:
            a0 = res["alpha"][0]
            assert np.allclose(res["zeta"], 1.0 / (1.0 + (shifts - shifts.min()) * a0), rtol=1e-14)
    # the base system's alpha/beta/|r| history is plain CG on A + sigma_min
    ms = oracle.cg_multishift(dims, U, m, shifts, b, 1e-30, 10, hist_len=10)
    sg = oracle.cg(dims, U, np.sqrt(m * m + shifts.min()), b, 1e-30, 10, hist_len=10)
    assert np.allclose(ms["alpha"], sg["alpha"], rtol=1e-10)
    assert np.allclose(ms["rnorm"], sg["rnorm"], rtol=1e-10)
    assert np.allclose(ms["beta"][:9], sg["beta"][:9], rtol=1e-10)


def test_rational_apply_against_dense_partial_fractions_and_plane_wave():
    """NEXT-1: y = c0 b + sum_i c_i (A+sigma_i)^-1 b  (the rational function of
    the RHMC whose poles are the shifts of Eq. 6).  Pins: (i) dense solves; (ii) the partial-fraction
    identity 1/((A+s1)(A+s2)) = [1/(A+s1) - 1/(A+s2)]/(s2-s1): applying both factors to y must give
    b back -- catches a wrong sign, a swapped or dropped coefficient, a dropped c0 (checked with a
    second case); (iii) free field, plane-wave b: y = (c0 + sum c_i/(lambda+sigma_i)) b."""
    dims = (4, 4, 4, 4)
    rng = np.random.default_rng(8)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m = 0.05
    shifts = np.array([0.3, 1e-3, 1.0, 0.02])
    c0, c = 0.7, np.array([0.5, -1.25, 2.0, 0.125])
    A, _, _ = dense_normal_operator(dims, U, m)
    eye = np.eye(A.shape[0])
    res = oracle.rational_apply(dims, U, m, shifts, c0, c, b, 1e-12, 5000)
    assert res["converged"]
    yd = c0 * b.reshape(-1) + sum(ci * np.linalg.solve(A + s * eye, b.reshape(-1)) for ci, s in zip(c, shifts))
    assert rel(res["y"].reshape(-1), yd) < 1e-9
    # (ii) partial fractions, checked with the operator only
    s1, s2 = 0.11, 0.83
    pf = oracle.rational_apply(dims, U, m, [s1, s2], 0.0, [1.0 / (s2 - s1), -1.0 / (s2 - s1)], b, 1e-12, 5000)
    back = oracle.mdagm(dims, U, m, oracle.mdagm(dims, U, m, pf["y"], sigma=s2), sigma=s1)
    assert rel(back, b) < 1e-9
    # with c0 = 1 and the same poles: (A+s1)(A+s2)(y - b) = b
    pf1 = oracle.rational_apply(dims, U, m, [s1, s2], 1.0, [1.0 / (s2 - s1), -1.0 / (s2 - s1)], b, 1e-12, 5000)
    back = oracle.mdagm(dims, U, m, oracle.mdagm(dims, U, m, pf1["y"] - b, sigma=s2), sigma=s1)
    assert rel(back, b) < 1e-9
    # (iii) free field plane wave
    dims = (4, 4, 6, 4)
    U1 = gen.unit_links(dims)
    xe = gen.site_coords(dims)[gen.half_index_of_parity(dims, 0)]
    p = np.array([2 * np.pi / 4, 0.0, 2 * np.pi * 2 / 6, 3 * np.pi / 4])
    phi = np.exp(1j * (xe @ p))[:, None] * np.array([0.3 - 0.2j, 1.0 + 0.5j, -0.7j])[None, :]
    lam = 0.37 ** 2 + np.sum(np.sin(p) ** 2)
    r = oracle.rational_apply(dims, U1, 0.37, shifts, c0, c, phi, 1e-13, 100)
    assert r["iters"] <= 2
    assert rel(r["y"], (c0 + np.sum(c / (lam + shifts))) * phi) < 1e-12


def _gell_mann():
    l = np.zeros((8, 3, 3), dtype=np.complex128)
    l[0][0, 1] = l[0][1, 0] = 1
    l[1][0, 1], l[1][1, 0] = -1j, 1j
    l[2][0, 0], l[2][1, 1] = 1, -1
    l[3][0, 2] = l[3][2, 0] = 1
    l[4][0, 2], l[4][2, 0] = -1j, 1j
    l[5][1, 2] = l[5][2, 1] = 1
    l[6][1, 2], l[6][2, 1] = -1j, 1j
    l[7] = np.diag([1, 1, -2]) / np.sqrt(3)
    return l


def _expm_herm(H, eps):
    w, v = np.linalg.eigh(H)
    return (v * np.exp(1j * eps * w)) @ v.conj().T


@pytest.mark.parametrize("dims,ap", [((2, 2, 2, 4), True), ((4, 2, 2, 2), True), ((2, 4, 2, 2), False)])
def test_fermion_force_against_finite_differences_of_the_action(dims, ap):
    """NEXT-3 (reading R21): dS/d eps under U_mu(x) -> exp(i eps T_a) U_mu(x) equals 2 Re Tr[i T_a F_mu(x)],
    with S = sum_i c_i Re phi^dag (A+sigma_i)^-1 phi evaluated by DENSE solves (no oracle code in S).
    Links on both parities, all four directions, across the antiperiodic boundary and with N_mu = 2
    (where x+mu = x-mu); catches a wrong sign, parity factor, conjugation, dropped 1/2 or eta."""
    rng = np.random.default_rng(12)
    U = gen.haar_like_links(dims, rng)
    phi = gen.gaussian_half_spinor(dims, rng)
    m = 0.4
    shifts = np.array([0.05, 0.7, 0.2])
    c = np.array([0.8, -0.45, 1.3])
    V = gen.volume(dims)

    def action(Uv):
        A, _, _ = dense_normal_operator(dims, Uv, m, antiperiodic_t=ap)
        eye = np.eye(A.shape[0])
        b = phi.reshape(-1)
        return sum(ci * np.real(np.vdot(b, np.linalg.solve(A + s * eye, b))) for ci, s in zip(c, shifts))

    A, _, _ = dense_normal_operator(dims, U, m, antiperiodic_t=ap)
    eye = np.eye(A.shape[0])
    xs = np.stack([np.linalg.solve(A + s * eye, phi.reshape(-1)).reshape(-1, 3) for s in shifts])
    F = oracle.fermion_force(dims, U, c, xs, antiperiodic_t=ap)
    # F is traceless anti-Hermitian
    assert np.abs(F + F.conj().transpose(0, 1, 3, 2)).max() < 1e-14
    assert np.abs(np.trace(F, axis1=2, axis2=3)).max() < 1e-14
    lam = _gell_mann()
    coords = gen.site_coords(dims)
    eps = 1e-5
    # sites chosen to include both parities and the last x3 slice (boundary-crossing forward hop)
    picks = [0, 1, V - 1, V - 2, V // 2 + 1]
    worst = 0.0
    for k, lex in enumerate(picks):
        for mu in range(4):
            a = (3 * k + mu) % 8
            Up, Um = U.copy(), U.copy()
            Up[lex, mu] = _expm_herm(lam[a], eps) @ U[lex, mu]
            Um[lex, mu] = _expm_herm(lam[a], -eps) @ U[lex, mu]
            fd = (action(Up) - action(Um)) / (2 * eps)
            an = 2 * np.real(np.trace(1j * lam[a] @ F[lex, mu]))
            worst = max(worst, abs(fd - an) / max(1e-3, abs(an)))
    assert worst < 1e-6, worst
    assert {int(coords[p].sum() % 2) for p in picks} == {0, 1}


@pytest.mark.parametrize("dims,ap", [((2, 2, 2, 4), True), ((2, 4, 2, 2), False)])
def test_fermion_force_with_backfield_against_finite_differences(dims, ap):
    """oracle_fermion_force_bf (reading R6 + R21): with links e^{i theta} U in D, dS/d eps under U_mu(x) -> exp(i eps
    T_a) U_mu(x) equals 2 Re Tr[i T_a F_mu(x)]; S by DENSE solves with the phased dense operator (no oracle code in S).
    Also: theta = 0 reproduces the plain force, and the phases absorbed into the links give the same force through
    the plain entry point (the force of a left multiplication does not care which factor carries the phase)."""
    rng = np.random.default_rng(19)
    U = gen.haar_like_links(dims, rng)
    phi = gen.gaussian_half_spinor(dims, rng)
    theta = gen.uniform_backfield(dims, rng)
    m = 0.4
    shifts = np.array([0.05, 0.7])
    c = np.array([0.8, -0.45])
    V = gen.volume(dims)

    def action(Uv):
        A, _, _ = dense_normal_operator(dims, Uv, m, antiperiodic_t=ap, theta=theta)
        b = phi.reshape(-1)
        return sum(ci * np.real(np.vdot(b, np.linalg.solve(A + s * np.eye(A.shape[0]), b))) for ci, s in zip(c, shifts))

    A, _, _ = dense_normal_operator(dims, U, m, antiperiodic_t=ap, theta=theta)
    xs = np.stack([np.linalg.solve(A + s * np.eye(A.shape[0]), phi.reshape(-1)).reshape(-1, 3) for s in shifts])
    F = oracle.fermion_force(dims, U, c, xs, antiperiodic_t=ap, theta=theta)
    assert np.abs(F + F.conj().transpose(0, 1, 3, 2)).max() < 1e-14
    assert np.abs(np.trace(F, axis1=2, axis2=3)).max() < 1e-14
    lam = _gell_mann()
    eps = 1e-5
    worst = 0.0
    for k, lex in enumerate([0, 1, V - 1, V // 2 + 1]):
        for mu in range(4):
            a = (3 * k + mu + 2) % 8
            Up, Um = U.copy(), U.copy()
            Up[lex, mu] = _expm_herm(lam[a], eps) @ U[lex, mu]
            Um[lex, mu] = _expm_herm(lam[a], -eps) @ U[lex, mu]
            fd = (action(Up) - action(Um)) / (2 * eps)
            an = 2 * np.real(np.trace(1j * lam[a] @ F[lex, mu]))
            worst = max(worst, abs(fd - an) / max(1e-3, abs(an)))
    assert worst < 1e-6, worst
    # phases absorbed into the links, plain entry point
    Uph = U * np.exp(1j * theta)[:, :, None, None]
    assert rel(oracle.fermion_force(dims, Uph, c, xs, antiperiodic_t=ap), F) < 1e-13
    # theta = 0 is the plain force; the phases matter
    F0 = oracle.fermion_force(dims, U, c, xs, antiperiodic_t=ap)
    assert np.array_equal(oracle.fermion_force(dims, U, c, xs, antiperiodic_t=ap, theta=np.zeros((V, 4))), F0)
    assert rel(F0, F) > 0.1


def _gauge_W(dims, U, c0, c1):
    """W = sum_x sum_{mu<nu} c0 ReTr P + c1 (ReTr R_{mu nu} + ReTr R_{nu mu}), with numpy rolls on the
    [x3,x2,x1,x0] grid -- independent of the oracle's path walker.  Returns (W, sum ReTr P, sum ReTr R)."""
    n0, n1, n2, n3 = dims
    G = U.reshape(n3, n2, n1, n0, 4, 3, 3)

    def sh(A, mu, k=1):                       # A(x + k mu)
        return np.roll(A, -k, axis=3 - mu)

    def dag(A):
        return A.conj().swapaxes(-1, -2)

    def retr(A):
        return np.real(np.trace(A, axis1=-2, axis2=-1)).sum()

    sp = sr = 0.0
    for mu in range(4):
        for nu in range(4):
            if nu == mu:
                continue
            Um, Un = G[..., mu, :, :], G[..., nu, :, :]
            if mu < nu:
                sp += retr(Um @ sh(Un, mu) @ dag(sh(Um, nu)) @ dag(Un))
            # R_{mu nu}: two steps along mu, one along nu (all ordered pairs mu != nu)
            sr += retr(Um @ sh(Um, mu) @ sh(Un, mu, 2) @ dag(sh(sh(Um, mu), nu)) @ dag(sh(Um, nu)) @ dag(Un))
    return c0 * sp + c1 * sr, sp, sr


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 4, 6, 2)])
def test_gauge_staples_finite_differences_sum_rule_unit_links_covariance(dims):
    """NEXT-4 (reading R22).  (i) d/d eps of W under U_mu(x) -> exp(i eps T_a) U_mu(x) = Re Tr[i T_a U_mu(x) S_mu(x)]
    -- any wrong path, ordering, dagger or coefficient fails it; (ii) sum_{x,mu} Re Tr[U S] = 4 c0 sum P +
    6 c1 sum R (a plaquette has 4 links, a rectangle 6), for each family separately; (iii) unit links:
    S = (6 c0 + 18 c1) 1; (iv) S'_mu(x) = g(x+mu) S_mu(x) g(x)^dagger under a gauge transformation."""
    rng = np.random.default_rng(14)
    U = gen.haar_like_links(dims, rng)
    V = gen.volume(dims)
    c0, c1 = oracle.SYMANZIK_C0, oracle.SYMANZIK_C1
    assert (c0, c1) == (5.0 / 3.0, -1.0 / 12.0)
    S = oracle.gauge_staples(dims, U)
    lam = _gell_mann()
    eps = 1e-5
    worst = 0.0
    for k, lex in enumerate([0, 3, V - 1, V // 2 + 1, V // 3]):
        for mu in range(4):
            a = (5 * k + mu) % 8
            Up, Um = U.copy(), U.copy()
            Up[lex, mu] = _expm_herm(lam[a], eps) @ U[lex, mu]
            Um[lex, mu] = _expm_herm(lam[a], -eps) @ U[lex, mu]
            fd = (_gauge_W(dims, Up, c0, c1)[0] - _gauge_W(dims, Um, c0, c1)[0]) / (2 * eps)
            an = np.real(np.trace(1j * lam[a] @ U[lex, mu] @ S[lex, mu]))
            worst = max(worst, abs(fd - an) / max(1e-2, abs(an)))
    assert worst < 1e-6, worst
    # (ii) loop counting, each family alone
    _, sp, sr = _gauge_W(dims, U, 1.0, 1.0)
    Sp = oracle.gauge_staples(dims, U, 1.0, 0.0)
    Sr = oracle.gauge_staples(dims, U, 0.0, 1.0)
    tot = lambda St: np.real(np.einsum("xmab,xmba->", U, St))
    assert abs(tot(Sp) - 4 * sp) < 1e-9 * abs(sp) and abs(tot(Sr) - 6 * sr) < 1e-9 * abs(sr)
    assert np.allclose(S, c0 * Sp + c1 * Sr, atol=1e-13)
    # (iii) unit links
    S1 = oracle.gauge_staples(dims, gen.unit_links(dims))
    assert np.allclose(S1, (6 * c0 + 18 * c1) * np.eye(3), atol=1e-13)
    # (iv) gauge covariance
    g = gen.haar_like_links(dims, rng)[:, 0]
    coords = gen.site_coords(dims)
    Ug = np.empty_like(U)
    fwd = np.empty((V, 4), dtype=np.int64)
    for mu in range(4):
        c = coords.copy()
        c[:, mu] = (c[:, mu] + 1) % dims[mu]
        fwd[:, mu] = c[:, 0] + dims[0] * (c[:, 1] + dims[1] * (c[:, 2] + dims[2] * c[:, 3]))
        Ug[:, mu] = g @ U[:, mu] @ g[fwd[:, mu]].conj().swapaxes(-1, -2)
    Sg = oracle.gauge_staples(dims, Ug)
    for mu in range(4):
        assert np.allclose(Sg[:, mu], g[fwd[:, mu]] @ S[:, mu] @ g.conj().swapaxes(-1, -2), atol=1e-12)


def test_multishift_rejects_bad_shifts():
    dims = (2, 2, 2, 2)
    U = gen.unit_links(dims)
    b = gen.gaussian_half_spinor(dims, 1)
    with pytest.raises(ValueError):
        oracle.cg_multishift(dims, U, 0.1, [0.1, -0.2], b, 1e-8, 10)


def test_oracle_regression_fixture():
    """tests/golden/oracle_regression.json (written by make_golden.py from oracle/ only) still
    matches: guards against an unannounced change of the oracle's arithmetic.  The 8^4 CG count
    (143) also equals the survey's independent scratch run."""
    import json
    import os
    import sys
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    sys.path.insert(0, here)
    import make_golden
    want = json.load(open(os.path.join(here, "oracle_regression.json")))
    got = make_golden.compute()
    assert got["cg_8x4_m0.01_iters"] == want["cg_8x4_m0.01_iters"] == 143
    assert got["multishift_8x4_iters"] == want["multishift_8x4_iters"]
    assert got["multishift_8x4_conv_iter"] == want["multishift_8x4_conv_iter"]
    assert abs(got["config1_4x4_dirac_norm2"] - want["config1_4x4_dirac_norm2"]) < 1e-9 * want["config1_4x4_dirac_norm2"]
    assert np.allclose(got["config1_4x4_dirac_site0"], want["config1_4x4_dirac_site0"], rtol=1e-12)
    assert abs(got["cg_8x4_alpha0"] - want["cg_8x4_alpha0"]) < 1e-12
    assert got["rational_4x4_iters"] == want["rational_4x4_iters"]
    for k in ("rational_4x4_norm2", "force_4x4_norm2", "staples_4x4_norm2", "staples_4x4_retr_US"):
        assert abs(got[k] - want[k]) < 1e-9 * abs(want[k]), k
    assert np.allclose(got["force_4x4_link0"], want["force_4x4_link0"], rtol=1e-10, atol=1e-12)
