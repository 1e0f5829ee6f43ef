"""Parity of the backfield path (the fourth argument of the paper's acc_Deo(u, out, in, backfield), Listing 2,
PAPER.md:320-326; reading R6 of DESIGN.md: every link enters D as e^{i theta_mu(x)} U_mu(x)) against the CPU
oracle's *_bf entry points, through the C ABI (-m gpu).  Tolerances as in test_gpu_parity.py.
"""
import numpy as np
import pytest

import lqcd_inputs as gen
import oracle

pytestmark = pytest.mark.gpu

TOL = {0: 1e-12, 1: 1e-5}


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def round_inputs(prec, U, psi, theta):
    """fp32 contexts see the inputs rounded to nearest (theta as a float32); the oracle runs in fp64 on the SAME
    rounded numbers (reading R14)."""
    if prec == 0:
        return U, psi, theta
    c = lambda a: a.astype(np.complex64).astype(np.complex128)
    return c(U), c(psi), theta.astype(np.float32).astype(np.float64)


def make_lattice(dims, prec=0, recon=0, ap=True, **opts):
    import paper_1701_00426_b200 as L
    return L.Lattice(dims, prec=prec, recon=recon, antiperiodic_t=ap, options=opts)


@pytest.mark.parametrize("fmt", [0, 1])
@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("recon", [0, 1])
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 2, 2, 2), (6, 4, 2, 8), (12, 10, 6, 4)])
def test_dslash_backfield_both_parities(dims, prec, recon, layout, fmt):
    """Haar-like links, phases uniform in (-pi, pi): both parities, 2^4 (every hop wraps), ragged sizes; both
    native formats (theta stored / (cos, sin) stored)."""
    rng = np.random.default_rng(61)
    U = gen.haar_like_links(dims, rng)
    psi = gen.gaussian_spinor(dims, rng)
    theta = gen.uniform_backfield(dims, rng)
    U, psi, theta = round_inputs(prec, U, psi, theta)
    if recon == 1 and prec == 1:
        U = oracle.reconstruct_row3(U)
    lat = make_lattice(dims, prec, recon, True, layout=layout, backfield_format=fmt)
    links = lat.pack_links(U)
    bf = lat.pack_backfield(theta)
    for out_parity in (0, 1):
        phi_in = oracle.full_to_half(dims, 1 - out_parity, psi)
        want = oracle.dslash_half(dims, U, out_parity, phi_in, theta=theta)
        plain = oracle.dslash_half(dims, U, out_parity, phi_in)
        assert rel(plain, want) > 0.1                      # the phases matter
        inp = lat.pack_spinor(phi_in, 1 - out_parity)
        out = lat.new_spinor()
        lat.dslash_backfield(out_parity, out, inp, links, bf)
        assert rel(lat.unpack_spinor(out, out_parity), want) < TOL[prec], (dims, prec, recon, layout, out_parity)
        # the explicit call leaves the context without a backfield
        lat.dslash(out_parity, out, inp, links)
        assert rel(lat.unpack_spinor(out, out_parity), plain) < TOL[prec]
        # attached to the context: the plain call applies it
        lat.set_backfield(bf)
        lat.dslash(out_parity, out, inp, links)
        assert rel(lat.unpack_spinor(out, out_parity), want) < TOL[prec]
        lat.set_backfield(None)
    lat.close()


def test_backfield_zero_is_bit_identical_to_plain():
    """theta = 0: e^{i0} = 1 exactly, so the BF kernel must reproduce the plain kernel bit for bit."""
    dims = (6, 6, 4, 10)
    rng = np.random.default_rng(62)
    U = gen.smooth_links(dims, 0.3, rng)
    phi = gen.gaussian_half_spinor(dims, rng)
    lat = make_lattice(dims)
    links = lat.pack_links(U)
    bf = lat.pack_backfield(np.zeros((lat.V, 4)))
    inp = lat.pack_spinor(phi, 0)
    a, b = lat.new_spinor(), lat.new_spinor()
    lat.dslash(1, a, inp, links)
    lat.dslash_backfield(1, b, inp, links, bf)
    assert np.array_equal(lat.unpack_spinor(a, 1), lat.unpack_spinor(b, 1))
    lat.close()


@pytest.mark.parametrize("ap", [True, False])
def test_backfield_absorbed_into_links_18real(ap):
    """With 3-row storage the phased links e^{i theta} U can be packed as ordinary links: the plain kernel on them
    must agree with the backfield kernel on (U, theta) -- an identity between two different CUDA paths that the
    oracle pins on the CPU (tests/test_oracle_pins.py) and that is checked against the oracle here as well."""
    dims = (4, 6, 4, 4)
    rng = np.random.default_rng(63)
    U = gen.smooth_links(dims, 0.5, rng)
    phi = gen.gaussian_half_spinor(dims, rng)
    theta = gen.uniform_backfield(dims, rng)
    Uph = U * np.exp(1j * theta)[:, :, None, None]
    lat = make_lattice(dims, ap=ap)
    want = oracle.dslash_half(dims, U, 1, phi, antiperiodic_t=ap, theta=theta)
    inp = lat.pack_spinor(phi, 0)
    out = lat.new_spinor()
    lat.dslash(1, out, inp, lat.pack_links(Uph))
    assert rel(lat.unpack_spinor(out, 1), want) < 1e-12
    lat.dslash_backfield(1, out, inp, lat.pack_links(U), lat.pack_backfield(theta))
    assert rel(lat.unpack_spinor(out, 1), want) < 1e-12
    lat.close()


@pytest.mark.parametrize("fmt", [0, 1])
@pytest.mark.parametrize("prec", [0, 1])
def test_mdagm_and_multishift_with_backfield(prec, fmt):
    """The normal operator and the multi-shift solve with a backfield attached to the context: mdagm element by
    element; the solve by reading R16 (true residuals with the ORACLE operator, iteration counts, lock-step
    scalars) and with the chunk graph on (the graph key holds the backfield pointer)."""
    dims = (8, 4, 6, 8)
    rng = np.random.default_rng(64)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    theta = gen.uniform_backfield(dims, rng)
    U, b, theta = round_inputs(prec, U, b, theta)
    mass, tol = 0.1, (1e-10 if prec == 0 else 1e-5)
    shifts = gen.rhmc_shifts(4)
    lat = make_lattice(dims, prec, backfield_format=fmt)
    links = lat.pack_links(U)
    bf = lat.pack_backfield(theta)
    be = lat.pack_spinor(b, 0)
    lat.set_backfield(bf)
    out = lat.new_spinor()
    lat.mdagm(out, be, links, mass, 0.37)
    assert rel(lat.unpack_spinor(out, 0), oracle.mdagm(dims, U, mass, b, sigma=0.37, theta=theta)) < TOL[prec]
    xs = [lat.new_spinor() for _ in shifts]
    res = lat.cg_multishift(xs, be, links, mass, shifts, tol, 4000)
    ref = oracle.cg_multishift(dims, U, mass, shifts, b, tol, 4000, hist_len=10, theta=theta)
    ref_plain = oracle.cg_multishift(dims, U, mass, shifts, b, tol, 4000)
    assert abs(res["iters"] - ref["iters"]) <= max(2, ref["iters"] // 50)
    assert lat.get_option("graph_active") == 1
    bn = np.linalg.norm(b)
    for i, s in enumerate(shifts):
        xg = lat.unpack_spinor(xs[i], 0)
        tr = np.linalg.norm(b - oracle.mdagm(dims, U, mass, xg, sigma=s, theta=theta)) / bn
        assert tr < (1.5 * tol if prec == 0 else 20 * tol), (i, tr)
        assert rel(xg, ref["x"][i]) < 10 * 7 / (mass * mass + s) * tol
        assert rel(ref_plain["x"][i], ref["x"][i]) > 1e-2          # a different system from the plain one
    if prec == 0:
        h = lat.solver_history()
        n = min(10, len(h["alpha"]), len(ref["alpha"]))
        assert np.allclose(h["alpha"][:n], ref["alpha"][:n], rtol=1e-10)
        assert np.allclose(h["beta"][:n], ref["beta"][:n], rtol=1e-10)
    # detaching gives the plain operator back (and a different graph key)
    lat.set_backfield(None)
    res2 = lat.cg_multishift(xs, be, links, mass, shifts, tol, 4000)
    assert abs(res2["iters"] - ref_plain["iters"]) <= max(2, ref_plain["iters"] // 50)
    for i in range(len(shifts)):
        assert rel(lat.unpack_spinor(xs[i], 0), ref_plain["x"][i]) < 10 * 7 / (mass * mass + shifts[i]) * tol
    lat.close()


@pytest.mark.parametrize("fmt", [0, 1])
def test_backfield_large_volume_sampled_sites(fmt):
    """32^4 (the bench configuration), fp64 12-real: sampled sites incl. corners and both x3 boundary slices
    against oracle.dirac_site with the phase field."""
    dims = (32, 32, 32, 32)
    rng = np.random.default_rng(65)
    U = gen.smooth_links(dims, 0.3, rng)
    psi = gen.gaussian_spinor(dims, rng)
    theta = gen.uniform_backfield(dims, rng)
    lat = make_lattice(dims, 0, 1, backfield_format=fmt)
    links = lat.pack_links(U)
    bf = lat.pack_backfield(theta)
    coords = [(0, 0, 0, 0), (31, 31, 31, 31), (0, 31, 0, 31), (31, 0, 31, 0), (1, 0, 0, 0), (0, 0, 0, 31), (5, 7, 11, 0)]
    coords += [tuple(int(v) for v in rng.integers(0, 32, 4)) for _ in range(200)]
    outs = {}
    for par in (0, 1):
        inp = lat.pack_spinor(oracle.full_to_half(dims, 1 - par, psi), 1 - par)
        out = lat.new_spinor()
        lat.dslash_backfield(par, out, inp, links, bf)
        outs[par] = lat.unpack_spinor(out, par)
    worst = 0.0
    for x in coords:
        par = sum(x) % 2
        lex = x[0] + 32 * (x[1] + 32 * (x[2] + 32 * x[3]))
        want = oracle.dirac_site(dims, U, psi, x, theta=theta)
        got = outs[par][lex // 2]
        worst = max(worst, np.linalg.norm(got - want) / np.linalg.norm(want))
    assert worst < 1e-12, worst
    lat.close()


@pytest.mark.parametrize("fmt", [0, 1])
@pytest.mark.parametrize("recon", [0, 1])
@pytest.mark.parametrize("prec", [0, 1])
def test_fermion_force_with_backfield(prec, recon, fmt):
    """lqcd_fermion_force with a backfield attached: F = TA[e^{i theta} U Q] with the y_i of the phased operator,
    element by element against oracle_fermion_force_bf (pinned by finite differences on the CPU)."""
    dims = (6, 4, 10, 8)
    rng = np.random.default_rng(67)
    U = gen.haar_like_links(dims, rng)
    theta = gen.uniform_backfield(dims, rng)
    n = 3
    xs = np.stack([gen.gaussian_half_spinor(dims, rng) for _ in range(n)])
    if prec == 1:
        U = U.astype(np.complex64).astype(np.complex128)
        xs = xs.astype(np.complex64).astype(np.complex128)
        theta = theta.astype(np.float32).astype(np.float64)
        if recon == 1:
            U = oracle.reconstruct_row3(U)
    c = np.array([0.7, -1.1, 0.4])
    lat = make_lattice(dims, prec, recon, backfield_format=fmt)
    links = lat.pack_links(U)
    lat.set_backfield(lat.pack_backfield(theta))
    got = lat.unpack_tamat(lat.fermion_force([lat.pack_spinor(x, 0) for x in xs], links, c))
    want = oracle.fermion_force(dims, U, c, xs, theta=theta)
    assert rel(got, want) < TOL[prec], (prec, recon, fmt, rel(got, want))
    assert rel(oracle.fermion_force(dims, U, c, xs), want) > 0.1          # the phases matter
    lat.close()


def test_backfield_errors():
    import paper_1701_00426_b200 as L
    dims = (4, 4, 4, 4)
    rng = np.random.default_rng(66)
    U = gen.smooth_links(dims, 0.3, rng)
    lat = make_lattice(dims)
    lat.pack_links(U)
    lat.pack_backfield(gen.uniform_backfield(dims, rng))
    with pytest.raises(L.LqcdError):            # the format is fixed once a backfield was packed
        lat.set_option("backfield_format", 1)
    with pytest.raises(L.LqcdError):
        lat.set_option("backfield_format", 2)       # out of range
    lat.close()
