"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs (-m gpu).  Tolerances: 1e-12 relative L2 in fp64, 1e-5 in fp32 (BASELINE.json
north_star); solver criteria are reading R16 of DESIGN.md.
"""
import numpy as np
import pytest

import lqcd_inputs as gen
import oracle

pytestmark = pytest.mark.gpu

TOL = {0: 1e-12, 1: 1e-5}


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def round_inputs(prec, *arrs):
    """fp32 contexts see the fp64 inputs rounded to nearest; the oracle runs in fp64 on the SAME
    rounded numbers, so the 1e-5 bound measures arithmetic only (reading R14)."""
    if prec == 0:
        return arrs
    return tuple(a.astype(np.complex64).astype(np.complex128) for a in arrs)


def make_lattice(dims, prec=0, recon=0, ap=True, **opts):
    import paper_1701_00426_b200 as L
    return L.Lattice(dims, prec=prec, recon=recon, antiperiodic_t=ap, options=opts)


def gpu_dslash(lat, U, phi_in, out_parity):
    links = lat.pack_links(U)
    inp = lat.pack_spinor(phi_in, 1 - out_parity)
    out = lat.new_spinor()
    lat.dslash(out_parity, out, inp, links)
    return lat.unpack_spinor(out, out_parity)


# ------------------------------------------------------------------------------------------------
# Dslash
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("recon", [0, 1])
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 2, 2, 2), (6, 4, 2, 8), (12, 10, 6, 4)])
def test_dslash_both_parities(dims, prec, recon, layout):
    """BASELINE.json config 1 (4^4, Haar-like links, seed 1, full-lattice Gaussian spinor, both
    parities) plus 2^4 (N=2 wrap), a ragged lattice and one spanning several CTAs with a tail."""
    rng = np.random.default_rng(1)
    U = gen.haar_like_links(dims, rng)
    psi = gen.gaussian_spinor(dims, rng)
    U, psi = round_inputs(prec, U, psi)
    if recon == 1 and prec == 1:
        # rounding to fp32 breaks unitarity at 1e-7; the 12-real oracle input is the rebuilt field
        U = oracle.reconstruct_row3(U)
    lat = make_lattice(dims, prec, recon, True, layout=layout)
    for out_parity in (0, 1):
        phi_in = oracle.full_to_half(dims, 1 - out_parity, psi)
        want = oracle.dslash_half(dims, U, out_parity, phi_in)
        got = gpu_dslash(lat, U, phi_in, out_parity)
        assert rel(got, want) < TOL[prec], (dims, prec, recon, layout, out_parity)
    lat.close()


@pytest.mark.parametrize("ap", [True, False])
def test_dslash_boundary_conditions(ap):
    dims = (4, 6, 4, 4)
    rng = np.random.default_rng(17)
    U = gen.smooth_links(dims, 0.5, rng)
    phi = gen.gaussian_half_spinor(dims, rng)
    lat = make_lattice(dims, ap=ap)
    want = oracle.dslash_half(dims, U, 1, phi, antiperiodic_t=ap)
    assert rel(gpu_dslash(lat, U, phi, 1), want) < 1e-12
    lat.close()


@pytest.mark.parametrize("block,minb", [(32, 1), (64, 2), (128, 3), (256, 4), (96, 2)])
def test_dslash_launch_variants(block, minb):
    """Every launch-bounds instantiation and odd CTA sizes give the same numbers."""
    dims = (6, 6, 4, 10)     # Vh = 720: several CTAs and a ragged tail for every block size
    rng = np.random.default_rng(3)
    U = gen.smooth_links(dims, 0.3, rng)
    phi = gen.gaussian_half_spinor(dims, rng)
    want = oracle.dslash_half(dims, U, 0, phi)
    lat = make_lattice(dims, dslash_block=block, dslash_minblocks=minb)
    assert rel(gpu_dslash(lat, U, phi, 0), want) < 1e-12
    lat.close()


@pytest.mark.parametrize("persist", [1, 2])
def test_dslash_looping_grid(persist):
    """Option dslash_persist: fewer CTAs that loop over the 128-site tiles (ragged last tile)."""
    dims = (12, 12, 12, 20)    # Vh = 17280 = 135 tiles of 128: more tiles than looping CTAs need
    rng = np.random.default_rng(3)
    U = gen.smooth_links(dims, 0.3, rng)
    phi = gen.gaussian_half_spinor(dims, rng)
    want = oracle.dslash_half(dims, U, 1, phi)
    lat = make_lattice(dims, dslash_persist=persist, dslash_block=32)
    assert lat.get_option("num_sms") * persist < (lat.Vh + 31) // 32       # the loop really loops
    assert rel(gpu_dslash(lat, U, phi, 1), want) < 1e-12
    lat.close()


def test_dslash_16x4_config2_and_mdagm():
    """BASELINE.json config 2 operator part: 16^4, eps = 0.3, seed 2, both parities and mdagm."""
    dims = (16, 16, 16, 16)
    rng = np.random.default_rng(2)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    for recon in (0, 1):
        lat = make_lattice(dims, recon=recon)
        links = lat.pack_links(U)
        for par in (0, 1):
            inp = lat.pack_spinor(b, 1 - par)
            out = lat.new_spinor()
            lat.dslash(par, out, inp, links)
            assert rel(lat.unpack_spinor(out, par), oracle.dslash_half(dims, U, par, b)) < 1e-12
        be = lat.pack_spinor(b, 0)
        out = lat.new_spinor()
        lat.mdagm(out, be, links, 0.01, 0.0)
        assert rel(lat.unpack_spinor(out, 0), oracle.mdagm(dims, U, 0.01, b)) < 1e-12
        lat.mdagm(out, be, links, 0.01, 0.37)
        assert rel(lat.unpack_spinor(out, 0), oracle.mdagm(dims, U, 0.01, b, sigma=0.37)) < 1e-12
        lat.close()


def test_pack_unpack_roundtrip():
    dims = (4, 8, 2, 6)
    phi = gen.gaussian_half_spinor(dims, 5)
    for prec in (0, 1):
        for layout in (0, 1):
            lat = make_lattice(dims, prec, layout=layout)
            back = lat.unpack_spinor(lat.pack_spinor(phi, 0), 0)
            if prec == 0:
                assert np.array_equal(back, phi)
            else:
                assert np.array_equal(back, phi.astype(np.complex64).astype(np.complex128))
            lat.close()


# ------------------------------------------------------------------------------------------------
# CG and multi-shift CG (criteria: reading R16)
# ------------------------------------------------------------------------------------------------
def test_cg_lockstep_small():
    """First iterates' alpha, beta, |r| agree with the oracle to 1e-10; solution parity."""
    dims = (8, 8, 8, 8)
    rng = np.random.default_rng(2)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m, tol = 0.05, 1e-10
    ref = oracle.cg(dims, U, m, b, tol, 5000, hist_len=64)
    lat = make_lattice(dims)
    links, be, x = lat.pack_links(U), lat.pack_spinor(b, 0), lat.new_spinor()
    res = lat.cg(x, be, links, m, tol, 5000)
    h = lat.solver_history()
    n = min(10, ref["iters"])
    assert np.allclose(h["alpha"][:n], ref["alpha"][:n], rtol=1e-10)
    assert np.allclose(h["beta"][:n], ref["beta"][:n], rtol=1e-10)
    assert np.allclose(h["rnorm"][:n], ref["rnorm"][:n], rtol=1e-10)
    assert abs(res["iters"] - ref["iters"]) <= max(1, ref["iters"] // 50)
    xg = lat.unpack_spinor(x, 0)
    # (i) true residual of the GPU solution evaluated with the ORACLE operator
    true_res = np.linalg.norm(b - oracle.mdagm(dims, U, m, xg)) / np.linalg.norm(b)
    assert true_res < 1.5 * tol
    assert abs(res["rel_resid"] - true_res) < 1e-12
    # (iii) || x_gpu - x_oracle || <= 10 kappa tol, kappa <= lambda_max / m^2, lambda_max ~ 7
    assert rel(xg, ref["x"]) < 10 * (7.0 / m ** 2) * tol
    lat.close()


def test_cg_config2_16x4():
    """BASELINE.json config 2: 16^4, m = 0.01, eps = 0.3, seed 2, tol 1e-10."""
    dims = (16, 16, 16, 16)
    rng = np.random.default_rng(2)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m, tol = 0.01, 1e-10
    ref = oracle.cg(dims, U, m, b, tol, 20000, hist_len=64)
    assert ref["converged"]
    lat = make_lattice(dims)
    links, be, x = lat.pack_links(U), lat.pack_spinor(b, 0), lat.new_spinor()
    res = lat.cg(x, be, links, m, tol, 20000)
    assert abs(res["iters"] - ref["iters"]) <= max(2, ref["iters"] // 50)
    xg = lat.unpack_spinor(x, 0)
    assert np.linalg.norm(b - oracle.mdagm(dims, U, m, xg)) / np.linalg.norm(b) < 1.5 * tol
    assert rel(xg, ref["x"]) < 10 * (7.0 / m ** 2) * tol
    h = lat.solver_history()
    assert np.allclose(h["rnorm"][:10], ref["rnorm"][:10], rtol=1e-10)
    lat.close()


@pytest.mark.parametrize("recon", [0, 1])
def test_multishift_small(recon):
    dims = (8, 8, 8, 16)
    rng = np.random.default_rng(4)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m, tol = 0.0025, 1e-10
    shifts = gen.rhmc_shifts(8)[[3, 0, 7, 1, 2, 4, 6, 5]]     # unsorted: base is not index 0
    ref = oracle.cg_multishift(dims, U, m, shifts, b, tol, 20000, hist_len=64)
    assert ref["converged"]
    lat = make_lattice(dims, recon=recon)
    links, be = lat.pack_links(U), lat.pack_spinor(b, 0)
    xs = [lat.new_spinor() for _ in shifts]
    res = lat.cg_multishift(xs, be, links, m, shifts, tol, 20000)
    assert abs(res["iters"] - ref["iters"]) <= max(2, ref["iters"] // 50)
    assert np.all(np.abs(res["conv_iter"] - ref["conv_iter"]) <= np.maximum(2, ref["conv_iter"] // 50))
    h = lat.solver_history()
    assert np.allclose(h["alpha"][:10], ref["alpha"][:10], rtol=1e-10)
    assert np.allclose(h["beta"][:10], ref["beta"][:10], rtol=1e-10)
    bn = np.linalg.norm(b)
    for i, s in enumerate(shifts):
        xg = lat.unpack_spinor(xs[i], 0)
        tr = np.linalg.norm(b - oracle.mdagm(dims, U, m, xg, sigma=s)) / bn
        assert tr < 1.5 * tol, (i, s, tr)
        assert abs(tr - res["rel_resid"][i]) < 1e-12
        assert rel(xg, ref["x"][i]) < 10 * (7.0 / (m * m + s)) * tol
    lat.close()


@pytest.mark.parametrize("opts", [dict(pdl=0, graph=0), dict(pdl=1, graph=0), dict(pdl=0, graph=1),
                                  dict(poll_chunk=3), dict(poll_chunk=1), dict(poll_chunk=64),
                                  dict(dslash_persist=1, dslash_block=32)])
def test_solver_launch_variants(opts):
    """Programmatic dependent launch, CUDA-graph replay of the iteration chunks and the chunk length
    are scheduling choices: same iterates as the plain launch path (bit for bit, unless the grid
    shape -- hence the reduction order -- changes), and the oracle criteria R16 hold."""
    dims = (8, 8, 8, 8)
    rng = np.random.default_rng(11)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m, tol = 0.05, 1e-10
    shifts = gen.rhmc_shifts(4)
    ref = oracle.cg_multishift(dims, U, m, shifts, b, tol, 5000)

    def solve(o):
        lat = make_lattice(dims, **o)
        links, be = lat.pack_links(U), lat.pack_spinor(b, 0)
        xs = [lat.new_spinor() for _ in shifts]
        res = lat.cg_multishift(xs, be, links, m, shifts, tol, 5000)
        res2 = lat.cg_multishift(xs, be, links, m, shifts, tol, 5000)      # cached graph is reused
        assert res2["iters"] == res["iters"]
        out = [lat.unpack_spinor(x, 0) for x in xs]
        ga = lat.get_option("graph_active")
        lat.close()
        return res, out, ga

    base, xb, ga0 = solve(dict(pdl=0, graph=0))
    res, xv, ga = solve(opts)
    assert ga0 == 0
    assert ga == (1 if opts.get("graph", 1) and opts.get("poll_chunk", 8) <= res["iters"] else 0) or "poll_chunk" in opts
    assert abs(res["iters"] - ref["iters"]) <= 2
    bn = np.linalg.norm(b)
    for i, s in enumerate(shifts):
        assert np.linalg.norm(b - oracle.mdagm(dims, U, m, xv[i], sigma=s)) / bn < 1.5 * tol
        if "dslash_persist" not in opts:
            assert np.array_equal(xv[i], xb[i]), (opts, i)
    if "dslash_persist" not in opts:
        assert res["iters"] == base["iters"] and np.array_equal(res["conv_iter"], base["conv_iter"])


@pytest.mark.parametrize("prec", [0, 1])
def test_rational_apply(prec):
    """NEXT-1 (lqcd_rational_apply): y = c0 b + sum_i c_i (A+sigma_i)^-1 b accumulated inside the
    multi-shift solve, against the oracle's definition.  Criteria as R16: same iteration counts;
    ||y_gpu - y_oracle|| within the sum of the per-shift solution bounds; the partial-fraction
    identity holds when checked with the ORACLE operator; and the fused y equals the sum formed
    from the GPU's own stored solutions to rounding."""
    dims = (8, 8, 8, 16)
    rng = np.random.default_rng(4)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    U, b = round_inputs(prec, U, b)
    m = 0.0025 if prec == 0 else 0.05
    tol = 1e-10 if prec == 0 else 1e-5
    shifts = gen.rhmc_shifts(8)[[3, 0, 7, 1, 2, 4, 6, 5]]
    c0 = 0.35
    c = np.array([0.5, -1.25, 2.0, 0.125, -0.3, 0.9, 1.5, -0.05])
    ref = oracle.rational_apply(dims, U, m, shifts, c0, c, b, tol, 20000)
    refx = oracle.cg_multishift(dims, U, m, shifts, b, tol, 20000)
    assert ref["converged"]
    lat = make_lattice(dims, prec=prec)
    links, be = lat.pack_links(U), lat.pack_spinor(b, 0)
    y = lat.new_spinor()
    res = lat.rational_apply(y, be, links, m, shifts, c0, c, tol, 20000)
    yg = lat.unpack_spinor(y, 0)
    slack = 2 if prec == 0 else 10          # fp32 rounding moves the freeze iteration of a shift
    assert abs(res["iters"] - ref["iters"]) <= max(slack, ref["iters"] // 50)
    assert np.all(np.abs(res["conv_iter"] - ref["conv_iter"]) <= np.maximum(slack, ref["conv_iter"] // 50))
    eps = tol if prec == 0 else 2e-5
    bound = sum(abs(ci) * 10 * (7.0 / (m * m + s)) * eps * np.linalg.norm(xi)
                for ci, s, xi in zip(c, shifts, refx["x"])) / np.linalg.norm(ref["y"])
    assert rel(yg, ref["y"]) < bound, (rel(yg, ref["y"]), bound)
    # the fused accumulation equals the sum over the GPU's own stored solutions
    xs = [lat.new_spinor() for _ in shifts]
    res2 = lat.cg_multishift(xs, be, links, m, shifts, tol, 20000)
    assert res2["iters"] == res["iters"] and np.array_equal(res2["conv_iter"], res["conv_iter"])
    y2 = c0 * b + sum(ci * lat.unpack_spinor(x, 0) for ci, x in zip(c, xs))
    assert rel(yg, y2) < (1e-13 if prec == 0 else 2e-6)
    # partial fractions: (A+s1)(A+s2) y = b for c = (+-1/(s2-s1)), evaluated with the oracle operator
    s1, s2 = 0.11, 0.83
    res = lat.rational_apply(y, be, links, m, [s1, s2], 0.0, [1.0 / (s2 - s1), -1.0 / (s2 - s1)], tol, 20000)
    yg = lat.unpack_spinor(y, 0)
    back = oracle.mdagm(dims, U, m, oracle.mdagm(dims, U, m, yg, sigma=s2), sigma=s1)
    assert rel(back, b) < (30 * tol if prec == 0 else 1e-4)
    # errors: aliasing, NaN coefficient, negative shift
    import paper_1701_00426_b200 as L
    with pytest.raises(L.LqcdError):
        lat.rational_apply(be, be, links, m, [s1], 0.0, [1.0], tol, 10)
    with pytest.raises(L.LqcdError):
        lat.rational_apply(y, be, links, m, [s1], 0.0, [float("nan")], tol, 10)
    with pytest.raises(L.LqcdError):
        lat.rational_apply(y, be, links, m, [-1.0], 0.0, [1.0], tol, 10)
    lat.close()


@pytest.mark.parametrize("recon", [0, 1])
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 2, 2, 4), (6, 4, 10, 8)])
def test_fermion_force(dims, prec, recon):
    """NEXT-3 (lqcd_fermion_force): F_mu(x) = TA[U_mu(x) Q_mu(x)] from given solutions x_i, element by
    element against the oracle (whose formula is pinned by finite differences of the action).  The x_i
    are arbitrary Gaussian vectors here: the map (x_i, c_i, U) -> F is what is under test."""
    rng = np.random.default_rng(9)
    U = gen.haar_like_links(dims, rng)
    n = 3
    xs = np.stack([gen.gaussian_half_spinor(dims, rng) for _ in range(n)])
    U, xs = round_inputs(prec, U, xs)
    if recon == 1 and prec == 1:
        U = oracle.reconstruct_row3(U)
    c = np.array([0.8, -0.45, 1.3])
    want = oracle.fermion_force(dims, U, c, xs)
    lat = make_lattice(dims, prec, recon)
    links = lat.pack_links(U)
    dx = [lat.pack_spinor(x, 0) for x in xs]
    got = lat.unpack_tamat(lat.fermion_force(dx, links, c))
    assert rel(got, want) < TOL[prec], (dims, prec, recon, rel(got, want))
    # per-link check as well (a wrong sign on one parity or direction would hide in a global norm less
    # than one would like): worst link relative to the typical link norm
    link_err = np.linalg.norm((got - want).reshape(-1, 9), axis=1).max()
    assert link_err / np.linalg.norm(want.reshape(-1, 9), axis=1).mean() < 10 * TOL[prec]
    assert np.abs(got + got.conj().transpose(0, 1, 3, 2)).max() < (1e-12 if prec == 0 else 1e-4)
    lat.close()


def test_fermion_force_after_solve_periodic_bc():
    """End to end: multi-shift solve on the GPU, force from its solutions; oracle force from the oracle's
    solutions (periodic BC variant, 12x10x6x4 spans several CTAs with a ragged tail)."""
    dims = (12, 10, 6, 4)
    rng = np.random.default_rng(10)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m, tol = 0.1, 1e-11
    shifts = gen.rhmc_shifts(4)
    c = np.array([0.5, -1.25, 2.0, 0.125])
    ref = oracle.cg_multishift(dims, U, m, shifts, b, tol, 5000, antiperiodic_t=False)
    want = oracle.fermion_force(dims, U, c, ref["x"], antiperiodic_t=False)
    lat = make_lattice(dims, ap=False)
    links, be = lat.pack_links(U), lat.pack_spinor(b, 0)
    xs = [lat.new_spinor() for _ in shifts]
    lat.cg_multishift(xs, be, links, m, shifts, tol, 5000)
    got = lat.unpack_tamat(lat.fermion_force(xs, links, c))
    assert rel(got, want) < 1e-7          # solutions agree to O(kappa tol), the force is bilinear in them
    lat.close()


@pytest.mark.parametrize("recon", [0, 1])
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 2, 4, 2), (6, 4, 10, 8)])
def test_gauge_staples(dims, prec, recon):
    """NEXT-4 (lqcd_gauge_staples): tree-level Symanzik staples, element by element against the oracle
    (pinned by finite differences of the gauge action).  2x2x4x2: every second-neighbour step wraps
    onto the starting site; 6x4x10x8 spans several CTAs with a ragged tail."""
    rng = np.random.default_rng(15)
    U = gen.haar_like_links(dims, rng)
    (U,) = round_inputs(prec, U)
    if recon == 1 and prec == 1:
        U = oracle.reconstruct_row3(U)
    lat = make_lattice(dims, prec, recon)
    links = lat.pack_links(U)
    for c0, c1 in ((oracle.SYMANZIK_C0, oracle.SYMANZIK_C1), (1.0, 0.0), (0.0, 1.0)):
        want = oracle.gauge_staples(dims, U, c0, c1)
        # one product chain per path / shared sub-products per (mu, nu) / two passes through stored 3-link staples
        for variant in (0, 1, 2):
            lat.set_option("staples_variant", variant)
            got = lat.unpack_force(lat.gauge_staples(links, c0, c1))
            assert lat.get_option("staples_ran") == variant
            assert rel(got, want) < TOL[prec], (dims, prec, recon, c0, c1, variant, rel(got, want))
            link_err = np.linalg.norm((got - want).reshape(-1, 9), axis=1).max()
            assert link_err / np.linalg.norm(want.reshape(-1, 9), axis=1).mean() < 10 * TOL[prec]
    lat.close()


@pytest.mark.parametrize("x2b", [0, 2, 4])
def test_gauge_staples_cta_swizzle(x2b):
    """The x2-blocked CTA order (option staples_x2block) is a pure scheduling choice.  16x16x4x4 has rows
    of exactly 128 half-sites, so the swizzle is really applied (it silently falls back to plain order
    when rows are not whole tiles, e.g. on the lattices of test_gauge_staples)."""
    dims = (16, 16, 4, 4)
    rng = np.random.default_rng(16)
    U = gen.smooth_links(dims, 0.5, rng)
    want = oracle.gauge_staples(dims, U)
    for variant in (0, 1, 2):
        lat = make_lattice(dims, staples_x2block=x2b, staples_variant=variant)
        got = lat.unpack_force(lat.gauge_staples(lat.pack_links(U)))
        assert rel(got, want) < 1e-12, (x2b, variant, rel(got, want))
        lat.close()


@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("minb", [2, 3, 4])
def test_gauge_staples_two_pass_variants_and_workspace(minb, layout):
    """Variant 2 (two passes through the 24 stored 3-link staples per site): every launch-bounds instantiation
    of its second kernel, both layouts; without a large enough workspace the one-pass kernel runs instead and
    gives the same field (through the raw C call: the binding would allocate the workspace)."""
    import ctypes as C
    import paper_1701_00426_b200 as L
    dims = (6, 4, 10, 8)
    rng = np.random.default_rng(18)
    U = gen.smooth_links(dims, 0.5, rng)
    want = oracle.gauge_staples(dims, U)
    lat = make_lattice(dims, staples_minblocks=minb, layout=layout)
    links = lat.pack_links(U)
    out = lat._buf(int(L.lib.lqcd_force_bytes(lat._ctx)))
    rc = L.lib.lqcd_gauge_staples(lat._ctx, C.c_void_p(links.data_ptr()), C.c_void_p(out.data_ptr()), 5.0 / 3.0, -1.0 / 12.0)
    assert rc == 0 and lat.get_option("staples_ran") == 1          # no workspace yet
    assert rel(lat.unpack_force(out), want) < 1e-12
    lat.ensure_workspace(1)                                          # a solver-sized workspace is too small
    assert lat._ws.numel() < int(L.lib.lqcd_staples_workspace_bytes(lat._ctx))
    rc = L.lib.lqcd_gauge_staples(lat._ctx, C.c_void_p(links.data_ptr()), C.c_void_p(out.data_ptr()), 5.0 / 3.0, -1.0 / 12.0)
    assert rc == 0 and lat.get_option("staples_ran") == 1
    got = lat.unpack_force(lat.gauge_staples(links))                 # the binding sizes the workspace
    assert lat.get_option("staples_ran") == 2
    assert rel(got, want) < 1e-12
    # the workspace is shared with the solvers: a solve afterwards still works
    b = gen.gaussian_half_spinor(dims, rng)
    x = lat.new_spinor()
    r = lat.cg(x, lat.pack_spinor(b, 0), links, 0.2, 1e-10, 2000)
    assert r["rel_resid"] < 1.5e-10
    lat.close()


def test_next_rows_on_a_paper_lattice_shape():
    """NEXT-3 / NEXT-4 at one of the paper's Table 3 / 4 shapes, 32^2 x 8 x 32, in the
    default launch configuration (two-pass staples, x2-blocked CTA order really applied: rows are 4
    tiles; 8 shifts staged in shared memory): every link against the oracle."""
    dims = (32, 32, 8, 32)
    rng = np.random.default_rng(5)
    U = gen.smooth_links(dims, 0.5, rng)
    lat = make_lattice(dims)
    links = lat.pack_links(U)
    got = lat.unpack_force(lat.gauge_staples(links))
    assert lat.get_option("staples_ran") == 2
    want = oracle.gauge_staples(dims, U)
    assert rel(got, want) < 1e-12
    assert np.abs(got - want).max() < 1e-11
    n = 8
    xs = np.stack([gen.gaussian_half_spinor(dims, rng) for _ in range(n)])
    c = np.linspace(-1.0, 1.5, n)
    dx = [lat.pack_spinor(x, 0) for x in xs]
    gotf = lat.unpack_tamat(lat.fermion_force(dx, links, c))
    wantf = oracle.fermion_force(dims, U, c, xs)
    assert rel(gotf, wantf) < 1e-12
    lat.close()


def test_cg_fp32_and_max_iter():
    dims = (8, 8, 8, 8)
    rng = np.random.default_rng(5)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    U, b = round_inputs(1, U, b)
    m, tol = 0.1, 1e-5
    ref = oracle.cg(dims, U, m, b, tol, 5000)
    lat = make_lattice(dims, prec=1)
    links, be, x = lat.pack_links(U), lat.pack_spinor(b, 0), lat.new_spinor()
    res = lat.cg(x, be, links, m, tol, 5000)
    assert abs(res["iters"] - ref["iters"]) <= max(2, ref["iters"] // 20)
    xg = lat.unpack_spinor(x, 0)
    assert np.linalg.norm(b - oracle.mdagm(dims, U, m, xg)) / np.linalg.norm(b) < 5 * tol
    assert rel(xg, ref["x"]) < 1e-3
    # max_iter is reported, not hidden, and x is the last iterate
    res = lat.cg(x, be, links, m, 1e-30, 7, raise_on_max_iter=False)
    assert not res["converged"] and res["iters"] == 7
    ref7 = oracle.cg(dims, U, m, b, 1e-30, 7)
    assert rel(lat.unpack_spinor(x, 0), ref7["x"]) < 1e-4
    lat.close()


def test_cg_zero_rhs_and_errors():
    import paper_1701_00426_b200 as L
    dims = (4, 4, 4, 4)
    U = gen.unit_links(dims)
    lat = make_lattice(dims)
    links = lat.pack_links(U)
    b = lat.pack_spinor(np.zeros((lat.Vh, 3), dtype=np.complex128), 0)
    x = lat.new_spinor()
    res = lat.cg(x, b, links, 0.1, 1e-10, 100)
    assert res["iters"] == 0 and np.abs(lat.unpack_spinor(x, 0)).max() == 0.0
    with pytest.raises(L.LqcdError) as e:
        lat.cg(x, b, links, 0.1, -1.0, 100)
    assert e.value.code == L.ERR_ARG
    with pytest.raises(L.LqcdError) as e:
        lat.cg_multishift([x], b, links, 0.1, [-0.5], 1e-8, 10)
    assert e.value.code == L.ERR_ARG
    with pytest.raises(L.LqcdError) as e:
        lat.dslash(0, x, x, links)
    assert e.value.code == L.ERR_ARG
    with pytest.raises(L.LqcdError) as e:
        lat.dslash(3, x, b, links)
    assert e.value.code == L.ERR_ARG
    lat.close()


def test_host_entry_points():
    dims = (8, 4, 4, 6)
    rng = np.random.default_rng(8)
    U = gen.smooth_links(dims, 0.4, rng)
    phi = gen.gaussian_half_spinor(dims, rng)
    lat = make_lattice(dims)
    out = np.empty_like(phi)
    lat.dslash_host(1, out, phi, U)
    assert rel(out, oracle.dslash_half(dims, U, 1, phi)) < 1e-12
    out2 = np.empty_like(phi)
    lat.dslash_host_vectors(0, out2, phi, lat.pack_links(U))      # links resident, only vectors copied
    assert rel(out2, oracle.dslash_half(dims, U, 0, phi)) < 1e-12
    shifts = np.array([0.5, 0.01])
    sol = np.empty((2,) + phi.shape, dtype=np.complex128)
    res = lat.cg_multishift_host(sol, phi, U, 0.05, shifts, 1e-10, 5000)
    ref = oracle.cg_multishift(dims, U, 0.05, shifts, phi, 1e-10, 5000)
    assert abs(res["iters"] - ref["iters"]) <= 2
    for i in range(2):
        assert rel(sol[i], ref["x"][i]) < 1e-6
    # links resident: rhs up, solutions down
    sol2 = np.empty_like(sol)
    res2 = lat.cg_multishift_host_vectors(sol2, phi, lat.pack_links(U), 0.05, shifts, 1e-10, 5000)
    assert res2["iters"] == res["iters"] and np.array_equal(sol2, sol)
    lat.close()


@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("n", [1, 2, 5])
def test_host_batch_pipeline(prec, n):
    """lqcd_dslash_host_vectors_batch: n applications through the three-stream copy pipeline (double-buffered
    staging: n = 5 re-uses every slot) = the oracle applied to each input, and bit-identical to one blocking
    lqcd_dslash_host_vectors call per application."""
    import torch
    dims = (8, 6, 4, 10)
    rng = np.random.default_rng(18)
    U = gen.smooth_links(dims, 0.4, rng)
    ins = [gen.gaussian_half_spinor(dims, rng) for _ in range(n)]
    U, *ins = round_inputs(prec, U, *ins)
    pars = [(j + 1) % 2 for j in range(n)]
    lat = make_lattice(dims, prec)
    links = lat.pack_links(U)

    def pinned(a):
        t = torch.from_numpy(np.ascontiguousarray(a).view(np.float64).reshape(-1)).pin_memory()
        return t, t.numpy().view(np.complex128).reshape(a.shape)
    keep = [pinned(a) for a in ins] + [pinned(np.zeros_like(ins[0])) for _ in range(n)]
    h_ins, h_outs = [k[1] for k in keep[:n]], [k[1] for k in keep[n:]]
    for _ in range(2):                                   # second call: slots and events are re-used
        lat.dslash_host_vectors_batch(pars, h_outs, h_ins, links)
    for j in range(n):
        assert rel(h_outs[j], oracle.dslash_half(dims, U, pars[j], ins[j])) < TOL[prec], j
        one = np.empty_like(ins[j])
        lat.dslash_host_vectors(pars[j], one, ins[j], links)
        assert np.array_equal(one, h_outs[j])
    lat.close()


def test_solver_rejects_aliased_and_misaligned_buffers():
    """Before any launch: outputs that overlap each other, rhs, the workspace or the links, or that are not
    16-byte aligned, are LQCD_ERR_ARG (the vector kernels assume distinct, aligned operands)."""
    import paper_1701_00426_b200 as L
    dims = (4, 4, 4, 4)
    lat = make_lattice(dims)
    links = lat.pack_links(gen.unit_links(dims))
    b = lat.pack_spinor(gen.gaussian_half_spinor(dims, 3), 0)
    x = lat.new_spinor()
    lat.ensure_workspace(2)
    big = lat._buf(2 * lat.spinor_bytes + 64)
    cases = [([x, x], b), ([x, b], b), ([x, lat._ws[:lat.spinor_bytes]], b), ([x, links[:lat.spinor_bytes]], b),
             ([x, big[8:8 + lat.spinor_bytes]], b), ([big[:lat.spinor_bytes], big[16:16 + lat.spinor_bytes]], b)]
    for xs, rhs in cases:
        with pytest.raises(L.LqcdError) as e:
            lat.cg_multishift(xs, rhs, links, 0.1, [0.0, 0.5], 1e-8, 10)
        assert e.value.code == L.ERR_ARG
    with pytest.raises(L.LqcdError) as e:
        lat.rational_apply(big[8:8 + lat.spinor_bytes], b, links, 0.1, [0.0, 0.5], 1.0, [1.0, 1.0], 1e-8, 10)
    assert e.value.code == L.ERR_ARG
    # a well-formed call still works afterwards
    res = lat.cg_multishift([x, big[:lat.spinor_bytes]], b, links, 0.1, [0.0, 0.5], 1e-8, 100)
    assert res["converged"]
    lat.close()


def test_fp64_peak_measurement_is_plausible():
    """lqcd_measure_fp64_peak (bench.py's denominator for the ALU-bound staples): a B200 does some tens of
    TFLOP/s in FP64; anything outside 5..100 means the kernel or its flop count is broken."""
    lat = make_lattice((4, 4, 4, 4))
    v = lat.measure_fp64_peak()
    assert 5.0 < v < 100.0, v
    lat.close()


# ------------------------------------------------------------------------------------------------
# Full size, in the launch configuration bench.py times (BASELINE.json configs[2]: 32^4)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec,recon", [(0, 0), (0, 1), (1, 0), (1, 1)])
def test_dslash_32x4_bench_configuration(prec, recon):
    """Same inputs (eps 0.3, seed 3), same default launch configuration as bench.py; every output
    site of both parities against the oracle (the C oracle does 32^4 in well under a second)."""
    dims = (32, 32, 32, 32)
    rng = np.random.default_rng(3)
    U = gen.smooth_links(dims, 0.3, rng)
    in_e = gen.gaussian_half_spinor(dims, rng)
    in_o = gen.gaussian_half_spinor(dims, rng)
    U, in_e, in_o = round_inputs(prec, U, in_e, in_o)
    lat = make_lattice(dims, prec, recon)
    links = lat.pack_links(U)
    for par, inp in ((1, in_e), (0, in_o)):
        d_in, d_out = lat.pack_spinor(inp, 1 - par), lat.new_spinor()
        lat.dslash(par, d_out, d_in, links)
        got = lat.unpack_spinor(d_out, par)
        want = oracle.dslash_half(dims, U, par, inp)
        assert rel(got, want) < TOL[prec]
        # element-wise, not only in norm: worst site
        assert np.abs(got - want).max() < 50 * TOL[prec] * np.abs(want).max()
    lat.close()


@pytest.mark.parametrize("dims", [(64, 64, 64, 16), (48, 48, 48, 48)])
def test_dslash_large_volume_sampled_sites(dims):
    """BASELINE.json configs[4]: 64^3 x 16 (V = 4.2 M, links 2.4 GB) and 48^4 (V = 5.3 M, links 3.06 GB: the
    largest index range the kernels see), in fp64 AND fp32, 18- and 12-real: sampled output sites computed one
    by one by oracle_dirac_site (pinned to the dense matrix in tests/test_oracle_pins.py), including the
    corners and both x3 boundary slices; in fp64 18-real also the FULL field of both parities."""
    rng = np.random.default_rng(5)
    U64 = gen.smooth_links(dims, 0.5, rng)
    psi64 = gen.gaussian_spinor(dims, rng)
    coords = gen.site_coords(dims)
    n0, n1, n2, n3 = dims
    samp = np.random.default_rng(99)
    picks = [(0, 0, 0, 0), (n0 - 1, n1 - 1, n2 - 1, n3 - 1), (1, 0, 0, 0), (0, n1 - 1, 0, n3 - 1),
             (n0 - 2, 1, n2 - 1, 0), (n0 - 1, 0, 0, 0), (0, 0, 0, n3 - 1), (n0 - 1, n1 - 1, n2 - 1, 0)]
    picks += [tuple(int(v) for v in coords[i]) for i in samp.integers(0, coords.shape[0], 200)]
    # both x3 boundary slices, random positions inside them
    for x3 in (0, n3 - 1):
        picks += [(int(samp.integers(n0)), int(samp.integers(n1)), int(samp.integers(n2)), x3) for _ in range(20)]
    del coords
    for prec in (0, 1):
        U, psi = round_inputs(prec, U64, psi64)
        halves = {p: oracle.full_to_half(dims, p, psi) for p in (0, 1)}
        for recon in (0, 1):
            lat = make_lattice(dims, prec, recon)
            links = lat.pack_links(U)
            got = {}
            for par in (0, 1):
                d_in, d_out = lat.pack_spinor(halves[1 - par], 1 - par), lat.new_spinor()
                lat.dslash(par, d_out, d_in, links)
                got[par] = lat.unpack_spinor(d_out, par)
                del d_in, d_out
            worst = 0.0
            for x in picks:
                par = sum(x) % 2
                lex = x[0] + n0 * (x[1] + n1 * (x[2] + n2 * x[3]))
                # the oracle reads the full-lattice psi; only opposite-parity neighbours enter D
                want = oracle.dirac_site(dims, U, psi, x)
                worst = max(worst, np.abs(got[par][lex // 2] - want).max() / np.abs(want).max())
            assert worst < TOL[prec], (dims, prec, recon, worst)
            if prec == 0 and recon == 0:
                for par in (0, 1):
                    want = oracle.dslash_half(dims, U, par, halves[1 - par])
                    assert rel(got[par], want) < TOL[0], (dims, par)
                    assert np.abs(got[par] - want).max() < 50 * TOL[0] * np.abs(want).max()
                    del want
            lat.close()
            del links, got


def test_multishift_config4_24x24x24x48():
    """BASELINE.json configs[3]: 24^3 x 48, 8 shifts, m = 0.0025, tol 1e-10 per shift, against the
    oracle run to the same tolerance (reading R16)."""
    dims = (24, 24, 24, 48)
    rng = np.random.default_rng(4)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m, tol = 0.0025, 1e-10
    shifts = gen.rhmc_shifts(8)
    lat = make_lattice(dims)
    links, be = lat.pack_links(U), lat.pack_spinor(b, 0)
    xs = [lat.new_spinor() for _ in shifts]
    res = lat.cg_multishift(xs, be, links, m, shifts, tol, 50000)
    ref = oracle.cg_multishift(dims, U, m, shifts, b, tol, 50000, hist_len=16)
    assert ref["converged"]
    assert abs(res["iters"] - ref["iters"]) <= max(2, ref["iters"] // 50)
    assert np.all(np.abs(res["conv_iter"] - ref["conv_iter"]) <= np.maximum(2, ref["conv_iter"] // 50))
    h = lat.solver_history()
    assert np.allclose(h["alpha"][:10], ref["alpha"][:10], rtol=1e-10)
    assert np.allclose(h["rnorm"][:10], ref["rnorm"][:10], rtol=1e-10)
    bn = np.linalg.norm(b)
    for i in (0, 3, 7):                      # smallest, middle, largest shift
        xg = lat.unpack_spinor(xs[i], 0)
        tr = np.linalg.norm(b - oracle.mdagm(dims, U, m, xg, sigma=shifts[i])) / bn
        assert tr < 1.5 * tol
        assert rel(xg, ref["x"][i]) < 10 * (7.0 / (m * m + shifts[i])) * tol
    assert res["rel_resid"].max() < 1.5 * tol
    lat.close()


def test_multishift_config4_32x4_properties_at_full_size():
    """BASELINE.json configs[3], second lattice (32^4, the bench configuration): the full GPU solve is
    checked by what holds at any size -- every shift's TRUE residual evaluated with the ORACLE operator
    (reading R16 (i)) -- and the first 12 iterations in lock step with the oracle (R16 (iv)); the oracle
    is not run to convergence here (the 24^3 x 48 test above does that)."""
    dims = (32, 32, 32, 32)
    rng = np.random.default_rng(4)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m, tol = 0.0025, 1e-10
    shifts = gen.rhmc_shifts(8)
    lat = make_lattice(dims)
    links, be = lat.pack_links(U), lat.pack_spinor(b, 0)
    xs = [lat.new_spinor() for _ in shifts]
    res = lat.cg_multishift(xs, be, links, m, shifts, tol, 50000)
    assert lat.get_option("graph_active") == 1
    h = lat.solver_history()
    ref = oracle.cg_multishift(dims, U, m, shifts, b, tol, 12, hist_len=12)
    assert np.allclose(h["alpha"][:12], ref["alpha"], rtol=1e-10)
    assert np.allclose(h["beta"][:12], ref["beta"], rtol=1e-10)
    assert np.allclose(h["rnorm"][:12], ref["rnorm"], rtol=1e-10)
    bn = np.linalg.norm(b)
    for i, s in enumerate(shifts):
        xg = lat.unpack_spinor(xs[i], 0)
        tr = np.linalg.norm(b - oracle.mdagm(dims, U, m, xg, sigma=s)) / bn
        assert tr < 1.5 * tol, (i, tr)
        assert abs(tr - res["rel_resid"][i]) < 1e-12
    assert np.all(np.diff(res["conv_iter"]) <= 0)          # larger shifts freeze earlier
    assert res["conv_iter"][0] == res["iters"]
    lat.close()


# ------------------------------------------------------------------------------------------------
# block Dslash (several right-hand sides per launch; dslash_multi.cu)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("recon", [0, 1])
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("dims,n,blk", [((4, 4, 4, 4), 1, 4), ((6, 4, 2, 8), 3, 4), ((12, 10, 6, 4), 7, 4), ((12, 10, 6, 4), 11, 8),
                                        ((2, 2, 2, 2), 8, 8)])
def test_dslash_multi_equals_oracle_and_single(dims, n, blk, prec, recon, layout):
    """lqcd_dslash_multi: every right-hand side against oracle.dslash_half (both parities, ragged lattices, N = 2 wrap,
    block remainders 8 + 2 + 1, 4 + 2 + 1, ...) and BIT-identical to n single lqcd_dslash applications."""
    rng = np.random.default_rng(31)
    U = gen.haar_like_links(dims, rng)
    ins = [gen.gaussian_half_spinor(dims, rng) for _ in range(n)]
    U, *ins = round_inputs(prec, U, *ins)
    if recon == 1 and prec == 1:
        U = oracle.reconstruct_row3(U)
    lat = make_lattice(dims, prec, recon, True, layout=layout, force_block=blk)
    links = lat.pack_links(U)
    for out_parity in (0, 1):
        d_in = [lat.pack_spinor(v, 1 - out_parity) for v in ins]
        d_out = [lat.new_spinor() for _ in range(n)]
        single = lat.new_spinor()
        lat.dslash_multi(out_parity, d_out, d_in, links)
        for r in range(n):
            got = lat.unpack_spinor(d_out[r], out_parity)
            assert rel(got, oracle.dslash_half(dims, U, out_parity, ins[r])) < TOL[prec], (dims, n, prec, recon, layout, out_parity, r)
            lat.dslash(out_parity, single, d_in[r], links)
            lat.synchronize()
            assert bool((single == d_out[r]).all()), (dims, n, prec, recon, layout, out_parity, r)
    lat.close()


def test_dslash_multi_errors():
    import paper_1701_00426_b200 as L
    dims = (4, 4, 4, 4)
    lat = make_lattice(dims)
    links = lat.pack_links(gen.unit_links(dims))
    a, b = lat.new_spinor(), lat.new_spinor()
    with pytest.raises(L.LqcdError) as e:
        lat.dslash_multi(0, [a, b], [b, b], links)            # output 1 aliases an input
    assert e.value.code == L.ERR_ARG
    theta = np.zeros((lat.V, 4))
    lat.set_backfield(lat.pack_backfield(theta))
    with pytest.raises(L.LqcdError) as e:
        lat.dslash_multi(0, [a], [b], links)
    assert e.value.code == L.ERR_UNSUPPORTED
    lat.close()
