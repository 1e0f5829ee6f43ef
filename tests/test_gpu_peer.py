"""-m gpu: the slab path over the library's own peer-to-peer transport (lqcd_peer_*) on
ONE GPU.  Each of P "virtual ranks" is a SlabLattice(transport="peer") with its own context, stream, fields and
peer block on cuda:0, driven by its own host thread; the ranks hand one another the device addresses of their
blocks (connect_local), exactly as processes do with CUDA IPC handles.  Kernels of different ranks must never
wait for one another on one GPU, so the ranks run in LOCK STEP: lqcd_set_phase_hook calls back after every launch
that publishes to the peers, the thread finishes its stream there and meets the others at a barrier.  Every flag a
kernel waits for is therefore already raised when the kernel starts -- but the code that runs is the real one:
face pushes into the neighbours' landing buffers, the Dslash variant that reads them, the publish / gather of
the dot products inside the Dslash, K1 and K2 kernels, the counters.  With P = 1 (the rank is its own neighbour;
stream order raises every flag in time) the solve also runs WITHOUT the hook, from the chunk graph.
Results must equal the oracle on the GLOBAL lattice and every rank must take the same decisions."""
import threading

import numpy as np
import pytest

import lqcd_inputs as gen
import oracle

pytestmark = pytest.mark.gpu


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def run_peer_ranks(world, make, work, lockstep=True):
    """make(r) -> SlabLattice on every rank (main thread), connect, then work(r, slab) on `world` threads."""
    from paper_1701_00426_b200.slab import SlabLattice
    slabs = [make(r) for r in range(world)]
    SlabLattice.connect_local(slabs)
    barrier = threading.Barrier(world)
    errs, outs = [], [None] * world
    if lockstep:
        for s in slabs:
            s.set_lockstep(barrier)

    def run(r):
        try:
            outs[r] = work(r, slabs[r])
            slabs[r].lat.synchronize()
        except BaseException as e:  # noqa: BLE001
            errs.append(e)
            barrier.abort()

    ts = [threading.Thread(target=run, args=(r,)) for r in range(world)]
    for t in ts:
        t.start()
    for t in ts:
        t.join(300)
    for s in slabs:
        s.close()
    if errs:
        raise errs[0]
    return outs


@pytest.mark.parametrize("layout", [0, 1])
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("world", [1, 2, 4])
def test_peer_dslash_equals_global_oracle(world, prec, layout):
    from paper_1701_00426_b200.slab import SlabLattice
    dims = (8, 6, 4, 16)
    rng = np.random.default_rng(71)
    U = gen.smooth_links(dims, 0.3, rng)
    psi = gen.gaussian_spinor(dims, rng)
    if prec == 1:
        U, psi = (a.astype(np.complex64).astype(np.complex128) for a in (U, psi))
    tol = 1e-12 if prec == 0 else 1e-5
    for ap in (True, False):
        for gp_out in (0, 1):
            phi_in = oracle.full_to_half(dims, 1 - gp_out, psi)
            want = oracle.dslash_half(dims, U, gp_out, phi_in, antiperiodic_t=ap)
            got = np.zeros_like(want)
            lock = threading.Lock()

            def work(r, sl):
                links = sl.pack_links(U)
                inp = sl.pack_spinor(phi_in, 1 - gp_out)
                out = sl.new_spinor()
                sl.dslash(gp_out, out, inp, links)
                sl.dslash(gp_out, out, inp, links)            # a second exchange of the same kind: the counters move on
                with lock:
                    sl.unpack_spinor(out, gp_out, got)

            run_peer_ranks(world, lambda r: SlabLattice(dims, world, r, prec=prec, antiperiodic_t=ap, transport="peer",
                                                        options=dict(layout=layout)), work)
            assert rel(got, want) < tol, (world, prec, layout, ap, gp_out, rel(got, want))


@pytest.mark.parametrize("world,lockstep", [(1, False), (1, True), (2, True), (4, True)])
def test_peer_mdagm_multishift_rational(world, lockstep):
    """The solvers over the peer transport: same iterations and scalars as the oracle and as the single-context
    run, R16 criteria with the ORACLE operator on the gathered global solutions; identical decisions on all ranks."""
    import paper_1701_00426_b200 as L
    from paper_1701_00426_b200.slab import SlabLattice
    dims = (8, 8, 4, 8)
    rng = np.random.default_rng(72)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m, tol = 0.05, 1e-10
    shifts = gen.rhmc_shifts(4)[[2, 0, 3, 1]]
    ref = oracle.cg_multishift(dims, U, m, shifts, b, tol, 5000, hist_len=16)
    want_A = oracle.mdagm(dims, U, m, b, sigma=0.37)
    lat = L.Lattice(dims)
    res1 = lat.cg_multishift([lat.new_spinor() for _ in shifts], lat.pack_spinor(b, 0), lat.pack_links(U), m, shifts, tol, 5000)
    lat.close()

    got_A = np.zeros_like(b)
    got_x = [np.zeros_like(b) for _ in shifts]
    got_y = np.zeros_like(b)
    lock = threading.Lock()
    c0, c = 0.35, np.array([0.5, -1.25, 2.0, 0.125])

    def work(r, sl):
        links = sl.pack_links(U)
        be = sl.pack_spinor(b, 0)
        out = sl.new_spinor()
        sl.mdagm(out, be, links, m, 0.37)
        xs = [sl.new_spinor() for _ in shifts]
        res = sl.cg_multishift(xs, be, links, m, shifts, tol, 5000)
        hist = sl.lat.solver_history()
        graph = sl.lat.get_option("graph_active")
        y = sl.new_spinor()
        resy = sl.rational_apply(y, be, links, m, shifts, c0, c, tol, 5000)
        res_b = sl.cg_multishift(xs, be, links, m, shifts, tol, 5000)       # again: counters and slots carry on
        with lock:
            sl.unpack_spinor(out, 0, got_A)
            for i, x in enumerate(xs):
                sl.unpack_spinor(x, 0, got_x[i])
            sl.unpack_spinor(y, 0, got_y)
        return res, hist, resy, graph, res_b

    outs = run_peer_ranks(world, lambda r: SlabLattice(dims, world, r, transport="peer"), work, lockstep=lockstep)
    assert rel(got_A, want_A) < 1e-12
    bn = np.linalg.norm(b)
    for res, hist, resy, graph, res_b in outs:
        assert graph == (0 if lockstep else 1)          # without the hook the chunk graph stays on
        assert res["iters"] == outs[0][0]["iters"] and np.array_equal(res["conv_iter"], outs[0][0]["conv_iter"])
        assert res_b["iters"] == res["iters"] and np.array_equal(res_b["conv_iter"], res["conv_iter"])
        assert abs(res["iters"] - ref["iters"]) <= 2 and abs(res["iters"] - res1["iters"]) <= 1
        assert resy["iters"] == res["iters"]
        assert np.allclose(hist["alpha"][:10], ref["alpha"][:10], rtol=1e-10)
        assert np.allclose(hist["beta"][:10], ref["beta"][:10], rtol=1e-10)
        assert np.array_equal(res["rel_resid"], outs[0][0]["rel_resid"])      # bit-identical sums on every rank
    for i, s in enumerate(shifts):
        tr = np.linalg.norm(b - oracle.mdagm(dims, U, m, got_x[i], sigma=s)) / bn
        assert tr < 1.5 * tol, (i, tr)
        assert abs(tr - outs[0][0]["rel_resid"][i]) < 1e-12
        assert rel(got_x[i], ref["x"][i]) < 10 * (7.0 / (m * m + s)) * tol
    y_ref = c0 * b + sum(ci * xi for ci, xi in zip(c, ref["x"]))
    bound = sum(abs(ci) * 10 * (7.0 / (m * m + s)) * tol * np.linalg.norm(xi)
                for ci, s, xi in zip(c, shifts, ref["x"])) / np.linalg.norm(y_ref)
    assert rel(got_y, y_ref) < bound


def test_peer_fp32_cg_max_iter_and_zero_rhs():
    """fp32 over the peer transport (P = 2, lock step), the max_iter exit and a zero right-hand side."""
    from paper_1701_00426_b200.slab import SlabLattice
    dims = (4, 4, 4, 8)
    rng = np.random.default_rng(73)
    U = gen.smooth_links(dims, 0.3, rng).astype(np.complex64).astype(np.complex128)
    b = gen.gaussian_half_spinor(dims, rng).astype(np.complex64).astype(np.complex128)
    ref = oracle.cg(dims, U, 0.2, b, 1e-5, 2000)
    got = np.zeros_like(b)
    lock = threading.Lock()

    def work(r, sl):
        links = sl.pack_links(U)
        be = sl.pack_spinor(b, 0)
        x = sl.new_spinor()
        res = sl.cg_multishift([x], be, links, 0.2, [0.0], 1e-5, 2000)
        short = sl.cg_multishift([sl.new_spinor()], be, links, 0.2, [0.0], 1e-5, 3, raise_on_max_iter=False)
        zero = sl.cg_multishift([sl.new_spinor()], sl.new_spinor(), links, 0.2, [0.0], 1e-5, 50)
        with lock:
            sl.unpack_spinor(x, 0, got)
        return res, short, zero

    outs = run_peer_ranks(2, lambda r: SlabLattice(dims, 2, r, prec=1, transport="peer"), work)
    for res, short, zero in outs:
        assert abs(res["iters"] - ref["iters"]) <= max(2, ref["iters"] // 50)
        assert not short["converged"] and short["iters"] == 3
        assert zero["iters"] == 0 and zero["converged"]
    assert np.linalg.norm(b - oracle.mdagm(dims, U, 0.2, got)) / np.linalg.norm(b) < 2e-5


@pytest.mark.parametrize("fmt", [0, 1])
@pytest.mark.parametrize("world", [1, 2])
def test_peer_backfield_dslash_and_solve(world, fmt):
    """The backfield over the peer transport: the hops that leave the slab take their phase from the slab's own
    (ghost-inclusive) phase field and their vector from the landing buffers."""
    from paper_1701_00426_b200.slab import SlabLattice
    dims = (8, 6, 4, 8)
    rng = np.random.default_rng(76)
    U = gen.smooth_links(dims, 0.3, rng)
    psi = gen.gaussian_spinor(dims, rng)
    theta = gen.uniform_backfield(dims, rng)
    shifts = gen.rhmc_shifts(3)
    b = oracle.full_to_half(dims, 0, psi)
    ref = oracle.cg_multishift(dims, U, 0.1, shifts, b, 1e-10, 4000, theta=theta)
    got = {0: np.zeros_like(b), 1: np.zeros_like(b)}
    got_x = [np.zeros_like(b) for _ in shifts]
    lock = threading.Lock()

    def work(r, sl):
        links = sl.pack_links(U)
        sl.lat.set_backfield(sl.pack_backfield(theta))
        outs = {}
        for gp in (1, 0):
            inp = sl.pack_spinor(oracle.full_to_half(dims, 1 - gp, psi), 1 - gp)
            outs[gp] = sl.new_spinor()
            sl.dslash(gp, outs[gp], inp, links)
        be = sl.pack_spinor(b, 0)
        xs = [sl.new_spinor() for _ in shifts]
        res = sl.cg_multishift(xs, be, links, 0.1, shifts, 1e-10, 4000)
        with lock:
            for gp in (0, 1):
                sl.unpack_spinor(outs[gp], gp, got[gp])
            for i, x in enumerate(xs):
                sl.unpack_spinor(x, 0, got_x[i])
        return res

    outs = run_peer_ranks(world, lambda r: SlabLattice(dims, world, r, transport="peer", options=dict(backfield_format=fmt)), work)
    for gp in (0, 1):
        want = oracle.dslash_half(dims, U, gp, oracle.full_to_half(dims, 1 - gp, psi), theta=theta)
        assert rel(got[gp], want) < 1e-12, (world, fmt, gp)
    for res in outs:
        assert abs(res["iters"] - ref["iters"]) <= 2
    for i, s in enumerate(shifts):
        tr = np.linalg.norm(b - oracle.mdagm(dims, U, 0.1, got_x[i], sigma=s, theta=theta)) / np.linalg.norm(b)
        assert tr < 1.5e-10, (i, tr)


@pytest.mark.parametrize("fmt", [0, 1])
@pytest.mark.parametrize("world", [1, 2, 4])
def test_peer_dslash_backfield_explicit_call(world, fmt):
    """lqcd_dslash_backfield (the paper's four-argument acc_Deo, phases given per call, nothing attached to the
    context) over the peer transport: the call must push the faces of ITS input before the kernel reads the landing
    buffers.  Two calls in a row with different inputs: a missing push would leave the first call's faces (or none)
    in the buffers and the boundary slices of the second result would be wrong."""
    from paper_1701_00426_b200.slab import SlabLattice
    dims = (8, 6, 4, 8)
    rng = np.random.default_rng(77)
    U = gen.smooth_links(dims, 0.3, rng)
    theta = gen.uniform_backfield(dims, rng)
    psis = [gen.gaussian_spinor(dims, rng), gen.gaussian_spinor(dims, rng)]
    got = {(k, gp): None for k in range(2) for gp in (0, 1)}
    for key in got:
        got[key] = np.zeros((dims[0] * dims[1] * dims[2] * dims[3] // 2, 3), dtype=np.complex128)
    lock = threading.Lock()

    def work(r, sl):
        links = sl.pack_links(U)
        bf = sl.pack_backfield(theta)
        outs = {}
        for k, psi in enumerate(psis):
            for gp in (1, 0):
                inp = sl.pack_spinor(oracle.full_to_half(dims, 1 - gp, psi), 1 - gp)
                outs[(k, gp)] = sl.new_spinor()
                sl.lat.dslash_backfield(sl.geo.local_parity(gp), outs[(k, gp)], inp, links, bf)
                sl._raise_hook_error()
        with lock:
            for key, buf in outs.items():
                sl.unpack_spinor(buf, key[1], got[key])

    run_peer_ranks(world, lambda r: SlabLattice(dims, world, r, transport="peer", options=dict(backfield_format=fmt)), work)
    for (k, gp), g in got.items():
        want = oracle.dslash_half(dims, U, gp, oracle.full_to_half(dims, 1 - gp, psis[k]), theta=theta)
        assert rel(g, want) < 1e-12, (world, fmt, k, gp, rel(g, want))


@pytest.mark.parametrize("nranks", [1, 2, 3, 8, 16])
def test_peer_protocol_selftest_under_real_concurrency(nranks):
    """lqcd_peer_selftest: the flags / slots / counters of the transport with ranks that run AT THE SAME TIME (one
    cooperative kernel, CTA r = rank r, uneven pace) and really wait for one another: 2000 rounds of (halo exchange,
    two all-reduces), every token and every rank-ordered sum checked on the device."""
    import paper_1701_00426_b200 as L
    lat = L.Lattice((4, 4, 4, 4))
    assert lat.peer_selftest(nranks, 2000) == 0
    if nranks > 2:        # the test can fail: consumers that do not wait read stale tokens / incomplete sums
        assert lat.peer_selftest(nranks, 2000, sabotage=True) > 0
    lat.close()


@pytest.mark.parametrize("ap", [True, False])
@pytest.mark.parametrize("world", [1, 2, 4])
def test_peer_fermion_force_equals_global_oracle(world, ap):
    """lqcd_fermion_force on slabs over the peer transport: every owned link against the oracle on the global lattice
    (the antiperiodic sign crosses the slab boundary inside the ghost data; the (-1)^p(x) of R21 is the GLOBAL parity)."""
    from paper_1701_00426_b200.slab import SlabLattice
    dims = (4, 6, 4, 8)
    rng = np.random.default_rng(77)
    U = gen.haar_like_links(dims, rng)
    n = 3
    xs = np.stack([gen.gaussian_half_spinor(dims, rng) for _ in range(n)])
    c = np.array([0.7, -1.1, 0.4])
    want = oracle.fermion_force(dims, U, c, xs, antiperiodic_t=ap)
    got = np.zeros_like(want)
    lock = threading.Lock()

    def work(r, sl):
        links = sl.pack_links(U)
        f = sl.fermion_force([sl.pack_spinor(x, 0) for x in xs], links, c)
        with lock:
            sl.unpack_tamat_owned(f, got)

    run_peer_ranks(world, lambda r: SlabLattice(dims, world, r, antiperiodic_t=ap, transport="peer"), work)
    assert rel(got, want) < 1e-12, (world, ap, rel(got, want))


def test_peer_wait_gives_up_instead_of_hanging():
    """A rank whose neighbour never shows up (here: rank 0 of 2 runs alone, with a 50 ms limit) must not hang the GPU:
    the boundary tiles of its Dslash give up, the count is readable, and a solve returns LQCD_ERR_CUDA."""
    import paper_1701_00426_b200 as L
    from paper_1701_00426_b200.slab import SlabLattice
    dims = (4, 4, 4, 8)
    rng = np.random.default_rng(75)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    slabs = [SlabLattice(dims, 2, r, transport="peer", options=dict(peer_wait_ms=50)) for r in range(2)]
    SlabLattice.connect_local(slabs)
    sl = slabs[0]
    links, be, out = sl.pack_links(U), sl.pack_spinor(b, 0), sl.new_spinor()
    assert sl.lat.get_option("peer_timeouts") == 0
    sl.dslash(1, out, be, links)                      # rank 1 never pushes its faces
    assert sl.lat.get_option("peer_timeouts") > 0
    with pytest.raises(L.LqcdError) as e:
        sl.cg_multishift([sl.new_spinor()], be, links, 0.2, [0.0], 1e-8, 8, raise_on_max_iter=False)
    assert e.value.code == L.ERR_CUDA and "timed out" in str(e.value)
    for s in slabs:
        s.close()


def test_peer_timeout_ends_a_long_solve_at_once():
    """A dead peer must cost ONE wait limit, not one per wait: with max_iter = 20000 and the chunk graph on (no lock-step
    hook), rank 0 of 2 runs alone.  Before the first timeout made the transport dead, every one of the 4 waits of every
    iteration spent the full limit again (here 4 x 0.1 s x 20000 iterations = over two hours of GPU time); now the first
    wait gives up after 0.1 s, every later wait returns at once, the host sees the count at its next poll and the call
    returns LQCD_ERR_CUDA within seconds -- and so does the next call over the same (dead) transport."""
    import time
    import paper_1701_00426_b200 as L
    from paper_1701_00426_b200.slab import SlabLattice
    dims = (4, 4, 4, 8)
    rng = np.random.default_rng(78)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    slabs = [SlabLattice(dims, 2, r, transport="peer", options=dict(peer_wait_ms=100)) for r in range(2)]
    SlabLattice.connect_local(slabs)
    sl = slabs[0]
    links, be = sl.pack_links(U), sl.pack_spinor(b, 0)
    xs = [sl.new_spinor(), sl.new_spinor()]
    sl.lat.synchronize()
    for attempt in range(2):
        t0 = time.time()
        with pytest.raises(L.LqcdError) as e:
            sl.cg_multishift(xs, be, links, 0.01, [0.0, 0.1], 1e-12, 20000, raise_on_max_iter=False)
        dt = time.time() - t0
        assert e.value.code == L.ERR_CUDA and "timed out" in str(e.value)
        assert dt < 20.0, (attempt, dt)
    assert sl.lat.get_option("peer_timeouts") > 0
    for s in slabs:
        s.close()


def test_peer_errors_and_disconnect():
    import paper_1701_00426_b200 as L
    from paper_1701_00426_b200.slab import SlabLattice
    dims = (4, 4, 4, 8)
    rng = np.random.default_rng(74)
    U = gen.smooth_links(dims, 0.3, rng)
    sl = SlabLattice(dims, 1, 0, transport="peer")
    lat = sl.lat
    links = sl.pack_links(U)
    with pytest.raises(L.LqcdError) as e:
        lat.gauge_staples(links)
    assert e.value.code == L.ERR_UNSUPPORTED                 # ghost depth 2 would be needed
    with pytest.raises(L.LqcdError):
        lat.peer_init(17, 0, 1, 9, 1, 1.0, 1.0)            # more than 16 ranks
    with pytest.raises(L.LqcdError):
        lat.peer_init(2, 0, 0, 9, 1, 1.0, 1.0)             # no ghost slice below
    assert len(lat.peer_export()) == 64                     # the IPC handle of the block can be taken
    lat.peer_disconnect()
    # an ordinary (periodic) lattice of the local extents again
    phi = gen.gaussian_half_spinor(sl.geo.local_dims, rng)
    Uloc = np.ascontiguousarray(sl.geo.extract_full(U))
    out = lat.new_spinor()
    lat.dslash(1, out, lat.pack_spinor(phi, 0), links)
    want = oracle.dslash_half(sl.geo.local_dims, Uloc, 1, phi, antiperiodic_t=False)
    assert rel(lat.unpack_spinor(out, 1), want) < 1e-12
    sl.close()
