"""-m gpu: the x3-slab path (NEXT-2) on ONE GPU.  Each of P "virtual ranks" is a SlabLattice with its own
context, fields and halo buffers on cuda:0, driven by its own host thread; the ranks meet in a
ThreadComm that exchanges faces by device copies and sums scalars on the host.  Kernels never wait on
one another (everything is on one stream; the HOST threads synchronise), so this is the real slab code
-- lqcd_dslash_slices, the halo kernels, the hooks of lqcd_set_slab, the owned-slice vector kernels and
the scalar kernels -- with only the transport replaced.  Results must equal the oracle on the GLOBAL
lattice, and the solver must take the same iterations as the single-context path."""
import threading

import numpy as np
import pytest

import lqcd_inputs as gen
import oracle

pytestmark = pytest.mark.gpu


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


class ThreadComm:
    """Transport between virtual ranks in one process (test infrastructure)."""

    class Shared:
        def __init__(self, world):
            self.world = world
            self.barrier = threading.Barrier(world)
            self.bufs = [None] * world
            self.vals = [None] * world

    def __init__(self, shared, rank):
        self.s, self.rank, self.world = shared, rank, shared.world
        self.up, self.down = (rank + 1) % self.world, (rank - 1) % self.world

    def exchange_start(self, send_up, send_down, recv_from_down, recv_from_up):
        s = self.s
        s.bufs[self.rank] = (send_up, send_down)
        s.barrier.wait()                       # every rank's pack kernels are enqueued (one stream)
        recv_from_down.copy_(s.bufs[self.down][0])
        recv_from_up.copy_(s.bufs[self.up][1])
        s.barrier.wait()                       # nobody repacks before every copy is enqueued
        return []

    def exchange_wait(self, handle):
        pass

    def allreduce_sum(self, t):
        s = self.s
        s.vals[self.rank] = t.cpu()
        s.barrier.wait()
        tot = sum(s.vals[r] for r in range(self.world))     # same order on every rank
        s.barrier.wait()
        t.copy_(tot)
        return t


def run_ranks(world, fn):
    """fn(rank, comm) on `world` threads; re-raises the first failure."""
    shared = ThreadComm.Shared(world)
    errs, outs = [], [None] * world

    def work(r):
        try:
            outs[r] = fn(r, ThreadComm(shared, r))
        except BaseException as e:  # noqa: BLE001
            errs.append(e)
            shared.barrier.abort()

    ts = [threading.Thread(target=work, args=(r,)) for r in range(world)]
    for t in ts:
        t.start()
    for t in ts:
        t.join(300)
    if errs:
        raise errs[0]
    return outs


@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("world", [1, 2, 4])
def test_slab_dslash_equals_global_oracle(world, prec):
    from paper_1701_00426_b200.slab import SlabLattice
    dims = (8, 6, 4, 16)
    rng = np.random.default_rng(31)
    U = gen.smooth_links(dims, 0.3, rng)
    psi = gen.gaussian_spinor(dims, rng)
    if prec == 1:
        U, psi = (a.astype(np.complex64).astype(np.complex128) for a in (U, psi))
    tol = 1e-12 if prec == 0 else 1e-5
    for gp_out in (0, 1):
        phi_in = oracle.full_to_half(dims, 1 - gp_out, psi)
        want = oracle.dslash_half(dims, U, gp_out, phi_in)
        for overlap in (True, False):
            got = np.zeros_like(want)
            lock = threading.Lock()

            def rank_fn(r, comm):
                sl = SlabLattice(dims, world, r, comm=comm, prec=prec)
                links = sl.pack_links(U)
                inp = sl.pack_spinor(phi_in, 1 - gp_out)
                out = sl.new_spinor()
                sl.dslash(gp_out, out, inp, links, overlap=overlap)
                with lock:
                    sl.unpack_spinor(out, gp_out, got)
                sl.close()

            run_ranks(world, rank_fn)
            assert rel(got, want) < tol, (world, prec, gp_out, overlap, rel(got, want))


@pytest.mark.parametrize("world", [1, 2])
def test_slab_mdagm_and_multishift_cg(world):
    import paper_1701_00426_b200 as L
    from paper_1701_00426_b200.slab import SlabLattice
    dims = (8, 8, 4, 8)
    rng = np.random.default_rng(32)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    m, tol = 0.05, 1e-10
    shifts = gen.rhmc_shifts(4)[[2, 0, 3, 1]]
    ref = oracle.cg_multishift(dims, U, m, shifts, b, tol, 5000, hist_len=16)
    want_A = oracle.mdagm(dims, U, m, b, sigma=0.37)
    # single-context run of the same problem
    lat = L.Lattice(dims)
    links1, b1 = lat.pack_links(U), lat.pack_spinor(b, 0)
    xs1 = [lat.new_spinor() for _ in shifts]
    res1 = lat.cg_multishift(xs1, b1, links1, m, shifts, tol, 5000)
    lat.close()

    got_A = np.zeros_like(b)
    got_x = [np.zeros_like(b) for _ in shifts]
    got_y = np.zeros_like(b)
    lock = threading.Lock()
    c0, c = 0.35, np.array([0.5, -1.25, 2.0, 0.125])

    def rank_fn(r, comm):
        sl = SlabLattice(dims, world, r, comm=comm)
        links = sl.pack_links(U)
        be = sl.pack_spinor(b, 0)
        out = sl.new_spinor()
        sl.mdagm(out, be, links, m, 0.37)
        xs = [sl.new_spinor() for _ in shifts]
        res = sl.cg_multishift(xs, be, links, m, shifts, tol, 5000)
        hist = sl.lat.solver_history()
        y = sl.new_spinor()
        resy = sl.rational_apply(y, be, links, m, shifts, c0, c, tol, 5000)
        with lock:
            sl.unpack_spinor(out, 0, got_A)
            for i, x in enumerate(xs):
                sl.unpack_spinor(x, 0, got_x[i])
            sl.unpack_spinor(y, 0, got_y)
        assert sl.lat.get_option("graph_active") == 0
        sl.close()
        return res, hist, resy

    outs = run_ranks(world, rank_fn)
    assert rel(got_A, want_A) < 1e-12
    bn = np.linalg.norm(b)
    for res, hist, resy in outs:                       # every rank took the same decisions
        assert res["iters"] == outs[0][0]["iters"] and np.array_equal(res["conv_iter"], outs[0][0]["conv_iter"])
        assert abs(res["iters"] - ref["iters"]) <= 2 and abs(res["iters"] - res1["iters"]) <= 1
        assert resy["iters"] == res["iters"]
        assert np.allclose(hist["alpha"][:10], ref["alpha"][:10], rtol=1e-10)
        assert np.allclose(hist["beta"][:10], ref["beta"][:10], rtol=1e-10)
        assert np.allclose(res["rel_resid"], outs[0][0]["rel_resid"])
    for i, s in enumerate(shifts):
        tr = np.linalg.norm(b - oracle.mdagm(dims, U, m, got_x[i], sigma=s)) / bn
        assert tr < 1.5 * tol, (i, tr)
        assert abs(tr - outs[0][0]["rel_resid"][i]) < 1e-12
        assert rel(got_x[i], ref["x"][i]) < 10 * (7.0 / (m * m + s)) * tol
    y_ref = c0 * b + sum(ci * xi for ci, xi in zip(c, ref["x"]))
    bound = sum(abs(ci) * 10 * (7.0 / (m * m + s)) * tol * np.linalg.norm(xi)
                for ci, s, xi in zip(c, shifts, ref["x"])) / np.linalg.norm(y_ref)
    assert rel(got_y, y_ref) < bound


@pytest.mark.parametrize("world", [1, 2])
def test_slab_dslash_and_solve_with_backfield(world):
    """The backfield in slab mode (hook transport): every rank packs the phases of its slab incl. the ghost slices,
    like the links.  Dslash = global oracle with phases; a multi-shift solve by R16 with the oracle's phased operator."""
    from paper_1701_00426_b200.slab import SlabLattice
    dims = (8, 6, 4, 8)
    rng = np.random.default_rng(33)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    theta = gen.uniform_backfield(dims, rng)
    shifts = gen.rhmc_shifts(3)
    want = oracle.dslash_half(dims, U, 1, b, theta=theta)
    ref = oracle.cg_multishift(dims, U, 0.1, shifts, b, 1e-10, 4000, theta=theta)
    got = np.zeros_like(want)
    got_x = [np.zeros_like(b) for _ in shifts]
    lock = threading.Lock()

    def rank_fn(r, comm):
        sl = SlabLattice(dims, world, r, comm=comm)
        links = sl.pack_links(U)
        sl.lat.set_backfield(sl.pack_backfield(theta))
        be = sl.pack_spinor(b, 0)
        out = sl.new_spinor()
        sl.dslash(1, out, be, links)
        xs = [sl.new_spinor() for _ in shifts]
        res = sl.cg_multishift(xs, be, links, 0.1, shifts, 1e-10, 4000)
        with lock:
            sl.unpack_spinor(out, 1, got)
            for i, x in enumerate(xs):
                sl.unpack_spinor(x, 0, got_x[i])
        sl.close()
        return res

    outs = run_ranks(world, rank_fn)
    assert rel(got, want) < 1e-12
    assert rel(oracle.dslash_half(dims, U, 1, b), want) > 0.1
    for res in outs:
        assert abs(res["iters"] - ref["iters"]) <= 2
    for i, s in enumerate(shifts):
        tr = np.linalg.norm(b - oracle.mdagm(dims, U, 0.1, got_x[i], sigma=s, theta=theta)) / np.linalg.norm(b)
        assert tr < 1.5e-10, (i, tr)


@pytest.mark.parametrize("world", [1, 2])
def test_slab_fermion_force_hook_transport(world):
    """lqcd_fermion_force on slabs with the hook transport, fp32 included."""
    from paper_1701_00426_b200.slab import SlabLattice
    dims = (4, 6, 4, 8)
    rng = np.random.default_rng(34)
    U = gen.haar_like_links(dims, rng)
    xs = np.stack([gen.gaussian_half_spinor(dims, rng) for _ in range(2)])
    c = np.array([0.9, -0.3])
    for prec in (0, 1):
        Uu, xx = (U, xs) if prec == 0 else (U.astype(np.complex64).astype(np.complex128), xs.astype(np.complex64).astype(np.complex128))
        want = oracle.fermion_force(dims, Uu, c, xx)
        got = np.zeros_like(want)
        lock = threading.Lock()

        def rank_fn(r, comm):
            sl = SlabLattice(dims, world, r, comm=comm, prec=prec)
            f = sl.fermion_force([sl.pack_spinor(x, 0) for x in xx], sl.pack_links(Uu), c)
            with lock:
                sl.unpack_tamat_owned(f, got)
            sl.close()

        run_ranks(world, rank_fn)
        assert rel(got, want) < (1e-12 if prec == 0 else 1e-5), (world, prec, rel(got, want))


@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("layout", [0, 1])
def test_single_face_halo_calls(prec, layout):
    """lqcd_halo_pack / lqcd_halo_unpack (one face per call): slice 2 of a vector, sign -1, lands in
    slice 0 of another; everything else of the target is untouched."""
    import paper_1701_00426_b200 as L
    dims = (4, 6, 2, 6)
    phi = gen.gaussian_half_spinor(dims, 41)
    if prec == 1:
        phi = phi.astype(np.complex64).astype(np.complex128)
    lat = L.Lattice(dims, prec=prec, options=dict(layout=layout))
    src = lat.pack_spinor(phi, 0)
    dst = lat.pack_spinor(2.0 * phi, 0)
    buf = lat._buf(lat.halo_bytes)
    lat.halo_pack(buf, src, 2, -1.0)
    lat.halo_unpack(dst, buf, 0)
    got = lat.unpack_spinor(dst, 0)
    s3 = dims[0] * dims[1] * dims[2] // 2
    want = 2.0 * phi
    want[:s3] = -phi[2 * s3:3 * s3]
    assert np.array_equal(got, want)
    with pytest.raises(L.LqcdError):
        lat.halo_pack(buf, src, 6, 1.0)
    lat.close()
