"""lqcd_mdagm_noalloc against lqcd_mdagm (-m gpu).  Collected last on purpose (the file name sorts after every
other test file): `pytest -x` stops at the first failure, and a failure here must not hide the parity tests.

Why the entry point exists: some users of this library cannot hand it a workspace because they cannot allocate
device memory at the point where they call it -- the library is embedded in a program whose own allocator has
already claimed the GPU's memory, or the caller runs in a service that forbids cudaMalloc / cudaFree after
start-up because both stall the whole device, or the job is planned to the last GB of HBM.  For them the normal
operator's odd-site temporary lives in a fixed 8 MiB array inside the library's device image (include/lqcd.h,
csrc/noalloc.cu) instead of a caller-owned workspace.

What is checked: on two calls in a row (different input, mass and shift, so that anything left in the shared
array by the first call would show in the second) the output equals that of the existing lqcd_mdagm path, which
keeps its temporary in a torch-allocated workspace, within the tolerance of the parity tests (1e-12 relative L2
in fp64, 1e-5 in fp32; the two paths launch the same kernels, so the difference is in fact zero); the oracle
confirms the first fp64 result independently; no workspace is set on the context that uses the new call and
torch's allocator hands out nothing during it; a lattice beyond the limit is refused with a message and nothing
is written.  Nothing here depends on what earlier tests left behind: the test passes alone in a fresh process
(where its first call performs the per-device address look-up) and after the rest of the suite.
"""
import numpy as np
import pytest

import lqcd_inputs as gen
import oracle

pytestmark = pytest.mark.gpu

TOL = {0: 1e-12, 1: 1e-5}


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


@pytest.mark.parametrize("prec,recon,dims", [(0, 0, (8, 6, 4, 12)), (0, 1, (16, 16, 16, 16)), (1, 0, (12, 10, 6, 4))])
def test_mdagm_noalloc_matches_workspace_path_twice(prec, recon, dims):
    import torch
    import paper_1701_00426_b200 as L

    rng = np.random.default_rng(2026)
    U = gen.smooth_links(dims, 0.4, rng)
    inputs = [gen.gaussian_half_spinor(dims, rng), gen.gaussian_half_spinor(dims, rng)]
    params = [(0.05, 0.0), (0.3, 0.37)]          # (mass, sigma) of the first and of the second call

    ref = L.Lattice(dims, prec=prec, recon=recon)          # existing path: temporary in a caller-owned workspace
    new = L.Lattice(dims, prec=prec, recon=recon)          # new path: never given a workspace
    assert ref.spinor_bytes <= L.binding.NOALLOC_SCRATCH_BYTES
    links = ref.pack_links(U)
    for call, (b, (mass, sigma)) in enumerate(zip(inputs, params)):
        be = ref.pack_spinor(b, L.EVEN)
        want_buf, got_buf = ref.new_spinor(), new.new_spinor()
        got_buf.fill_(0xFF)                                # a skipped launch would leave NaN patterns behind
        ref.mdagm(want_buf, be, links, mass, sigma)
        ref.synchronize()
        before = torch.cuda.memory_stats()["allocation.all.allocated"]
        new.mdagm_noalloc(got_buf, be, links, mass, sigma)
        new.synchronize()
        assert torch.cuda.memory_stats()["allocation.all.allocated"] == before     # the binding allocates nothing either
        assert new._ws is None                             # and no workspace was ever attached to this context
        want = ref.unpack_spinor(want_buf, L.EVEN)
        got = new.unpack_spinor(got_buf, L.EVEN)
        assert np.all(np.isfinite(got))
        assert rel(got, want) < TOL[prec], (call, rel(got, want))
        if prec == 0 and call == 0 and recon == 0:         # and the existing path is the oracle's operator
            assert rel(got, oracle.mdagm(dims, U, mass, b, sigma=sigma)) < TOL[0]
    ref.close()
    new.close()


def test_mdagm_noalloc_refuses_what_does_not_fit():
    import paper_1701_00426_b200 as L

    lat = L.Lattice((32, 32, 32, 32), prec=L.F64)          # one half vector = 25 MB > 8 MiB
    assert lat.spinor_bytes > L.binding.NOALLOC_SCRATCH_BYTES
    out, inp = lat.new_spinor(), lat.new_spinor()
    links = lat._buf(16)                                   # never dereferenced: the size check comes before any launch
    out.zero_()
    n0 = lat.launches
    with pytest.raises(L.LqcdError) as e:
        lat.mdagm_noalloc(out, inp, links, 0.1)
    assert e.value.code == L.ERR_WORKSPACE
    assert str(lat.spinor_bytes) in str(e.value) and str(L.binding.NOALLOC_SCRATCH_BYTES) in str(e.value)
    assert lat.launches == n0 and int(out.count_nonzero()) == 0
    lat.close()
    # fp32 halves the vector: 32^3 x 16 fits
    lat = L.Lattice((32, 32, 32, 16), prec=L.F32)
    assert lat.spinor_bytes <= L.binding.NOALLOC_SCRATCH_BYTES
    lat.close()
