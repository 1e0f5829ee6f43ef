"""-m "not gpu": the C-ABI library loads and exports every symbol include/lqcd.h declares; argument
checks that happen before any CUDA call; the product never routes through the oracle; the
multi-process (replica) plumbing of bench.py under gloo with world_size 2."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    """every function include/*.h declares: the ABI (lqcd.h) and the diagnostics beside it (lqcd_diag.h)"""
    names = set()
    for h in sorted(os.listdir(os.path.join(ROOT, "include"))):
        if not h.endswith(".h"):
            continue
        src = open(os.path.join(ROOT, "include", h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(lqcd_[a-z_0-9]+)\s*\(", src))
    return sorted(names)


def test_library_exports_every_declared_symbol():
    import paper_1701_00426_b200 as L
    names = declared_symbols()
    assert len(names) >= 18 and "lqcd_dslash" in names and "lqcd_cg_multishift" in names
    for n in names:
        assert hasattr(L.lib, n), n
    # and the binding gives every one of them a signature
    from paper_1701_00426_b200 import binding
    assert sorted(binding._sig) == names
    assert b"sm_100a" in L.lib.lqcd_version()


def test_library_contains_sm100a_code_only():
    import paper_1701_00426_b200 as L
    out = subprocess.run(["cuobjdump", "-lelf", L.lib_path], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    archs = set(re.findall(r"sm_\d+a?", out.stdout))
    assert archs == {"sm_100a"}, archs


def test_argument_errors_before_any_cuda_call():
    import paper_1701_00426_b200 as L
    ctx = C.c_void_p()
    bad = [((4, 4, 4, 3), 0, 0, 1), ((4, 4, 0, 4), 0, 0, 1), ((4, 4, 4, 4), 7, 0, 1),
           ((4, 4, 4, 4), 0, 5, 1), ((4, 4, 4, 4), 0, 0, 2), ((2048, 2048, 2048, 2), 0, 0, 1)]
    for dims, prec, recon, ap in bad:
        rc = L.lib.lqcd_create(C.byref(ctx), (C.c_int * 4)(*dims), prec, recon, ap, 0, None)
        assert rc == L.ERR_ARG, (dims, prec, recon, ap, rc)
        assert ctx.value is None
        assert L.lib.lqcd_last_error(None) != b""
    assert L.lib.lqcd_create(None, (C.c_int * 4)(4, 4, 4, 4), 0, 0, 1, 0, None) == L.ERR_ARG
    # null contexts are rejected, sizes of a null context are 0
    assert L.lib.lqcd_destroy(None) == L.ERR_ARG
    assert L.lib.lqcd_spinor_bytes(None) == 0 and L.lib.lqcd_links_bytes(None) == 0
    assert L.lib.lqcd_dslash(None, 0, None, None, None) == L.ERR_ARG
    assert L.lib.lqcd_cg(None, None, None, None, 0.1, 1e-8, 10, None, None) == L.ERR_ARG


def test_no_gpu_means_loud_failure_not_fallback():
    import torch
    import paper_1701_00426_b200 as L
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    ctx = C.c_void_p()
    rc = L.lib.lqcd_create(C.byref(ctx), (C.c_int * 4)(4, 4, 4, 4), 0, 0, 1, 0, None)
    assert rc == L.ERR_CUDA and b"no CPU fallback" in L.lib.lqcd_last_error(None)
    with pytest.raises(L.LqcdError):
        L.Lattice((4, 4, 4, 4))


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1701_00426_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "staggered_oracle" not in txt and "liboracle" not in txt, f
    for f in ("oracle/staggered_oracle.c", "oracle/oracle.py"):
        txt = open(os.path.join(ROOT, f)).read()
        assert "paper_1701_00426_b200" not in txt.replace("under paper_1701_00426_b200/", "") or f.endswith(".c")
        assert "lqcd.h" not in txt and "liblqcd" not in txt


def test_fastdiv_formula():
    """The multiply-high division used for the site decode (common.cuh make_fastdiv), re-derived:
    q = (n * ceil(2^(31+l)/d)) >> (31+l) for n < 2^31, l = ceil(log2 d)."""
    rng = np.random.default_rng(0)
    for d in [1, 2, 3, 4, 5, 6, 7, 8, 12, 16, 18, 24, 31, 32, 36, 48, 64, 96, 1000, 65535]:
        if d == 1:
            continue
        l = int(np.ceil(np.log2(d)))
        m = ((1 << (32 + l - 1)) + d - 1) // d
        assert m < (1 << 32)
        ns = np.concatenate([rng.integers(0, 2 ** 31 - 1, 2000), [0, 1, d - 1, d, d + 1, 2 ** 31 - 1]])
        for n in ns:
            n = int(n)
            assert ((n * m) >> 32) >> (l - 1) == n // d


def test_staple_cta_swizzle_is_a_permutation():
    """The CTA order of the staples kernel (staples.cu staple_cta), re-derived: t enumerates (b, x3, j, tx)
    and lands on tile tx + tiles_row*((b*x2b + j) + N2*x3): every tile exactly once."""
    for N2, N3, tiles_row, x2b in [(32, 32, 4, 8), (8, 32, 4, 2), (4, 4, 1, 4), (12, 6, 3, 4), (32, 8, 4, 16)]:
        n = tiles_row * N2 * N3
        seen = np.zeros(n, dtype=int)
        for t0 in range(n):
            t = t0
            tx = t % tiles_row; t //= tiles_row
            j = t % x2b; t //= x2b
            x3 = t % N3
            b = t // N3
            seen[tx + tiles_row * ((b * x2b + j) + N2 * x3)] += 1
        assert (seen == 1).all(), (N2, N3, tiles_row, x2b)


def test_slab_segment_map_covers_exactly_the_owned_packets():
    """solver.cu seg_idx, re-derived: flat packet k of the owned slices -> plane*stride + off + (k mod len).
    Layout 0: 3 complex planes of Vh sites (2 reals per site), packets of N reals."""
    N0, N1, N2, N3 = 8, 4, 2, 6
    s3, Vh = (N0 // 2) * N1 * N2, (N0 // 2) * N1 * N2 * N3
    for N in (2, 4):                      # double2 / float4 packets
        for x3_lo, x3_hi in ((1, 5), (0, 6), (2, 3)):
            ln = (x3_hi - x3_lo) * s3 * 2 // N
            stride, off = Vh * 2 // N, x3_lo * s3 * 2 // N
            got = sorted((k // ln) * stride + off + k % ln for k in range(3 * ln))
            want = sorted(p * stride + (x3 * s3 * 2 // N) + q for p in range(3) for x3 in range(x3_lo, x3_hi)
                          for q in range(s3 * 2 // N))
            assert got == want


def test_shift_recipe_and_generators_are_deterministic():
    import lqcd_inputs as gen
    s = gen.rhmc_shifts(8)
    assert np.allclose(s, [1e-4, 3.72759372e-4, 1.38949549e-3, 5.17947468e-3, 1.93069773e-2, 7.19685673e-2, 2.68269580e-1, 1.0])
    a = gen.smooth_links((4, 4, 2, 2), 0.3, 2)
    b = gen.smooth_links((4, 4, 2, 2), 0.3, 2)
    assert np.array_equal(a, b)
    eye = np.einsum("nmab,nmcb->nmac", a, a.conj())
    assert np.abs(eye - np.eye(3)).max() < 1e-14 and np.abs(np.linalg.det(a) - 1).max() < 1e-14
    # eps = 0.3 links are "smoothed toward identity": Re tr U / 3 well above a Haar sample's ~0
    assert np.mean(np.trace(a, axis1=-2, axis2=-1).real) / 3 > 0.8
    with pytest.raises(ValueError):
        gen.gaussian_spinor((4, 4, 3, 4), 1)


_WORKER = r"""
import os, sys
sys.path.insert(0, %r)
from paper_1701_00426_b200 import dist as D
rank, local_rank, world = D.init("gloo")
assert world == 2 and rank in (0, 1)
D.barrier(world)
# device time differs per rank: the job time is the MAX
t = D.max_over_ranks(10.0 + 5.0 * rank, world)
assert t == 15.0, t
seeds = (D.replica_seed(3, 0), D.replica_seed(3, 1))
assert seeds[0] != seeds[1] and D.replica_seed(3, rank) == seeds[rank]
ns = D.aggregate_ns_per_site(t, 5, 1000, world)     # 15 ms / (5 steps * 1000 sites * 2 ranks)
assert abs(ns - 1500.0) < 1e-9, ns
D.barrier(world)
D.finalize(world)
print("rank", rank, "ok")
"""


def test_replica_plumbing_gloo_world2(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(_WORKER % ROOT)
    port = 29600 + os.getpid() % 300
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, o
        assert f"rank {r} ok" in o


def test_peer_face_map_matches_the_landing_buffer_layout():
    """Host re-derivation of peer_store_faces (csrc/solver.cu): packet k0 of the owned range [x3_lo, x3_hi) of plane pl,
    if it lies in the first / last owned slice, lands at packet pl * slice + (offset inside the slice) of the landing
    buffer -- which is laid out like a half vector of ONE slice.  Checked against the site indices: every face site
    of every plane is hit exactly once, and the landing index equals the face index f = idxh - x3 * s3 that the
    Dslash reads (csrc/dslash.cu, HALO)."""
    for dims, per in (((4, 4, 2, 6), 2), ((8, 4, 4, 8), 2), ((4, 2, 2, 4), 1)):      # per = reals per site and plane
        for N in (2, 4):                                                            # reals per packet (fp64 / fp32)
            n0, n1, n2, n3 = dims
            s3 = n0 // 2 * n1 * n2
            if (s3 * per) % N:
                continue
            x3_lo, x3_hi = 1, n3 - 1
            nplanes = 3 if per == 2 else 6
            length = (x3_hi - x3_lo) * s3 * per // N
            slice_ = s3 * per // N
            hit_down, hit_up = set(), set()
            for k0 in range(nplanes * length):
                pl, off = divmod(k0, length)
                real0 = (x3_lo * s3 * per) + off * N                 # first real of the packet inside plane pl
                site, x3 = real0 // per, (real0 // per) // s3
                if off < slice_:
                    assert x3 == x3_lo
                    land = pl * slice_ + off
                    assert land * N == pl * s3 * per + (site - x3_lo * s3) * per + real0 % per
                    hit_down.add(land)
                if off >= length - slice_:
                    assert x3 == x3_hi - 1
                    land = pl * slice_ + (off - (length - slice_))
                    assert land * N == pl * s3 * per + (site - (x3_hi - 1) * s3) * per + real0 % per
                    hit_up.add(land)
            assert hit_down == hit_up == set(range(nplanes * slice_))


def test_traffic_json_matches_the_kernel_bench_launches(tmp_path, monkeypatch):
    """profiles/traffic.json must hold the entry bench.py looks up for the default options (a re-templated kernel
    without a fresh ncu capture would make bench.py fail on the GPU box), and sweep.traffic_from_ncu must parse an
    `ncu --page raw --csv` export into that key format."""
    import json
    import bench
    import sweep

    class FakeLat:
        def get_option(self, name):
            return {"dslash_minblocks": 0, "layout": 0, "l2_hints": 0}[name]

    class FakeL:
        F64, F32, RECON_18, RECON_12 = 0, 1, 0, 1
    name = bench.dslash_kernel_name(FakeLat(), FakeL, FakeL.F64, FakeL.RECON_18)
    table = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
    assert name in table and table[name]["dram_bytes"] > 6e8
    assert bench.ncu_traffic(name)["dram_bytes"] == table[name]["dram_bytes"]
    # the committed capture is of THIS checkout's kernel sources (else bench.py reports roofline.traffic = null)
    assert table[name]["source_hash"] == sweep.kernel_source_hash() and bench.ncu_traffic(name)["stale"] is False
    with pytest.raises(SystemExit):
        bench.ncu_traffic("dslash_kernel<double,9,9>")
    # the parser, on a fabricated export, writing into a scratch root
    (tmp_path / "profiles").mkdir()
    monkeypatch.setattr(sweep, "ROOT", str(tmp_path))
    csvp = tmp_path / "raw.csv"
    csvp.write_text('"ID","Kernel Name","dram__bytes_read.sum","dram__bytes_write.sum","gpu__time_duration.sum"\n'
                    '"","","Mbyte","Kbyte","us"\n'
                    '"0","void dslash_kernel<double, 0, 0, 0, 2, 0, 0, 0>(Geom, int, T1 *)","600.5","5000","94.0"\n'
                    '"1","void dslash_kernel<double, 0, 0, 0, 2, 0, 0, 0>(Geom, int, T1 *)","601.5","7000","96.0"\n')
    sweep.traffic_from_ncu(str(csvp), "abc1234", "test")
    got = json.load(open(tmp_path / "profiles" / "traffic.json"))
    ent = got[name]
    assert ent["launches_captured"] == 2 and ent["commit"] == "abc1234" and ent["source_hash"] == sweep.kernel_source_hash()
    assert abs(ent["dram_bytes"] - (601.0e6 + 6.0e6)) < 1 and abs(ent["ncu_duration_us"] - 95.0) < 1e-9
