"""Volume sweep and solve-to-tolerance runs (BASELINE.json configs[3] and configs[4]).

    python sweep.py --ladder            # config 5: ns/site, GB/s vs volume
    python sweep.py --multishift        # config 4: 24^3x48 and 32^4 solves
    python sweep.py --dims 16,16,16,16 --ladder
    python sweep.py --slab              # NEXT-2: slab path (torchrun for N > 1)
    python sweep.py --backfield         # Dslash with the backfield, both storage formats, all precisions / link formats
    python sweep.py --staples --dims 32,32,32,32 --variants 2 --options 'staples_minblocks=2;staples_minblocks=3'

Prints one JSON line per measurement and, with --md FILE, appends a Markdown table.  Timing is by
CUDA events on the launching stream after warm-up.  Volumes whose links fit the 126 MB L2 are
labelled "L2" (they are not HBM measurements).  Inputs are the seeded synthetic
fields of lqcd_inputs; nothing here touches oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

L2_BYTES = 126e6
BYTES = {(0, 0): 1248, (0, 1): 864, (1, 0): 624, (1, 1): 432}
LADDER = [(8,) * 4, (12,) * 4, (16,) * 4, (20,) * 4, (24,) * 4, (32, 32, 8, 32), (32, 32, 32, 8), (32,) * 4,
          (32, 32, 32, 36), (40,) * 4, (64, 64, 64, 16), (48,) * 4]


def ev_time_us(torch, fn, n, warm):
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(n):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / n * 1e3


def iter_time_us(torch, lat, links, b, shifts, mass, n_lo, n_hi):
    """(multi-shift) CG time per iteration from two fixed-length solves (unreachable tol)."""
    xs = [lat.new_spinor() for _ in shifts]

    def solve(n):
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        lat.cg_multishift(xs, b, links, mass, shifts, 1e-300, n, raise_on_max_iter=False)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    solve(n_lo)
    t_lo = min(solve(n_lo) for _ in range(2))
    t_hi = min(solve(n_hi) for _ in range(2))
    return (t_hi - t_lo) / (n_hi - n_lo) * 1e3


def ladder(dims_list, eps, seed, out):
    import numpy as np
    import torch
    import lqcd_inputs as gen
    import paper_1701_00426_b200 as L

    for dims in dims_list:
        V = gen.volume(dims)
        Vh = V // 2
        t0 = time.time()
        rng = np.random.default_rng(seed)
        U = gen.smooth_links(dims, eps, rng)
        ie, io = gen.gaussian_half_spinor(dims, rng), gen.gaussian_half_spinor(dims, rng)
        gen_s = time.time() - t0
        for prec in (0, 1):
            for recon in (0, 1):
                lat = L.Lattice(dims, prec=prec, recon=recon)
                links = lat.pack_links(U)
                a, b = lat.pack_spinor(ie, 0), lat.pack_spinor(io, 1)
                oo, oe = lat.new_spinor(), lat.new_spinor()

                def step():
                    lat.dslash(1, oo, a, links)
                    lat.dslash(0, oe, b, links)
                n = max(20, min(500, int(2e8 / V)))
                us = ev_time_us(torch, step, n, 5) / 2
                rec = dict(kind="dslash", dims="x".join(map(str, dims)), V=V, prec=("f64", "f32")[prec],
                           links=(18, 12)[recon], us=round(us, 2), ns_per_site=round(us * 1e3 / Vh, 4),
                           GBs=round(BYTES[(prec, recon)] * Vh / us / 1e3, 1),
                           GFLOPs=round(570 * Vh / us / 1e3, 1),
                           regime="L2" if lat.links_bytes < L2_BYTES else "HBM", gen_s=round(gen_s, 1))
                out(rec)
                if recon == 0:
                    it_us = iter_time_us(torch, lat, links, a, [0.0], 0.01, 20, 220)   # config 5: 200 iterations
                    es = 8 if prec == 0 else 4
                    by = (2 * (18 * 8 + 12) + 6 + 18 + 30) * es
                    out(dict(kind="cg", dims=rec["dims"], V=V, prec=rec["prec"], links=18, us_per_iter=round(it_us, 2),
                             iter_per_s=round(1e6 / it_us, 1), GBs=round(by * Vh / it_us / 1e3, 1), regime=rec["regime"]))
                lat.close()
                del links, a, b, oo, oe
        del U


def multishift(dims_list, out):
    import numpy as np
    import torch
    import lqcd_inputs as gen
    import paper_1701_00426_b200 as L

    for dims in dims_list:
        rng = np.random.default_rng(4)
        U = gen.smooth_links(dims, 0.3, rng)
        b = gen.gaussian_half_spinor(dims, rng)
        shifts = gen.rhmc_shifts(8)
        lat = L.Lattice(dims)
        links, be = lat.pack_links(U), lat.pack_spinor(b, 0)
        xs = [lat.new_spinor() for _ in shifts]
        lat.cg_multishift(xs, be, links, 0.0025, shifts, 1e-10, 50, raise_on_max_iter=False)   # warm-up
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        res = lat.cg_multishift(xs, be, links, 0.0025, shifts, 1e-10, 50000)
        dt = time.perf_counter() - t0
        out(dict(kind="multishift_solve", dims="x".join(map(str, dims)), mass=0.0025, tol=1e-10, iters=res["iters"],
                 conv_iter=res["conv_iter"].tolist(), max_true_rel_resid=float(res["rel_resid"].max()),
                 seconds=round(dt, 4), iter_per_s=round(res["iters"] / dt, 1)))
        lat.close()


def slab(dims_list, out, transports=("peer", "hooks")):
    """Strong-scaling Dslash / multi-shift CG of ONE lattice split into x3 slabs, one per rank (torchrun for
    WORLD_SIZE > 1; alone it measures the slab path's own overhead against the plain single-context run).
    Transports: "peer" = the library's own peer-to-peer transport (CUDA IPC between the processes), "hooks" =
    torch.distributed (NCCL) called back from inside the solver."""
    import numpy as np
    import torch
    import lqcd_inputs as gen
    import paper_1701_00426_b200 as L
    from paper_1701_00426_b200 import dist as D
    from paper_1701_00426_b200.slab import SlabLattice

    rank, local_rank, world = D.init("nccl")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    shifts = gen.rhmc_shifts(8)

    def iter_us(solver, xs, a, links):
        def solve(n):
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            solver(xs, a, links, 0.0025, shifts, 1e-300, n, raise_on_max_iter=False)
            e1.record()
            torch.cuda.synchronize()
            return e0.elapsed_time(e1)
        solve(16)
        t_lo, t_hi = min(solve(16), solve(16)), min(solve(80), solve(80))
        return D.max_over_ranks((t_hi - t_lo) / 64 * 1e3, world, device)

    for dims in dims_list:
        rng = np.random.default_rng(3)
        U = gen.smooth_links(dims, 0.3, rng)
        ie, io = gen.gaussian_half_spinor(dims, rng), gen.gaussian_half_spinor(dims, rng)
        V = gen.volume(dims)
        name = "x".join(map(str, dims))
        if world == 1:       # the plain single-context path on the same inputs: what the slab path's overhead is measured against
            lat = L.Lattice(dims, device=local_rank)
            links = lat.pack_links(U)
            a, b = lat.pack_spinor(ie, 0), lat.pack_spinor(io, 1)
            oo, oe = lat.new_spinor(), lat.new_spinor()

            def step0():
                lat.dslash(1, oo, a, links)
                lat.dslash(0, oe, b, links)
            us = ev_time_us(torch, step0, 200, 10) / 2
            out(dict(kind="slab_dslash", dims=name, world=1, transport="none (plain context)", overlap=False, us=round(us, 2),
                     ns_per_site=round(us * 1e3 / (V // 2), 4), GBs_aggregate=round(1248 * (V // 2) / us / 1e3, 1)))
            xs = [lat.new_spinor() for _ in shifts]
            it = iter_us(lat.cg_multishift, xs, a, links)
            out(dict(kind="slab_multishift8", dims=name, world=1, transport="none (plain context)", us_per_iter=round(it, 2),
                     iter_per_s=round(1e6 / it, 1), graph=lat.get_option("graph_active")))
            lat.close()
            del links, a, b, oo, oe, xs
        for transport in transports:
            sl = SlabLattice(dims, world, rank, device=local_rank, transport=transport)
            if transport == "peer" and world > 1:
                sl.connect_ipc()
            links = sl.pack_links(U)
            a, b = sl.pack_spinor(ie, 0), sl.pack_spinor(io, 1)
            oo, oe = sl.new_spinor(), sl.new_spinor()
            for overlap in ((False,) if transport == "peer" else (True, False)):
                def step():
                    sl.dslash(1, oo, a, links, overlap=overlap)
                    sl.dslash(0, oe, b, links, overlap=overlap)
                D.barrier(world)
                us = D.max_over_ranks(ev_time_us(torch, step, 200, 10) / 2, world, device)
                if rank == 0:
                    out(dict(kind="slab_dslash", dims=name, world=world, transport=transport, overlap=overlap,
                             us=round(us, 2), ns_per_site=round(us * 1e3 / (V // 2), 4),
                             GBs_aggregate=round(1248 * (V // 2) / us / 1e3, 1)))
            xs = [sl.new_spinor() for _ in shifts]
            D.barrier(world)
            it = iter_us(sl.cg_multishift, xs, a, links)
            if rank == 0:
                out(dict(kind="slab_multishift8", dims=name, world=world, transport=transport, us_per_iter=round(it, 2),
                         iter_per_s=round(1e6 / it, 1), graph=sl.lat.get_option("graph_active")))
            sl.close()
            del links, a, b, oo, oe, xs
    D.barrier(world)
    D.finalize(world)


def backfield(dims_list, out):
    """Dslash with the backfield (the paper's fourth acc_Deo argument): plain / theta stored (format 0) / (cos, sin) stored
    (format 1), fp64 and fp32, 18- and 12-real links; us per launch over 500 alternating (D_oe, D_eo) pairs."""
    import numpy as np
    import torch
    import lqcd_inputs as gen
    import paper_1701_00426_b200 as L

    for dims in dims_list:
        rng = np.random.default_rng(5)
        U = gen.smooth_links(dims, 0.5, rng)
        ie, io = gen.gaussian_half_spinor(dims, rng), gen.gaussian_half_spinor(dims, rng)
        theta = gen.uniform_backfield(dims, np.random.default_rng(33))
        Vh = gen.volume(dims) // 2
        for prec in (0, 1):
            for recon in (0, 1):
                rec = dict(kind="backfield", dims="x".join(map(str, dims)), prec=("f64", "f32")[prec], links=(18, 12)[recon])
                for label, fmt, add in (("plain_us", None, 0), ("theta_us", 0, 64), ("cossin_us", 1, 128)):
                    lat = L.Lattice(dims, prec=prec, recon=recon, options=dict(backfield_format=fmt or 0))
                    links = lat.pack_links(U)
                    if fmt is not None:
                        lat.set_backfield(lat.pack_backfield(theta))
                    a, b, oo, oe = lat.pack_spinor(ie, 0), lat.pack_spinor(io, 1), lat.new_spinor(), lat.new_spinor()

                    def step():
                        lat.dslash(1, oo, a, links)
                        lat.dslash(0, oe, b, links)
                    us = ev_time_us(torch, step, 500, 10) / 2
                    rec[label] = round(us, 1)
                    by = (BYTES[(prec, recon)] + add // (1 + prec)) * Vh
                    rec[label.replace("_us", "_GBs")] = round(by / us / 1e3, 0)
                    lat.close()
                    del links, a, b, oo, oe
                out(rec)


def staples(dims_list, out, variants=(0, 1, 2), precs=(0, 1), recons=(0, 1), option_sets=({},)):
    """NEXT-4: gauge staples, the three algorithm variants, fp64 / fp32, 18- / 12-real links; option_sets: extra
    lqcd_set_option settings to sweep (e.g. staples_minblocks, staples_x2block), one run per set."""
    import numpy as np
    import torch
    import lqcd_inputs as gen
    import paper_1701_00426_b200 as L

    flop_site = 4 * (84 * 198 + 24 * 36)       # the definition's count: 84 SU(3) products per link
    for dims in dims_list:
        rng = np.random.default_rng(5)
        U = gen.smooth_links(dims, 0.5, rng)
        V = gen.volume(dims)
        for prec in precs:
            for recon in recons:
                for variant in variants:
                    for opts in option_sets:
                        lat = L.Lattice(dims, prec=prec, recon=recon, options=dict(opts, staples_variant=variant))
                        links = lat.pack_links(U)
                        buf = lat.gauge_staples(links)
                        us = ev_time_us(torch, lambda: lat.gauge_staples(links, out=buf), 10, 2)
                        out(dict(kind="staples", dims="x".join(map(str, dims)), prec=("f64", "f32")[prec], links=(18, 12)[recon],
                                 variant=variant, options=",".join(f"{k}={v}" for k, v in opts.items()) or "-",
                                 ran=lat.get_option("staples_ran"), us=round(us, 1), ns_per_site=round(us * 1e3 / V, 3),
                                 TFLOPs=round(flop_site * V / us / 1e6, 2)))
                        lat.close()
                        del links, buf


_UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
_TIME_US = {"ns": 1e-3, "us": 1.0, "usecond": 1.0, "nsecond": 1e-3, "ms": 1e3, "msecond": 1e3, "s": 1e6, "second": 1e6}
KERNEL_SOURCES = ("dslash.cu", "su3.cuh", "common.cuh")      # what the headline kernel is compiled from
SRC_DIR = os.path.join(os.path.dirname(os.path.abspath(__file__)), "paper_1701_00426_b200", "csrc")


def kernel_source_hash():
    """sha256 (first 16 hex digits) over the sources of the Dslash kernel: profiles/traffic.json carries the hash of the
    build its ncu capture was taken from, bench.py compares it with the checkout it runs."""
    import hashlib
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        with open(os.path.join(SRC_DIR, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def launches_from_ncu(csv_path, md_path):
    """Aggregate an `ncu --metrics gpu__time_duration.sum --csv --log-file X.csv` launch list into a Markdown table
    (launches, total / avg / min / max us, share of the summed device time) per kernel and grid; appended to md_path."""
    import csv
    lines = open(csv_path, errors="replace").read().splitlines()
    start = next(i for i, ln in enumerate(lines) if ln.startswith('"ID"'))
    rows = list(csv.reader(lines[start:]))
    hdr = rows[0]
    col = {n: hdr.index(n) for n in ("Kernel Name", "Grid Size", "Metric Name", "Metric Unit", "Metric Value")}
    acc, order = {}, []
    for r in rows[1:]:
        if len(r) <= col["Metric Value"] or r[col["Metric Name"]] != "gpu__time_duration.sum":
            continue
        key = (r[col["Kernel Name"]].split("(")[0].strip(), r[col["Grid Size"]])
        us = float(r[col["Metric Value"]].replace(",", "")) * _TIME_US[r[col["Metric Unit"]]]
        if key not in acc:
            acc[key] = []
            order.append(key)
        acc[key].append(us)
    total = sum(sum(v) for v in acc.values())
    n_all = sum(len(v) for v in acc.values())
    with open(md_path, "a") as f:
        f.write(f"\n{n_all} launches, {total / 1e3:.1f} ms of summed device time\n\n"
                "| launches | total us | avg us | min us | max us | share | kernel |\n|---|---|---|---|---|---|---|\n")
        for key in order:
            v = acc[key]
            f.write(f"| {len(v)} | {sum(v):.1f} | {sum(v) / len(v):.2f} | {min(v):.2f} | {max(v):.2f} | "
                    f"{100 * sum(v) / total:.1f} % | `{key[0]}` grid {key[1]} |\n")
    print(json.dumps({"launches": n_all, "total_ms": total / 1e3, "kernels": len(acc)}))


def traffic_from_ncu(csv_path, commit, source):
    """Write profiles/traffic.json from `ncu -i X.ncu-rep --page raw --csv > csv_path` (an `ncu --set full`
    capture): per kernel (demangled name, template arguments without spaces), the mean over the captured
    launches of dram__bytes_read.sum + dram__bytes_write.sum, with the commit the capture was taken at.
    bench.py reads the entry of the kernel it launches and refuses a file that lacks it."""
    import csv
    import re
    rows = list(csv.reader(open(csv_path)))
    hdr, units = rows[0], rows[1]
    col = {n: hdr.index(n) for n in ("Kernel Name", "dram__bytes_read.sum", "dram__bytes_write.sum", "gpu__time_duration.sum")}
    acc = {}
    for r in rows[2:]:
        m = re.match(r"(?:void )?([A-Za-z_0-9]+<[^(]*>|[A-Za-z_0-9]+)\(", r[col["Kernel Name"]])
        if not m:
            continue
        name = m.group(1).replace(" ", "")
        rd = float(r[col["dram__bytes_read.sum"]]) * _UNIT[units[col["dram__bytes_read.sum"]]]
        wr = float(r[col["dram__bytes_write.sum"]]) * _UNIT[units[col["dram__bytes_write.sum"]]]
        acc.setdefault(name, []).append((rd, wr, float(r[col["gpu__time_duration.sum"]])))
    path = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        with open(path) as f:
            table = json.load(f)
    except Exception:
        table = {}
    for name, v in acc.items():
        n = len(v)
        table[name] = {"dram_bytes": sum(a + b for a, b, _ in v) / n, "dram_read_bytes": sum(a for a, _, _ in v) / n,
                       "dram_write_bytes": sum(b for _, b, _ in v) / n, "launches_captured": n,
                       "ncu_duration_us": sum(t for _, _, t in v) / n, "commit": commit, "source": source,
                       "source_hash": kernel_source_hash(), "hashed_files": list(KERNEL_SOURCES)}
    with open(path, "w") as f:
        json.dump(table, f, indent=1, sort_keys=True)
        f.write("\n")
    print(json.dumps({k: table[k] for k in acc}, indent=1))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--traffic-from-ncu", default=None, metavar="RAW.csv",
                    help="write profiles/traffic.json from an `ncu --page raw --csv` export (no GPU needed)")
    ap.add_argument("--commit", default="", help="with --traffic-from-ncu: the commit the capture was taken at")
    ap.add_argument("--source", default="", help="with --traffic-from-ncu: the profiles/*.md that describes the capture")
    ap.add_argument("--launches-from-ncu", default=None, metavar="LAUNCHES.csv",
                    help="aggregate an `ncu --metrics gpu__time_duration.sum --csv` log into a table appended to --md (no GPU needed)")
    ap.add_argument("--ladder", action="store_true")
    ap.add_argument("--multishift", action="store_true")
    ap.add_argument("--staples", action="store_true", help="NEXT-4 gauge staples timing")
    ap.add_argument("--slab", action="store_true", help="x3-slab path (run under torchrun for more than one GPU)")
    ap.add_argument("--dims", default=None, help="comma-separated N0,N1,N2,N3 (repeatable with ';')")
    ap.add_argument("--variants", default="0,1,2", help="with --staples: algorithm variants to time")
    ap.add_argument("--precs", default="0,1", help="with --staples: 0 = fp64, 1 = fp32")
    ap.add_argument("--recons", default="0,1", help="with --staples: 0 = 18-real, 1 = 12-real links")
    ap.add_argument("--options", default="", help="with --staples: option sets to sweep, e.g. "
                    "'staples_minblocks=2,staples_x2block=4;staples_minblocks=3,staples_x2block=0' (one run per ';' set)")
    ap.add_argument("--backfield", action="store_true", help="Dslash with / without the backfield, both storage formats")
    ap.add_argument("--eps", type=float, default=0.5)
    ap.add_argument("--seed", type=int, default=5)
    ap.add_argument("--md", default=None)
    args = ap.parse_args()
    if args.traffic_from_ncu:
        traffic_from_ncu(args.traffic_from_ncu, args.commit, args.source)
        return
    if args.launches_from_ncu:
        launches_from_ncu(args.launches_from_ncu, args.md or os.path.join(ROOT, "profiles", "launches.md"))
        return
    dims_list = None
    if args.dims:
        dims_list = [tuple(int(x) for x in d.split(",")) for d in args.dims.split(";")]
    rows = []

    def out(rec):
        rows.append(rec)
        print(json.dumps(rec), flush=True)

    if args.ladder:
        ladder(dims_list or LADDER, args.eps, args.seed, out)
    if args.multishift:
        multishift(dims_list or [(24, 24, 24, 48), (32, 32, 32, 32)], out)
    if args.staples:
        ints = lambda t: tuple(int(v) for v in t.split(","))   # noqa: E731
        sets = [dict((kv.split("=")[0], int(kv.split("=")[1])) for kv in st.split(",") if kv) for st in args.options.split(";")] \
            if args.options else [{}]
        staples(dims_list or [(16,) * 4, (32, 32, 32, 8), (32,) * 4], out, ints(args.variants), ints(args.precs), ints(args.recons), sets)
    if args.backfield:
        backfield(dims_list or [(32, 32, 32, 32)], out)
    if args.slab:
        slab(dims_list or [(32, 32, 32, 32)], out)
    if args.md:
        with open(args.md, "a") as f:
            for kind in ("dslash", "cg", "multishift_solve", "slab_dslash", "slab_multishift8", "staples", "backfield"):
                sel = [r for r in rows if r["kind"] == kind]
                if not sel:
                    continue
                keys = [k for k in sel[0] if k != "kind"]
                f.write(f"\n### {kind}\n\n| " + " | ".join(keys) + " |\n|" + "---|" * len(keys) + "\n")
                for r in sel:
                    f.write("| " + " | ".join(str(r[k]) for k in keys) + " |\n")


if __name__ == "__main__":
    main()
