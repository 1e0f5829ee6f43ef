#!/usr/bin/env python
"""bench.py -- staggered Dslash / CG throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Workload = BASELINE.json configs[2] ("config 3" of SURVEY.md section 8(d)): 32^4 lattice, fp64,
18-real links, U = exp(i*0.3*H) seed 3, fixed Gaussian inputs.  One STEP = D_oe (odd <- even)
followed by D_eo (even <- odd) from FIXED inputs (no ping-pong: rho(D) > 1 would overflow),
i.e. one pass over all V sites; the default --steps 1000 is twice the config's "1000
applications, parities alternated" (longer, so that the clock sampler sees the timed region).  metric = Dslash ns/site = step time / V (= time of one parity / (V/2)).

The JSON line also carries: roofline (HBM, algorithmic 1248 B/site against MEASURED_PEAKS.json),
e2e (same metric through lqcd_dslash_host_vectors with host vectors, copies inside the timed region; links
resident as the operator -- the all-inclusive lqcd_dslash_host figure is reported beside it as cold_links),
cpu_baseline (the oracle on the host cores, bounded sample), clocks, gpu_launches, and `extra`
(12-real, fp32, CG and multi-shift CG iter/s with their own algorithmic-bytes rooflines).

--impl reference times the CPU oracle (this tier has no reference implementation).
Links (604 MB) exceed the 126 MB L2, so successive applications cannot reuse them from cache
("inputs larger than L2" rule); stated in config.l2.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

DIMS = (32, 32, 32, 32)
EPS, SEED = 0.3, 3
FLOP_PER_SITE = 570          # 8*66 + 7*6, SURVEY.md section 8(a) a4
BYTES_PER_SITE = {("f64", 18): 1248, ("f64", 12): 864, ("f32", 18): 624, ("f32", 12): 432}
FALLBACK_HBM_GBS = 6650.0    # /opt/skills/guides/B200_PROFILING.md fallback
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the headline kernel, from the ncu --set full
# capture summarised in profiles/ncu_dslash_r1d.md (629.3 MB read + 5.3 MB written; algorithmic 654.3 MB)
NCU_DRAM_TRAFFIC_BYTES = 634.6e6


def measured_hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                smax = float(r[1])
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax,
                "reasons": sorted(reasons), "samples": len(sm)}


def timed_loop(torch, fn, steps, warmup, world, dist_mod, device):
    """W untimed + exactly K timed steps, barrier + synchronize on both sides, CUDA events on the
    launching (current) stream, MAX over ranks.  Returns total ms."""
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    dist_mod.barrier(world)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    dist_mod.barrier(world)
    return dist_mod.max_over_ranks(e0.elapsed_time(e1), world, device)


def cpu_oracle_dslash(U, psi, min_seconds=10.0, max_reps=50):
    """The oracle as it stands on the host cores: full-lattice D psi (both parities = one step)."""
    import oracle
    oracle.dirac_full(DIMS, U, psi)           # page in
    reps, t0 = 0, time.perf_counter()
    while True:
        oracle.dirac_full(DIMS, U, psi)
        reps += 1
        dt = time.perf_counter() - t0
        if dt >= min_seconds or reps >= max_reps:
            break
    V = psi.shape[0]
    return dt / reps * 1e9 / V, reps, oracle.num_threads()


def run_reference(args):
    """--impl reference: this tier has no reference implementation, so the arm times the CPU oracle
    (oracle/staggered_oracle.c, as it stands) on the same config and metric.  Each step is a
    bounded sample of the workload: a contiguous range of S lattice sites of the 32^4 problem,
    S chosen from one calibration pass so that W+K steps end within ~2 minutes.  Rank 0 only."""
    from paper_1701_00426_b200 import dist as D
    rank, _, _ = D.env_world()
    if rank != 0:
        return
    import numpy as np
    import lqcd_inputs as gen
    import oracle
    rng = np.random.default_rng(SEED)
    U = gen.smooth_links(DIMS, EPS, rng)
    psi = gen.gaussian_spinor(DIMS, rng)
    V = psi.shape[0]
    out = np.zeros_like(psi)
    t0 = time.perf_counter()
    oracle.dirac_range(DIMS, U, psi, out, 0, V)                  # calibration + page-in, untimed
    t_full = time.perf_counter() - t0
    budget = 100.0 / max(1, args.steps + args.warmup)              # seconds per step
    S = int(min(V, max(4096, V * budget / t_full)))
    starts = [(k * 7919 * 4096) % (V - S + 1) for k in range(args.steps + args.warmup)]
    for k in range(args.warmup):
        oracle.dirac_range(DIMS, U, psi, out, starts[k], starts[k] + S)
    t0 = time.perf_counter()
    for k in range(args.warmup, args.warmup + args.steps):
        oracle.dirac_range(DIMS, U, psi, out, starts[k], starts[k] + S)
    dt = time.perf_counter() - t0
    ns = dt * 1e9 / (args.steps * S)
    cores = oracle.num_threads()
    sample = f"{args.steps} steps x {S} contiguous sites of the 32^4 lattice (oracle_dirac_range), all {cores} threads"
    line = {
        "impl": "reference", "metric": "dslash_ns_per_site", "value": ns, "unit": "ns/site",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(),
        "cpu_baseline": {"value": ns, "unit": "ns/site", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": ns, "unit": "ns/site", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config():
    return {"workload": "BASELINE.json configs[2]: Dslash on 32^4, fp64, 18-real links; one step = D_oe then D_eo "
                        "from fixed inputs (V sites)",
            "dims": list(DIMS), "links": "U = exp(i*0.3*H) re-unitarised, seed 3", "spinors": "Gaussian, fixed",
            "bc": "periodic x0-x2, antiperiodic x3",
            "l2": "inputs larger than L2 (links 604 MB vs 126 MB L2); no flush needed"}


def solver_iter_rate(torch, lat, L, links, b_e, shifts, mass, n_lo=24, n_hi=120, rational=False):
    """Time per (multi-shift) CG iteration by differencing two fixed-length solves (tol is
    unreachable, so every shift stays active: worst-case K2 traffic).  Setup, the true-residual
    epilogue and the final sync cancel in the difference."""
    xs = [lat.new_spinor() for _ in shifts]

    def solve(n):
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        if rational:   # lqcd_rational_apply: y accumulated in K2, the x_i are never stored
            res = lat.rational_apply(xs[0], b_e, links, mass, shifts, 0.5, [1.0] * len(shifts), 1e-300, n,
                                     raise_on_max_iter=False)
        else:
            res = lat.cg_multishift(xs, b_e, links, mass, shifts, 1e-300, n, raise_on_max_iter=False)
        e1.record()
        torch.cuda.synchronize()
        assert res["iters"] == n, res
        return e0.elapsed_time(e1)

    solve(n_lo)                                   # warm-up
    t_lo = min(solve(n_lo) for _ in range(2))
    t_hi = min(solve(n_hi) for _ in range(2))
    return (t_hi - t_lo) / (n_hi - n_lo)          # ms per iteration


def ensure_built():
    """A fresh checkout has no .so (git-ignored): compile it (nvcc, sm_100a) before the first import.
    This builds the CUDA library; it never substitutes another code path."""
    if not os.path.exists(os.path.join(ROOT, "paper_1701_00426_b200", "liblqcd_b200.so")):
        import __graft_entry__
        __graft_entry__.build()


def run_ours(args):
    import numpy as np
    import torch
    import lqcd_inputs as gen
    if int(os.environ.get("RANK", "0")) == 0:
        ensure_built()
    else:                                    # other ranks wait for rank 0's build
        t0 = time.time()
        while not os.path.exists(os.path.join(ROOT, "paper_1701_00426_b200", "liblqcd_b200.so")) and time.time() - t0 < 600:
            time.sleep(1.0)
    import paper_1701_00426_b200 as L
    from paper_1701_00426_b200 import dist as D

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the lqcd_b200 path has no CPU fallback")
    rank, local_rank, world = D.init("nccl")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    peak, peak_src = measured_hbm_peak()

    # ---- inputs (seeded, synthetic) -- replicas: seed offset per rank
    rng = np.random.default_rng(D.replica_seed(SEED, rank))
    U = gen.smooth_links(DIMS, EPS, rng)
    in_e = gen.gaussian_half_spinor(DIMS, rng)
    in_o = gen.gaussian_half_spinor(DIMS, rng)
    V = gen.volume(DIMS)
    Vh = V // 2

    lat = L.Lattice(DIMS, prec=L.F64, recon=L.RECON_18, device=local_rank)
    links = lat.pack_links(U)
    d_in_e, d_in_o = lat.pack_spinor(in_e, L.EVEN), lat.pack_spinor(in_o, L.ODD)
    d_out_e, d_out_o = lat.new_spinor(), lat.new_spinor()

    def step():
        lat.dslash(L.ODD, d_out_o, d_in_e, links)     # D_oe
        lat.dslash(L.EVEN, d_out_e, d_in_o, links)    # D_eo

    # ---- headline: K steps, inputs resident in HBM -------------------------------------------
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    n0 = lat.launches
    ms = timed_loop(torch, step, args.steps, args.warmup, world, D, device)
    launches = lat.launches - n0 - 2 * args.warmup
    clocks = sampler.stop() if rank == 0 else None
    ns_site = D.aggregate_ns_per_site(ms, args.steps, V, world)
    us_launch = ms * 1e3 / (2 * args.steps)
    achieved = BYTES_PER_SITE[("f64", 18)] * Vh / (us_launch * 1e-6) / 1e9

    # ---- e2e: lqcd_dslash_host, pinned host buffers, copies inside the timed region ----------
    def pinned(a):
        t = torch.from_numpy(np.ascontiguousarray(a).view(np.float64).reshape(-1)).pin_memory()
        return t, t.numpy().view(np.complex128).reshape(a.shape)
    keep_U, hU = pinned(U)
    keep_i, h_in_e = pinned(in_e)
    keep_j, h_in_o = pinned(in_o)
    keep_o, h_out = pinned(np.zeros_like(in_e))

    # (a) the step's inputs are the two vectors; the link field is the OPERATOR: resident on the device,
    #     uploaded once per gauge configuration and reused by every application
    def e2e_step():
        lat.dslash_host_vectors(L.ODD, h_out, h_in_e, links)
        lat.dslash_host_vectors(L.EVEN, h_out, h_in_o, links)
    e2e_steps = max(1, min(args.steps, 50))
    e2e_ms = timed_loop(torch, e2e_step, e2e_steps, 2, world, D, device)
    h2d = 2 * in_e.nbytes
    d2h = 2 * in_e.nbytes

    # (b) worst case, nothing resident: the 604 MB canonical link field crosses PCIe in every call too
    def e2e_cold_step():
        lat.dslash_host(L.ODD, h_out, h_in_e, hU)
        lat.dslash_host(L.EVEN, h_out, h_in_o, hU)
    cold_steps = max(1, min(args.steps, 5))
    cold_ms = timed_loop(torch, e2e_cold_step, cold_steps, 1, world, D, device)
    del keep_U, hU

    line = None
    if rank == 0:
        extra = {}
        # ---- other Dslash variants (config 3's 12-real arm, config 5's fp32) -------------------
        for prec, pname in ((L.F64, "f64"), (L.F32, "f32")):
            for recon, rn in ((L.RECON_18, 18), (L.RECON_12, 12)):
                if prec == L.F64 and recon == L.RECON_18:
                    continue
                lt = L.Lattice(DIMS, prec=prec, recon=recon, device=local_rank)
                lk = lt.pack_links(U)
                a, b_, o1, o2 = lt.pack_spinor(in_e, 0), lt.pack_spinor(in_o, 1), lt.new_spinor(), lt.new_spinor()

                def st():
                    lt.dslash(L.ODD, o1, a, lk)
                    lt.dslash(L.EVEN, o2, b_, lk)
                t = timed_loop(torch, st, 100, 5, 1, D, device)
                us = t * 1e3 / 200
                gbs = BYTES_PER_SITE[(pname, rn)] * Vh / (us * 1e-6) / 1e9
                extra[f"dslash_{pname}_{rn}real"] = {"ns_per_site": us * 1e3 / Vh, "GBs": gbs, "frac": gbs / peak,
                                                     "GFLOPs": FLOP_PER_SITE * Vh / (us * 1e-6) / 1e9}
                lt.close()
                del lk, a, b_, o1, o2
        # ---- CG and multi-shift CG iteration rates (configs 2/4 shaped, on 32^4) --------------
        ms_it = solver_iter_rate(torch, lat, L, links, d_in_e, [0.0], 0.01)
        by = 2928
        extra["cg_f64"] = {"iter_per_s": 1e3 / ms_it, "us_per_iter": ms_it * 1e3, "bytes_per_site_iter": by,
                           "GBs": by * Vh / (ms_it * 1e-3) / 1e9, "frac": by * Vh / (ms_it * 1e-3) / 1e9 / peak}
        shifts = gen.rhmc_shifts(8)
        ms_it = solver_iter_rate(torch, lat, L, links, d_in_e, shifts, 0.0025)
        by = 2544 + 144 + 144 + 96 + 7 * 192
        extra["multishift8_f64"] = {"iter_per_s": 1e3 / ms_it, "us_per_iter": ms_it * 1e3, "bytes_per_site_iter": by,
                                    "GBs": by * Vh / (ms_it * 1e-3) / 1e9, "frac": by * Vh / (ms_it * 1e-3) / 1e9 / peak,
                                    "note": "all 8 shifts active (worst case)"}
        ms_it = solver_iter_rate(torch, lat, L, links, d_in_e, shifts, 0.0025, rational=True)
        by = 2544 + 144 + 144 + 96 + 7 * 96
        extra["rational8_f64"] = {"iter_per_s": 1e3 / ms_it, "us_per_iter": ms_it * 1e3, "bytes_per_site_iter": by,
                                  "GBs": by * Vh / (ms_it * 1e-3) / 1e9, "frac": by * Vh / (ms_it * 1e-3) / 1e9 / peak,
                                  "note": "lqcd_rational_apply, 8 shifts all active: y += c_i alpha_i p_i fused, x_i never stored"}
        # ---- NEXT-3: fermion-force outer products from 8 solutions (n Dslash + 2 outer-product launches)
        xs8 = [lat.new_spinor() for _ in shifts]
        lat.cg_multishift(xs8, d_in_e, links, 0.0025, shifts, 1e-300, 8, raise_on_max_iter=False)
        fbuf = lat.fermion_force(xs8, links, [1.0] * 8)
        t_f = timed_loop(torch, lambda: lat.fermion_force(xs8, links, [1.0] * 8, force=fbuf), 20, 3, 1, D, device) / 20
        by = 8 * 1248 * Vh + V * (576 + 48 * 8 + 256)
        extra["fermion_force8_f64"] = {"ms": t_f, "ns_per_site": t_f * 1e6 / V, "bytes": by, "GBs": by / (t_f * 1e-3) / 1e9,
                                       "frac": by / (t_f * 1e-3) / 1e9 / peak,
                                       "note": "8 x D_oe (1248 B per odd site) + outer products (576 links + 48*8 vectors + 256 B of 8-real force per site)"}
        del xs8, fbuf
        # ---- NEXT-4: tree-level Symanzik gauge staples (ALU / cache bound: 84 SU(3) products per link)
        sbuf = lat.gauge_staples(links)
        t_s = timed_loop(torch, lambda: lat.gauge_staples(links, out=sbuf), 10, 3, 1, D, device) / 10
        flop_site = 4 * (84 * 198 + 24 * 36)
        try:
            with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
                mhz = float(json.load(f)["sm_max_mhz"])
        except Exception:
            mhz = 1965.0
        fp64_peak = 148 * 64 * 2 * mhz * 1e6 / 1e12          # 64 FP64 FMA lanes per SM
        extra["gauge_staples_f64"] = {"ms": t_s, "ns_per_site": t_s * 1e6 / V, "flop_per_site": flop_site,
                                      "TFLOPs": flop_site * V / (t_s * 1e-3) / 1e12, "bound": "alu",
                                      "peak_TFLOPs": fp64_peak, "frac": flop_site * V / (t_s * 1e-3) / 1e12 / fp64_peak,
                                      "note": "2 plaquette + 6 rectangle paths per nu, c0 = 5/3, c1 = -1/12"}
        del sbuf
        # ---- CPU oracle beside it -------------------------------------------------------------
        psi = np.zeros((V, 3), dtype=np.complex128)
        psi[gen.half_index_of_parity(DIMS, 0)] = in_e
        psi[gen.half_index_of_parity(DIMS, 1)] = in_o
        cpu_ns, reps, cores = cpu_oracle_dslash(U, psi, min_seconds=args.cpu_seconds)
        line = {
            "metric": "dslash_ns_per_site", "value": ns_site, "unit": "ns/site", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": dict(workload_config(), parallelism=f"replicas x{world} (no collective)"),
            "GFLOPs": FLOP_PER_SITE * V * world / (ms / args.steps * 1e-3) / 1e9,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": NCU_DRAM_TRAFFIC_BYTES, "traffic_source": "profiles/ncu_dslash_r1d.md (ncu --set full, per launch)",
                         "peak_source": peak_src, "kernel": "dslash_kernel<double,0,0,0,2,0>",
                         "bytes_per_launch": BYTES_PER_SITE[("f64", 18)] * Vh, "us_per_launch": us_launch,
                         "frac_of_nominal_8TBs": achieved / 8000.0},
            "e2e": {"value": e2e_ms * 1e6 / (e2e_steps * V * world), "unit": "ns/site", "steps": e2e_steps,
                    "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "api": "lqcd_dslash_host_vectors x2 per step: pinned canonical host vectors in and out, links resident "
                           "(the operator; uploaded once per configuration, PAPER.md:276)",
                    "cold_links": {"value": cold_ms * 1e6 / (cold_steps * V * world), "unit": "ns/site", "steps": cold_steps,
                                   "h2d_bytes_per_step": 2 * (U.nbytes + in_e.nbytes), "d2h_bytes_per_step": 2 * in_e.nbytes,
                                   "api": "lqcd_dslash_host x2 per step: the canonical link field is uploaded and packed in every call"}},
            "gpu_launches": launches,
            "clocks": clocks,
            "cpu_baseline": {"value": cpu_ns, "unit": "ns/site", "cores": cores, "kind": "oracle",
                             "sample": f"{reps} full-lattice applications of oracle_dirac_full at 32^4"},
            "extra": extra,
        }
    lat.close()
    D.barrier(world)
    D.finalize(world)
    if line is not None:
        print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=10.0, dest="cpu_seconds")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
