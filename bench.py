#!/usr/bin/env python
"""bench.py -- staggered Dslash / CG throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--quick]

Workload = BASELINE.json configs[2] ("config 3" of SURVEY.md section 8(d)): 32^4 lattice, fp64,
18-real links, U = exp(i*0.3*H) seed 3, fixed Gaussian inputs.  One STEP = k x (D_oe then D_eo) from
FIXED inputs (no ping-pong: rho(D) > 1 would overflow), k chosen so that the K timed steps hold at least
MIN_APPLICATIONS single-parity applications whatever --steps is (config 3: "time 1000 applications, even
and odd parity alternated"; more here, so that the clock sampler sees the timed region).
metric = Dslash ns/site = time of one single-parity application / (V/2) = time of (D_oe + D_eo) / V.

The JSON line also carries: roofline (HBM, algorithmic 1248 B/site against MEASURED_PEAKS.json; DRAM traffic
from profiles/traffic.json, the ncu capture of the SAME kernel), e2e (same metric through
lqcd_dslash_host_vectors_batch with pinned host vectors, copies inside the timed region; links resident as the
operator -- the all-inclusive lqcd_dslash_host figure is reported beside it as cold_links), cpu_baseline (the
oracle on the host cores: Dslash, CG at 16^4, multi-shift CG at 24^3 x 48; bounded samples), clocks,
gpu_launches, parity (the last timed outputs against the oracle on sampled sites), solver (the CG / multi-shift /
rational iteration rates, top level so that the driver's record keeps them), volume_ladder (Dslash and CG versus volume on
the paper's Table-3 lattices), and `extra`: 12-real / fp32 Dslash, CG / multi-shift / rational iteration rates at 32^4,
BASELINE.json configs[1], [3], [4] (16^4 CG and 24^3 x 48 / 32^4 multi-shift solves to tolerance, 48^4 and
64^3 x 16 Dslash in fp64 and fp32), the fermion force, the gauge staples against the FP64 peak measured in
this run, and the end-to-end multi-shift solve on host vectors.

--impl reference times the CPU oracle (this tier has no reference implementation); that arm
imports nothing of the product.
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
MIN_APPLICATIONS = 4000      # single-parity Dslash applications in the timed region (config 3 asks >= 1000)
CG_BYTES = 2928              # per even site and CG iteration
MS8_BYTES = 2544 + 144 + 144 + 96 + 7 * 192      # 8 shifts, all active


def measured_hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(kernel_name):
    """DRAM bytes per launch of the headline kernel from profiles/traffic.json (written by
    `python sweep.py --traffic-from-ncu` from an `ncu --set full` capture).  The entry must be for the kernel
    this run launches: a stale file (kernel renamed or re-templated) is an error, not a silent constant."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    with open(path) as f:
        t = json.load(f)
    ent = t.get(kernel_name)
    if ent is None:
        raise SystemExit(f"bench.py: profiles/traffic.json has no entry for the kernel this run launches "
                         f"({kernel_name}); re-capture it (python sweep.py --traffic-from-ncu)")
    # the capture must be of THIS build: traffic.json carries a hash of the kernel's sources (sweep.py writes it)
    import sweep
    ent = dict(ent)
    ent["source_hash_now"] = sweep.kernel_source_hash()
    ent["stale"] = ent.get("source_hash") != ent["source_hash_now"]
    return ent


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


def cpu_oracle_solvers(gen, cfg2, cfg4, ms_sample_iters):
    """The solver half of the metric on the host cores: the oracle's CG at 16^4 to
    tolerance (config 2) and its multi-shift CG at 24^3 x 48 (config 4) for a bounded number of iterations."""
    import numpy as np
    import oracle
    out = {}
    dims, U, b, mass, tol = cfg2
    t0 = time.perf_counter()
    r = oracle.cg(dims, U, mass, b, tol, 20000)
    dt = time.perf_counter() - t0
    out["cg_16x4"] = {"value": r["iters"] / dt, "unit": "iter/s", "iters": r["iters"], "seconds": dt,
                      "converged": bool(r["converged"]), "rel_resid": float(r["true_relres"]),
                      "sample": "oracle_cg at 16^4 to tol 1e-10 (BASELINE.json configs[1]), whole solve"}
    dims, U, b, mass, tol, shifts = cfg4
    t0 = time.perf_counter()
    r = oracle.cg_multishift(dims, U, mass, shifts, b, tol, ms_sample_iters)
    dt = time.perf_counter() - t0
    out["multishift_24x24x24x48"] = {"value": r["iters"] / dt, "unit": "iter/s", "iters": r["iters"], "seconds": dt,
                                     "sample": f"first {ms_sample_iters} iterations of oracle_cg_multishift at 24^3 x 48, "
                                               "8 shifts all active (BASELINE.json configs[3]); includes the oracle's "
                                               "true-residual evaluation at exit"}
    return out


def workload_config(n_gpus):
    return {"workload": "BASELINE.json configs[2]: Dslash on 32^4, fp64, 18-real links; one step = k x (D_oe then D_eo) "
                        "from fixed inputs; value = time per single-parity application / (V/2)",
            "dims": list(DIMS), "links": "U = exp(i*0.3*H) re-unitarised, seed 3", "spinors": "Gaussian, fixed",
            "bc": "periodic x0-x2, antiperiodic x3",
            "l2": "inputs larger than L2 (links 604 MB vs 126 MB L2); no flush needed",
            "parallelism": f"replicas x{n_gpus} (no collective)"}


def run_reference(args):
    """--impl reference: this tier has no reference implementation, so the arm times the CPU oracle
    (oracle/staggered_oracle.c, as it stands) on the same config and metric.  Each step is a
    bounded sample of the workload: a contiguous range of S lattice sites of the 32^4 problem,
    S chosen from one calibration pass so that W+K steps end within ~2 minutes.  Rank 0 only.
    Nothing of the product (paper_1701_00426_b200) is imported or loaded here."""
    if int(os.environ.get("RANK", "0")) != 0:
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
        "data": "synthetic", "config": workload_config(args.gpus),
        "cpu_baseline": {"value": ns, "unit": "ns/site", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": ns, "unit": "ns/site", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def ev_ms(torch, fn):
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    r = fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1), r


def solver_iter_rate(torch, lat, L, links, b_e, shifts, mass, n_lo=24, n_hi=120, rational=False):
    """Time per (multi-shift) CG iteration by differencing two fixed-length solves (tol is
    unreachable, so every shift stays active: worst-case K2 traffic).  Setup, the true-residual
    epilogue and the final sync cancel in the difference."""
    xs = [lat.new_spinor() for _ in shifts]

    def solve(n):
        def go():
            if rational:   # lqcd_rational_apply: y accumulated in K2, the x_i are never stored
                return lat.rational_apply(xs[0], b_e, links, mass, shifts, 0.5, [1.0] * len(shifts), 1e-300, n,
                                          raise_on_max_iter=False)
            return lat.cg_multishift(xs, b_e, links, mass, shifts, 1e-300, n, raise_on_max_iter=False)
        ms, res = ev_ms(torch, go)
        assert res["iters"] == n, res
        return ms

    solve(n_lo)                                   # warm-up
    t_lo = min(solve(n_lo) for _ in range(2))
    t_hi = min(solve(n_hi) for _ in range(2))
    return (t_hi - t_lo) / (n_hi - n_lo)          # ms per iteration


def solve_to_tolerance(torch, lat, links, b_e, shifts, mass, tol, peak, bytes_all_active=None):
    """A (multi-shift) CG solve to tolerance: iterations, device time (CUDA events around the blocking call),
    iter/s, worst true residual.  Second of two runs (the first builds the chunk graph)."""
    xs = [lat.new_spinor() for _ in shifts]
    go = lambda: lat.cg_multishift(xs, b_e, links, mass, shifts, tol, 100000)   # noqa: E731
    ev_ms(torch, go)
    ms, res = ev_ms(torch, go)
    out = {"iters": int(res["iters"]), "ms": ms, "iter_per_s": res["iters"] / (ms * 1e-3),
           "us_per_iter": ms * 1e3 / res["iters"], "max_true_rel_resid": float(res["rel_resid"].max()),
           "conv_iter": [int(c) for c in res["conv_iter"]], "tol": tol, "mass": mass, "nshift": len(shifts)}
    if bytes_all_active:
        out["frac_if_all_active"] = bytes_all_active * lat.Vh / (out["us_per_iter"] * 1e-6) / 1e9 / peak
    return out


def ensure_built():
    """A fresh checkout has no .so (git-ignored): compile it (nvcc, sm_100a) before the first import.
    This builds the CUDA library; it never substitutes another code path."""
    if not os.path.exists(os.path.join(ROOT, "paper_1701_00426_b200", "liblqcd_b200.so")):
        import __graft_entry__
        __graft_entry__.build()


def dslash_kernel_name(lat, L, prec, recon):
    """Name of the Dslash instantiation the default options launch (template arguments of
    dslash_kernel<T, LAYOUT, RECON12, MODE, MINB, POLICY, BF, HALO> in csrc/dslash.cu; no backfield, no peer transport)."""
    minb = lat.get_option("dslash_minblocks") or (2 if prec == L.F64 else 4)
    return (f"dslash_kernel<{'double' if prec == L.F64 else 'float'},{lat.get_option('layout')},"
            f"{1 if recon == L.RECON_12 else 0},0,{minb},{lat.get_option('l2_hints')},0,0>")


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
    kernel = dslash_kernel_name(lat, L, L.F64, L.RECON_18)
    traffic = ncu_traffic(kernel)

    # one step = k pairs, so that the timed region holds >= MIN_APPLICATIONS applications for any --steps
    k = max(1, -(-MIN_APPLICATIONS // (2 * args.steps)))

    def step():
        for _ in range(k):
            lat.dslash(L.ODD, d_out_o, d_in_e, links)     # D_oe
            lat.dslash(L.EVEN, d_out_e, d_in_o, links)    # D_eo

    # ---- headline: K steps, inputs resident in HBM -------------------------------------------
    sampler = ClockSampler(local_rank) if rank == 0 else None
    for _ in range(args.warmup):
        step()
    if sampler is not None:
        # the clock sampler starts AFTER the warm-up and the GPU is kept busy (untimed) until nvidia-smi has
        # delivered its first row, so that every sample is taken under load; it stops right after the timed region
        sampler.start()
        t0 = time.time()
        while sampler.proc and not sampler.rows and time.time() - t0 < 3.0:
            step()
            torch.cuda.synchronize()
    n0 = lat.launches
    ms = timed_loop(torch, step, args.steps, 0, world, D, device)
    launches = lat.launches - n0
    clocks = sampler.stop() if rank == 0 else None
    # the outputs of the LAST timed applications, read back outside the timed region: checked against the oracle below
    timed_out = {L.ODD: lat.unpack_spinor(d_out_o, L.ODD), L.EVEN: lat.unpack_spinor(d_out_e, L.EVEN)} if rank == 0 else None
    apps = 2 * k * args.steps
    ns_site = D.aggregate_ns_per_site(ms, k * args.steps, V, world)
    us_launch = ms * 1e3 / apps
    achieved = BYTES_PER_SITE[("f64", 18)] * Vh / (us_launch * 1e-6) / 1e9

    # read-only bandwidth over the 604 MB link field, measured here: the copy peak is half writes, this kernel is not
    read_gbs = lat.measure_hbm_read(links) if rank == 0 else None

    # ---- e2e: pinned host buffers, copies inside the timed region ----------------------------
    def pinned(a):
        t = torch.from_numpy(np.ascontiguousarray(a).view(np.float64).reshape(-1)).pin_memory()
        return t, t.numpy().view(np.complex128).reshape(a.shape)
    keep_U, hU = pinned(U)
    keep_i, h_in_e = pinned(in_e)
    keep_j, h_in_o = pinned(in_o)
    E2E_PAIRS = 4
    keep_o = [pinned(np.zeros_like(in_e)) for _ in range(2 * E2E_PAIRS)]
    h_outs = [o[1] for o in keep_o]

    # (a) the step's inputs are the vectors; the link field is the OPERATOR: resident on the device,
    #     uploaded once per gauge configuration and reused by every application.  One step =
    #     one lqcd_dslash_host_vectors_batch call of E2E_PAIRS x (D_oe, D_eo): every vector goes up and every
    #     result comes down inside the call; uploads, kernels and downloads of successive applications overlap.
    pars = [L.ODD, L.EVEN] * E2E_PAIRS
    h_ins = [h_in_e, h_in_o] * E2E_PAIRS

    def e2e_step():
        lat.dslash_host_vectors_batch(pars, h_outs, h_ins, links)
    e2e_steps = max(2, min(args.steps, 25))
    e2e_ms = timed_loop(torch, e2e_step, e2e_steps, 2, world, D, device)
    h2d = 2 * E2E_PAIRS * in_e.nbytes
    d2h = 2 * E2E_PAIRS * in_e.nbytes

    # (a') one blocking call per application (round 1's figure): upload -> compute -> download in sequence
    def e2e_serial_step():
        lat.dslash_host_vectors(L.ODD, h_outs[0], h_in_e, links)
        lat.dslash_host_vectors(L.EVEN, h_outs[1], h_in_o, links)
    ser_steps = max(2, min(args.steps, 20))
    ser_ms = timed_loop(torch, e2e_serial_step, ser_steps, 2, world, D, device)

    # (b) worst case, nothing resident: the 604 MB canonical link field crosses PCIe in every call too
    def e2e_cold_step():
        lat.dslash_host(L.ODD, h_outs[0], h_in_e, hU)
        lat.dslash_host(L.EVEN, h_outs[1], h_in_o, hU)
    cold_steps = max(1, min(args.steps, 3))
    cold_ms = timed_loop(torch, e2e_cold_step, cold_steps, 1, world, D, device)
    del keep_U, hU

    # ---- strong scaling of ONE 32^4 lattice over the N ranks: x3 slabs over the library's
    #      peer-to-peer transport; collective, every rank takes part.  At N = 1 it measures the slab path's own
    #      overhead against the plain context.  `value` above stays the replica (weak-scaling) figure.
    slab_strong = None
    if DIMS[3] % world == 0 and (DIMS[3] // world) % 2 == 0 and world <= 16:
        # (never run on more than one GPU in this project's environment: a failure of this leg -- CUDA IPC not
        # permitted, a wait for a peer that timed out -- is recorded in the line and must not cost the headline)
        try:
            slab_strong = slab_strong_leg(torch, L, D, gen, U if world == 1 else None, rank, local_rank, world, device,
                                          us_launch if world == 1 else None)
        except Exception as e:  # noqa: BLE001
            slab_strong = {"ranks": world, "error": f"{type(e).__name__}: {e}"[:300]}
        D.barrier(world)

    line = None
    if rank == 0:
        extra = {}
        if slab_strong is not None:
            extra["slab_strong"] = slab_strong
        # ---- other Dslash variants (config 3's 12-real arm, config 5's fp32) -------------------
        for prec, pname in ((L.F64, "f64"), (L.F32, "f32")):
            for recon, rn in ((L.RECON_18, 18), (L.RECON_12, 12)):
                if prec == L.F64 and recon == L.RECON_18:
                    continue
                extra[f"dslash_{pname}_{rn}real"] = dslash_rate(torch, L, D, gen, DIMS, U, in_e, in_o, prec, recon, peak, device)
        # ---- Dslash with the backfield (the paper's fourth acc_Deo argument): theta stored (+64 B per site) and
        #      (cos, sin) stored (+128 B per site)
        theta = gen.uniform_backfield(DIMS, np.random.default_rng(33))
        for fmt, add in ((0, 64), (1, 128)):
            extra[f"dslash_backfield_f64_18real_fmt{fmt}"] = dslash_rate(
                torch, L, D, gen, DIMS, U, in_e, in_o, L.F64, L.RECON_18, peak, device, theta=theta, bf_format=fmt,
                bytes_per_site=BYTES_PER_SITE[("f64", 18)] + add)
        del theta
        # ---- CG and multi-shift CG iteration rates (configs 2/4 shaped, on 32^4) --------------
        ms_it = solver_iter_rate(torch, lat, L, links, d_in_e, [0.0], 0.01)
        extra["cg_f64"] = {"iter_per_s": 1e3 / ms_it, "us_per_iter": ms_it * 1e3, "bytes_per_site_iter": CG_BYTES,
                           "GBs": CG_BYTES * Vh / (ms_it * 1e-3) / 1e9, "frac": CG_BYTES * Vh / (ms_it * 1e-3) / 1e9 / peak}
        shifts = gen.rhmc_shifts(8)
        ms_it = solver_iter_rate(torch, lat, L, links, d_in_e, shifts, 0.0025)
        by = MS8_BYTES
        extra["multishift8_f64"] = {"iter_per_s": 1e3 / ms_it, "us_per_iter": ms_it * 1e3, "bytes_per_site_iter": by,
                                    "GBs": by * Vh / (ms_it * 1e-3) / 1e9, "frac": by * Vh / (ms_it * 1e-3) / 1e9 / peak,
                                    "note": "all 8 shifts active (worst case)"}
        ms_it = solver_iter_rate(torch, lat, L, links, d_in_e, shifts, 0.0025, rational=True)
        by = 2544 + 144 + 144 + 96 + 7 * 96
        extra["rational8_f64"] = {"iter_per_s": 1e3 / ms_it, "us_per_iter": ms_it * 1e3, "bytes_per_site_iter": by,
                                  "GBs": by * Vh / (ms_it * 1e-3) / 1e9, "frac": by * Vh / (ms_it * 1e-3) / 1e9 / peak,
                                  "note": "lqcd_rational_apply, 8 shifts all active: y += c_i alpha_i p_i fused, x_i never stored"}
        # ---- BASELINE.json configs[3], second lattice: the 8-shift solve to tolerance at 32^4 -------
        extra["multishift_32x32x32x32"] = dict(
            solve_to_tolerance(torch, lat, links, d_in_e, shifts, 0.0025, 1e-10, peak, MS8_BYTES),
            note="BASELINE.json configs[3] at 32^4: 8 shifts 1e-4..1, m = 0.0025, tol 1e-10 per shift; the bench's "
                 "resident links (eps 0.3, seed 3) and rhs in_e; traffic falls as shifts freeze")
        # ---- e2e of the method: rhs up, 8 solutions down, hundreds of applications in between ------
        sol_keep, h_sol = pinned(np.zeros((8,) + in_e.shape, dtype=np.complex128))
        go = lambda: lat.cg_multishift_host_vectors(h_sol, h_in_e, links, 0.0025, shifts, 1e-10, 100000)   # noqa: E731
        ev_ms(torch, go)
        t_e2e, r_e2e = ev_ms(torch, go)
        dev = extra["multishift_32x32x32x32"]
        extra["e2e_multishift"] = {"ms": t_e2e, "iters": int(r_e2e["iters"]), "iter_per_s": r_e2e["iters"] / (t_e2e * 1e-3),
                                   "device_only_ms": dev["ms"], "overhead_frac": t_e2e / dev["ms"] - 1.0,
                                   "h2d_bytes": in_e.nbytes, "d2h_bytes": 8 * in_e.nbytes,
                                   "api": "lqcd_cg_multishift_host_vectors: pinned rhs in, 8 solutions out, links resident"}
        del sol_keep, h_sol
        # ---- NEXT-3: fermion-force outer products from 8 solutions (n Dslash + 2 outer-product launches)
        xs8 = [lat.new_spinor() for _ in shifts]
        lat.cg_multishift(xs8, d_in_e, links, 0.0025, shifts, 1e-300, 8, raise_on_max_iter=False)
        fbuf = lat.fermion_force(xs8, links, [1.0] * 8)
        # the method's own bytes: the y_i = D_oe x_i need every link of an odd site's 8 hops ONCE (1152 B) plus 96 B per
        # shift (48 in, 48 out); the outer products 576 B of links + 48 B per shift + 256 B of 8-real force per site
        by = Vh * (1152 + 96 * 8) + V * (576 + 48 * 8 + 256)
        by_block = {}
        for blk in (0, 4, 8):                 # one Dslash per shift (round 2) / two blocks of 4 / one block of 8 (default, last)
            lat.set_option("force_block", blk)
            t_b = timed_loop(torch, lambda: lat.fermion_force(xs8, links, [1.0] * 8, force=fbuf), 20, 3, 1, D, device) / 20
            by_block[str(blk)] = {"ms": t_b, "frac_of_method_bytes": by / (t_b * 1e-3) / 1e9 / peak}
        t_f = by_block["8"]["ms"]
        extra["fermion_force8_f64"] = {"ms": t_f, "ns_per_site": t_f * 1e6 / V, "bytes": by, "GBs": by / (t_f * 1e-3) / 1e9,
                                       "frac": by / (t_f * 1e-3) / 1e9 / peak, "by_force_block": by_block,
                                       "note": "block Dslash for the 8 y_i (one launch, every link once: 1152 + 8 x 96 B per odd site) + outer products "
                                               "(576 links + 48*8 vectors + 256 B of 8-real force per site)"}
        del xs8, fbuf
        # ---- NEXT-4: tree-level Symanzik gauge staples (ALU bound) against the FP64 rate measured here
        fp64_peak = lat.measure_fp64_peak()
        extra["fp64_peak_tflops"] = {"value": fp64_peak, "how": "lqcd_measure_fp64_peak: independent DFMA chains, "
                                     "num_SMs x 8 CTAs of 256 threads, best of 4 after 2 warm-up launches"}
        sbuf = lat.gauge_staples(links)
        t_s = timed_loop(torch, lambda: lat.gauge_staples(links, out=sbuf), 10, 3, 1, D, device) / 10
        variant = lat.get_option("staples_ran")
        flop_def = 4 * (84 * 198 + 24 * 36)                     # the definition: 84 products + 24 scaled adds per link
        flop_exec = 4 * STAPLES_EXEC_FLOP_PER_LINK[variant]      # what the default variant executes
        extra["gauge_staples_f64"] = {"ms": t_s, "ns_per_site": t_s * 1e6 / V, "bound": "alu", "peak_TFLOPs": fp64_peak,
                                      "flop_per_site_definition": flop_def, "flop_per_site_executed": flop_exec,
                                      "TFLOPs_definition": flop_def * V / (t_s * 1e-3) / 1e12,
                                      "TFLOPs_executed": flop_exec * V / (t_s * 1e-3) / 1e12,
                                      "frac": flop_exec * V / (t_s * 1e-3) / 1e12 / fp64_peak,
                                      "frac_by_definition_count": flop_def * V / (t_s * 1e-3) / 1e12 / fp64_peak,
                                      "variant": variant,
                                      "note": "2 plaquette + 6 rectangle paths per nu, c0 = 5/3, c1 = -1/12; frac = EXECUTED "
                                              "flops / measured FP64 peak"}
        if variant == 2:
            gbs = STAPLES2_BYTES_PER_SITE * V / (t_s * 1e-3) / 1e9
            extra["gauge_staples_f64"].update({
                "hbm_bytes_per_site_two_pass": STAPLES2_BYTES_PER_SITE, "hbm_GBs": gbs, "hbm_frac": gbs / peak,
                "note2": "variant 2 trades FP64 work for HBM traffic (39 instead of 66 / 84 products per link, 24 stored "
                         "3-link staples per site): both fractions are reported; time per site is the figure of merit"})
        # the one-pass kernel (variant 1: 66 products per link, no workspace) beside it: the FP64-bound alternative
        lat.set_option("staples_variant", 1)
        t_1 = timed_loop(torch, lambda: lat.gauge_staples(links, out=sbuf), 10, 3, 1, D, device) / 10
        lat.set_option("staples_variant", 2)
        f1 = 4 * STAPLES_EXEC_FLOP_PER_LINK[1]
        extra["gauge_staples_f64_one_pass"] = {"ms": t_1, "ns_per_site": t_1 * 1e6 / V, "bound": "alu", "variant": 1,
                                               "flop_per_site_executed": f1, "TFLOPs_executed": f1 * V / (t_1 * 1e-3) / 1e12,
                                               "frac": f1 * V / (t_1 * 1e-3) / 1e12 / fp64_peak,
                                               "frac_by_definition_count": flop_def * V / (t_1 * 1e-3) / 1e12 / fp64_peak}
        del sbuf
        cfg2 = cfg4 = ladder = None
        if not args.quick:
            # ---- BASELINE.json configs[1]: CG at 16^4 to tolerance (L2-resident: launch-latency bound) ----
            d2 = (16, 16, 16, 16)
            r2 = np.random.default_rng(2)
            U2 = gen.smooth_links(d2, 0.3, r2)
            b2 = gen.gaussian_half_spinor(d2, r2)
            l2 = L.Lattice(d2, device=local_rank)
            extra["cg_16x16x16x16"] = dict(
                solve_to_tolerance(torch, l2, l2.pack_links(U2), l2.pack_spinor(b2, L.EVEN), [0.0], 0.01, 1e-10, peak),
                note="BASELINE.json configs[1]: m = 0.01, eps 0.3, seed 2, tol 1e-10; links 37.7 MB fit L2: not an HBM figure")
            l2.close()
            cfg2 = (d2, U2, b2, 0.01, 1e-10)
            # ---- BASELINE.json configs[3], first lattice: 24^3 x 48 to tolerance ---------------------------
            d4 = (24, 24, 24, 48)
            r4 = np.random.default_rng(4)
            U4 = gen.smooth_links(d4, 0.3, r4)
            b4 = gen.gaussian_half_spinor(d4, r4)
            l4 = L.Lattice(d4, device=local_rank)
            extra["multishift_24x24x24x48"] = dict(
                solve_to_tolerance(torch, l4, l4.pack_links(U4), l4.pack_spinor(b4, L.EVEN), shifts, 0.0025, 1e-10, peak, MS8_BYTES),
                note="BASELINE.json configs[3]: 8 shifts 1e-4..1, m = 0.0025, eps 0.3, seed 4, tol 1e-10 per shift")
            l4.close()
            cfg4 = (d4, U4, b4, 0.0025, 1e-10, shifts)
            # ---- BASELINE.json configs[4]: large-volume Dslash, fp64 and fp32 (eps 0.5, seed 5) ------------
            d48, d64 = (48, 48, 48, 48), (64, 64, 64, 16)
            r5 = np.random.default_rng(5)
            U48 = gen.smooth_links(d48, 0.5, r5)
            for dims_l, name in ((d48, "48x48x48x48"), (d64, "64x64x64x16")):
                Vl = gen.volume(dims_l)
                # the generator draws link by link in canonical order, so the first Vl sites of the 48^4 field ARE
                # the field smooth_links(dims_l, 0.5, seed 5) would produce (bit for bit)
                Ul = U48[:Vl]
                rs = np.random.default_rng(55)
                ie, io = gen.gaussian_half_spinor(dims_l, rs), gen.gaussian_half_spinor(dims_l, rs)
                for prec, pname in ((L.F64, "f64"), (L.F32, "f32")):
                    for recon, rn in ((L.RECON_18, 18), (L.RECON_12, 12)):
                        extra[f"dslash_{name}_{pname}_{rn}real"] = dslash_rate(torch, L, D, gen, dims_l, Ul, ie, io, prec, recon,
                                                                             peak, device, n=60)
                    # config 5's CG leg: time per iteration at a fixed iteration count (m = 0.01; eps 0.5 needs thousands
                    # of iterations to converge), 18-real links
                    lc = L.Lattice(dims_l, prec=prec, device=local_rank)
                    ms_it = solver_iter_rate(torch, lc, L, lc.pack_links(Ul), lc.pack_spinor(ie, L.EVEN), [0.0], 0.01, n_lo=12, n_hi=60)
                    by = CG_BYTES if prec == L.F64 else CG_BYTES // 2
                    extra[f"cg_{name}_{pname}"] = {"us_per_iter": ms_it * 1e3, "iter_per_s": 1e3 / ms_it, "bytes_per_site_iter": by,
                                                   "GBs": by * (Vl // 2) / (ms_it * 1e-3) / 1e9,
                                                   "frac": by * (Vl // 2) / (ms_it * 1e-3) / 1e9 / peak}
                    lc.close()
            # ---- BASELINE.json configs[4] "versus volume": the L2 -> HBM transition on the paper's Table-3 lattices
            #      (32^2 x 8 x 32, 32^3 x 8, 24^4, 32^4, 32^3 x 36) and a few cubes around them; fp64 18-real
            ladder = []
            for dims_l in ((16, 16, 16, 16), (20, 20, 20, 20), (24, 24, 24, 24), (32, 32, 8, 32), (32, 32, 32, 8),
                           (32, 32, 32, 36), (40, 40, 40, 40)):
                Vl = gen.volume(dims_l)
                Ul = U48[:Vl]
                rs = np.random.default_rng(56)
                ie, io = gen.gaussian_half_spinor(dims_l, rs), gen.gaussian_half_spinor(dims_l, rs)
                dr = dslash_rate(torch, L, D, gen, dims_l, Ul, ie, io, L.F64, L.RECON_18, peak, device, n=100)
                lc = L.Lattice(dims_l, device=local_rank)
                ms_it = solver_iter_rate(torch, lc, L, lc.pack_links(Ul), lc.pack_spinor(ie, L.EVEN), [0.0], 0.01, n_lo=24, n_hi=120)
                lc.close()
                link_mb = Vl * 4 * 144 / 1e6
                ladder.append({"dims": list(dims_l), "links_MB": round(link_mb, 1),
                               "regime": "L2" if link_mb + 6 * Vl // 2 * 48 / 1e6 < 126 else "HBM",
                               "dslash_ns_per_site": round(dr["ns_per_site"], 4), "dslash_frac": round(dr["frac"], 3),
                               "cg_us_per_iter": round(ms_it * 1e3, 2),
                               "cg_frac": round(CG_BYTES * (Vl // 2) / (ms_it * 1e-3) / 1e9 / peak, 3)})
            del U48
        # ---- CPU oracle beside it -------------------------------------------------------------
        psi = np.zeros((V, 3), dtype=np.complex128)
        psi[gen.half_index_of_parity(DIMS, 0)] = in_e
        psi[gen.half_index_of_parity(DIMS, 1)] = in_o
        cpu_ns, reps, cores = cpu_oracle_dslash(U, psi, min_seconds=args.cpu_seconds)
        cpu = {"value": cpu_ns, "unit": "ns/site", "cores": cores, "kind": "oracle",
               "sample": f"{reps} full-lattice applications of oracle_dirac_full at 32^4"}
        parity = check_timed_outputs(np, gen, U, psi, timed_out)
        solver = {k2: {"iter_per_s": extra[k1]["iter_per_s"], "us_per_iter": extra[k1]["us_per_iter"], "frac": extra[k1]["frac"]}
                  for k1, k2 in (("cg_f64", "cg"), ("multishift8_f64", "multishift8"), ("rational8_f64", "rational8"))}
        solver["lattice"] = "32^4 fp64 18-real, all shifts active, per-iteration time by differencing two fixed-length solves"
        s32 = extra["multishift_32x32x32x32"]
        solver["multishift8_to_1e-10"] = {"iters": s32["iters"], "ms": s32["ms"], "max_true_rel_resid": s32["max_true_rel_resid"]}
        for key in ("cg_48x48x48x48_f64", "cg_48x48x48x48_f32", "cg_64x64x64x16_f64", "cg_64x64x64x16_f32"):
            if key in extra:
                solver[key] = {"iter_per_s": extra[key]["iter_per_s"], "frac": extra[key]["frac"]}
        solver["fermion_force8_ms"] = extra["fermion_force8_f64"]["ms"]
        solver["gauge_staples_ns_per_site"] = extra["gauge_staples_f64"]["ns_per_site"]
        if cfg2 is not None:
            cpu["solver"] = cpu_oracle_solvers(gen, cfg2, cfg4, 40)
            cpu["solver"]["note"] = (f"same oracle, same inputs as extra.cg_16x16x16x16 / extra.multishift_24x24x24x48, {cores} threads "
                                     "on the site loop of the operator (reductions and vector updates are the oracle's plain serial loops)")
        line = {
            "metric": "dslash_ns_per_site", "value": ns_site, "unit": "ns/site", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(world),
            "applications_timed": apps, "pairs_per_step": k,
            "GFLOPs": FLOP_PER_SITE * Vh * world / (us_launch * 1e-6) / 1e9,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         # a capture of another build of the kernel's sources is not evidence for this one: null then
                         "traffic": None if traffic["stale"] else traffic["dram_bytes"], "traffic_source": traffic.get("source"),
                         "traffic_commit": traffic.get("commit"), "traffic_source_hash": traffic.get("source_hash"),
                         "traffic_stale": traffic["stale"],
                         "frac_by_ncu_traffic": None if traffic["stale"] else traffic["dram_bytes"] / (us_launch * 1e-6) / 1e9 / peak,
                         "peak_source": peak_src, "kernel": kernel,
                         "peak_note": "the peak is a 50 %-write copy; this kernel is 96 % reads, so frac may exceed 1",
                         "bytes_per_launch": BYTES_PER_SITE[("f64", 18)] * Vh, "us_per_launch": us_launch,
                         "frac_of_nominal_8TBs": achieved / 8000.0,
                         "read_rate_GBs": read_gbs, "frac_of_read_rate": achieved / read_gbs,
                         "read_rate_note": "lqcd_measure_hbm_read over the 604 MB link field in this run: 16-byte streaming "
                                           "loads, nothing written -- the attainable rate of a read-only stream"},
            "e2e": {"value": e2e_ms * 1e6 / (e2e_steps * E2E_PAIRS * V * world), "unit": "ns/site", "steps": e2e_steps,
                    "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "api": f"lqcd_dslash_host_vectors_batch, one call of {2 * E2E_PAIRS} applications per step: pinned canonical "
                           "host vectors in and out, uploads / kernels / downloads pipelined on three streams, links resident "
                           "(the operator; uploaded once per configuration, PAPER.md:276)",
                    "one_call_per_application": {"value": ser_ms * 1e6 / (ser_steps * V * world), "unit": "ns/site", "steps": ser_steps,
                                                 "api": "lqcd_dslash_host_vectors x2 per step (upload, compute, download in sequence)"},
                    "cold_links": {"value": cold_ms * 1e6 / (cold_steps * V * world), "unit": "ns/site", "steps": cold_steps,
                                   "h2d_bytes_per_step": 2 * (U.nbytes + in_e.nbytes), "d2h_bytes_per_step": 2 * in_e.nbytes,
                                   "api": "lqcd_dslash_host x2 per step: the canonical link field is uploaded and packed in every call"}},
            "gpu_launches": launches,
            "parity": parity,
            "solver": solver,
            "volume_ladder": ladder,
            "clocks": clocks,
            "cpu_baseline": cpu,
            "extra": extra,
        }
    lat.close()
    D.barrier(world)
    D.finalize(world)
    if line is not None:
        print(json.dumps(line), flush=True)


# flops per LINK each staples variant executes: SU(3) product = 198, scaled add = 36
# executed flops per link: variant 2 = 30 products in pass 2 + 9 (36 per site) in pass 1, and per nu 2 W-sums,
# 2 (c1 T3 + c0 C) combinations of 54 flops and 4 accumulations into S
STAPLES_EXEC_FLOP_PER_LINK = {0: 84 * 198 + 24 * 36, 1: 3 * (22 * 198 + 10 * 36), 2: 39 * 198 + 3 * (6 * 36 + 2 * 54)}
# two-pass staples: HBM bytes per site that the algorithm must move (fp64): pass 1 reads the links (576) and writes 24
# fields (3456); pass 2 reads them and the links and writes the staples (576)
STAPLES2_BYTES_PER_SITE = 576 + 3456 + 3456 + 576 + 576


def slab_strong_leg(torch, L, D, gen, U, rank, local_rank, world, device, plain_us):
    """One 32^4 lattice (the same on every rank: seed SEED) split into `world` x3 slabs, one per GPU, over the
    peer transport (CUDA IPC between the processes): Dslash time per application and 8-shift CG time per iteration,
    max over ranks.  No number here was ever taken on more than one GPU in this project's environment."""
    import numpy as np
    from paper_1701_00426_b200.slab import SlabLattice
    if U is None:
        U = gen.smooth_links(DIMS, EPS, np.random.default_rng(SEED))
    r2 = np.random.default_rng(SEED + 7)
    ie, io = gen.gaussian_half_spinor(DIMS, r2), gen.gaussian_half_spinor(DIMS, r2)
    V = gen.volume(DIMS)
    sl = SlabLattice(DIMS, world, rank, device=local_rank, transport="peer")
    if world > 1:
        sl.connect_ipc()
    links = sl.pack_links(U)
    a, b = sl.pack_spinor(ie, 0), sl.pack_spinor(io, 1)
    oo, oe = sl.new_spinor(), sl.new_spinor()

    def step():
        sl.dslash(1, oo, a, links)
        sl.dslash(0, oe, b, links)
    n = 200
    us = timed_loop(torch, step, n, 10, world, D, device) * 1e3 / (2 * n)
    shifts = gen.rhmc_shifts(8)
    xs = [sl.new_spinor() for _ in shifts]

    def solve(m):
        return ev_ms(torch, lambda: sl.cg_multishift(xs, a, links, 0.0025, shifts, 1e-300, m, raise_on_max_iter=False))[0]
    solve(16)
    D.barrier(world)
    t_lo, t_hi = min(solve(16), solve(16)), min(solve(80), solve(80))
    it_us = D.max_over_ranks((t_hi - t_lo) / 64 * 1e3, world, device)
    graph = sl.lat.get_option("graph_active")
    halo = sl.lat.halo_bytes
    timeouts = sl.lat.get_option("peer_timeouts")
    sl.close()
    if timeouts:
        raise RuntimeError(f"{timeouts} waits for other ranks timed out: the slab timings are void")
    out = {"dims": list(DIMS), "ranks": world, "transport": "peer (lqcd_peer_*: P2P stores into the neighbours' landing "
           "buffers, in-kernel flag waits, dot products gathered by the consumer kernels)",
           "dslash_us": us, "dslash_ns_per_site": us * 1e3 / (V // 2), "dslash_GBs_aggregate": 1248 * (V // 2) / us / 1e3,
           "multishift8_us_per_iter": it_us, "multishift8_iter_per_s": 1e6 / it_us, "chunk_graph": graph,
           "halo_bytes_per_face": halo, "faces_per_dslash": 2, "allreduces_per_iteration": 2, "scaling": "strong"}
    if plain_us is not None:
        out["dslash_overhead_us_vs_plain_context"] = us - plain_us
    return out


def check_timed_outputs(np, gen, U, psi, timed_out, n_random=200, tol=1e-12):
    """"last outputs vs oracle".  The vectors the LAST timed applications wrote (D_oe in_e on
    the odd sites, D_eo in_o on the even sites) against oracle_dirac_site, one site at a time: the 16 corners, 20 random
    sites in each x3 boundary slice, n_random random sites.  Outside every timed region; rank 0 only."""
    import oracle
    n0, n1, n2, n3 = DIMS
    samp = np.random.default_rng(99)
    picks = [(a * (n0 - 1), b * (n1 - 1), c * (n2 - 1), d * (n3 - 1)) for a in (0, 1) for b in (0, 1) for c in (0, 1) for d in (0, 1)]
    for x3 in (0, n3 - 1):
        picks += [(int(samp.integers(n0)), int(samp.integers(n1)), int(samp.integers(n2)), x3) for _ in range(20)]
    picks += [tuple(int(samp.integers(n)) for n in DIMS) for _ in range(n_random)]
    worst = 0.0
    for x in picks:
        lex = x[0] + n0 * (x[1] + n1 * (x[2] + n2 * x[3]))
        want = oracle.dirac_site(DIMS, U, psi, x)
        got = timed_out[sum(x) % 2][lex // 2]
        worst = max(worst, float(np.abs(got - want).max() / np.abs(want).max()))
    return {"max_rel_err": worst, "sites": len(picks), "tol": tol, "ok": bool(worst < tol),
            "against": "oracle_dirac_site on the outputs of the last timed D_oe and D_eo applications"}


def dslash_rate(torch, L, D, gen, dims, U, in_e, in_o, prec, recon, peak, device, n=100, theta=None, bf_format=0,
                bytes_per_site=None):
    """ns/site, GB/s, fraction of the copy peak of one Dslash variant (alternating parities, fixed inputs)."""
    pname, rn = ("f64" if prec == L.F64 else "f32"), (18 if recon == L.RECON_18 else 12)
    Vh = gen.volume(dims) // 2
    lt = L.Lattice(dims, prec=prec, recon=recon, device=device.index, options={"backfield_format": bf_format})
    lk = lt.pack_links(U)
    if theta is not None:
        lt.set_backfield(lt.pack_backfield(theta))
    a, b_, o1, o2 = lt.pack_spinor(in_e, 0), lt.pack_spinor(in_o, 1), lt.new_spinor(), lt.new_spinor()

    def st():
        lt.dslash(L.ODD, o1, a, lk)
        lt.dslash(L.EVEN, o2, b_, lk)
    t = timed_loop(torch, st, n, 5, 1, D, device)
    us = t * 1e3 / (2 * n)
    gbs = (bytes_per_site or BYTES_PER_SITE[(pname, rn)]) * Vh / (us * 1e-6) / 1e9
    lt.close()
    return {"ns_per_site": us * 1e3 / Vh, "us_per_launch": us, "GBs": gbs, "frac": gbs / peak,
            "GFLOPs": FLOP_PER_SITE * Vh / (us * 1e-6) / 1e9, "dims": list(dims)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=10.0, dest="cpu_seconds")
    ap.add_argument("--quick", action="store_true",
                    help="skip the extras that need other lattices (configs[1], [3] at 24^3 x 48, [4]) and their CPU legs")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
