"""Writes tests/golden/oracle_regression.json from oracle/ only (never from the CUDA path)."""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import lqcd_inputs as gen  # noqa: E402
import oracle  # noqa: E402


def compute():
    out = {}
    dims = (4, 4, 4, 4)
    rng = np.random.default_rng(1)
    U = gen.haar_like_links(dims, rng)
    psi = gen.gaussian_spinor(dims, rng)
    d = oracle.dirac_full(dims, U, psi)
    out["config1_4x4_dirac_norm2"] = float(np.vdot(d, d).real)
    out["config1_4x4_dirac_site0"] = [[float(z.real), float(z.imag)] for z in d[0]]
    dims = (8, 8, 8, 8)
    rng = np.random.default_rng(2)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    res = oracle.cg(dims, U, 0.01, b, 1e-10, 20000, hist_len=3)
    out["cg_8x4_m0.01_iters"] = int(res["iters"])
    out["cg_8x4_alpha0"] = float(res["alpha"][0])
    ms = oracle.cg_multishift(dims, U, 0.0025, gen.rhmc_shifts(8), b, 1e-10, 20000)
    out["multishift_8x4_iters"] = int(ms["iters"])
    out["multishift_8x4_conv_iter"] = [int(c) for c in ms["conv_iter"]]
    # rows added from SURVEY.md section 8(f): rational function, fermion force, gauge staples
    dims = (4, 4, 4, 4)
    rng = np.random.default_rng(7)
    U = gen.smooth_links(dims, 0.3, rng)
    b = gen.gaussian_half_spinor(dims, rng)
    shifts, c = gen.rhmc_shifts(4), np.array([0.5, -1.25, 2.0, 0.125])
    ra = oracle.rational_apply(dims, U, 0.05, shifts, 0.35, c, b, 1e-12, 5000)
    out["rational_4x4_norm2"] = float(np.vdot(ra["y"], ra["y"]).real)
    out["rational_4x4_iters"] = int(ra["iters"])
    xs = oracle.cg_multishift(dims, U, 0.05, shifts, b, 1e-12, 5000)["x"]
    F = oracle.fermion_force(dims, U, c, xs)
    out["force_4x4_norm2"] = float(np.vdot(F, F).real)
    out["force_4x4_link0"] = [[float(z.real), float(z.imag)] for z in F[0, 0].reshape(-1)]
    S = oracle.gauge_staples(dims, U)
    out["staples_4x4_norm2"] = float(np.vdot(S, S).real)
    out["staples_4x4_retr_US"] = float(np.real(np.einsum("xmab,xmba->", U, S)))
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.json")
    with open(path, "w") as f:
        json.dump(compute(), f, indent=1)
    print(open(path).read())
