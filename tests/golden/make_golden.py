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
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.json")
    with open(path, "w") as f:
        json.dump(compute(), f, indent=1)
    print(open(path).read())
