"""Writes tests/golden/config1_oracle.json from the CPU oracle and the seeded input generator only (no CUDA path).

    python tests/golden/make_golden.py

BASELINE.json config 1: 4^4, fp64, kappa = 0.12, links exp(i*0.3*H), periodic x,y,z / antiperiodic t, Gaussian source.
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)


def compute():
    from oracle import bqo
    from paper_2111_04457_b200 import inputs
    L, kappa = (4, 4, 4, 4), 0.12
    seed = inputs.BASE_SEED + 1
    U = inputs.gauge(L, seed, 0.3)
    b = inputs.spinor(L, seed)
    d = bqo.dirac_apply(U, b, kappa)
    dd = bqo.dirac_apply_dag(U, b, kappa)
    A = bqo.clover_build(U, 1.0, kappa)
    dc = bqo.dirac_apply(U, b, kappa, A=A)
    x, info = bqo.bicgstab(U, b, kappa, tol=1e-12)
    plaq = np.mean([np.einsum("...ab,...bc,...dc,...ad->...", U[..., mu, :, :], np.roll(U[..., nu, :, :], -1, axis=3 - mu),
                              np.roll(U[..., mu, :, :], -1, axis=3 - nu).conj(), U[..., nu, :, :].conj()).real.mean() / 3
                    for mu in range(4) for nu in range(mu + 1, 4)])
    c = lambda z: [float(np.real(z)), float(np.imag(z))]
    return {
        "_what": "BASELINE.json config 1 (4^4, kappa 0.12, eps 0.3, seed 21110445701): oracle/ + seeded inputs only; a drift guard, not a pin",
        "U[0,0,0,0,mu=0][0][0]": c(U[0, 0, 0, 0, 0, 0, 0]),
        "b[0,0,0,0][0][0]": c(b[0, 0, 0, 0, 0, 0]),
        "mean_plaquette": float(plaq),
        "norm2_b": float(np.vdot(b, b).real),
        "norm2_Db": float(np.vdot(d, d).real),
        "<b,Db>": c(np.vdot(b, d)),
        "<b,Ddag b>": c(np.vdot(b, dd)),
        "norm2_Dclover_b_csw1": float(np.vdot(dc, dc).real),
        "Db[3,2,1,0][2][1]": c(d[3, 2, 1, 0, 2, 1]),
        "norm2_x": float(np.vdot(x, x).real),
        "bicgstab_iters_full_D_tol1e-12": int(info["iters"]),
    }


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_oracle.json")
    with open(out, "w") as f:
        json.dump(compute(), f, indent=1)
    print("wrote", out)
