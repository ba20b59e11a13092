#!/usr/bin/env python
"""Writes tests/golden/gate<N>_oracle_samples.txt: expected values of the forward + adjoint pressure projection of the
headline workload (BASELINE.json configs[3], the channel-gate; default N = 256) computed by the fp64 CPU oracle ALONE.

    python tests/golden/make_gate_golden.py [--config gate|chamber] [--n 256] [--tol 1e-10] [--samples 4096]

It imports only oracle/ (the definition: Jacobi-PCG in fp64, Eq. 4 / L115-124 Eqs. 6-7 with the readings
of DESIGN.md section 3) and the seeded input generators (paper_2405_14903_b200/workloads.py, no method arithmetic).
Nothing of the CUDA path is imported, linked or executed; no value in the output comes from it.

Inputs (the same ones tests/test_gpu_fullsize.py feeds to the library): workloads.config4_params(N), the initial
velocity Uhat = config4_initial_velocity (seed 1004), the gate at time level 3 (config4_solid(P, 3): rotated by
0.15 rad, u_s = omega x (x - c)), Dirichlet p = 1 / 0 on -x / +x, g = dJ/dU^{n+1} ~ N(0, 1) from default_rng(77).
Outputs sampled at `samples` seeded flat indices per array (stored with the values, so the file does not depend on
NumPy's generator staying the same): p, U^{n+1} (u, v, w), y, dJ/dUhat (u, v, w), dJ/dalpha (u), dJ/dU_s (u), plus the
2-norms of the full arrays.  At N = 256 one run is two Jacobi-PCG solves of 16.8 M unknowns (hours on one core).

--config chamber writes chamber<N>_oracle_samples.txt for the chamber-pump shape (BASELINE.json configs[2]):
workloads.config3_params(N), the static chamber with the wall velocity of time level `--step` (default 12 there:
sin(2 pi 12/50) = 0.998), Dirichlet p = 0 on +x, Uhat = 0.05 N(0, 1) from default_rng(1003), g ~ N(0, 1) from
default_rng(78).
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import nf_oracle as orc  # noqa: E402
from paper_2405_14903_b200 import workloads as wl  # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=256)
    ap.add_argument("--tol", type=float, default=1e-10)
    ap.add_argument("--samples", type=int, default=4096)
    ap.add_argument("--config", default="gate", choices=["gate", "chamber"])
    ap.add_argument("--step", type=int, default=-1)
    ap.add_argument("--out", default="")
    args = ap.parse_args()
    n = args.n
    out = args.out or os.path.join(os.path.dirname(os.path.abspath(__file__)), "%s%d_oracle_samples.txt" % (args.config, n))
    if args.config == "gate":
        step = 3 if args.step < 0 else args.step
        P = wl.config4_params(n)
        U0 = wl.config4_initial_velocity(P)
        phi, us = wl.config4_solid(P, step)
        rng = np.random.default_rng(77)
    else:
        step = 12 if args.step < 0 else args.step
        P = wl.config3_params(n)
        phi, us = wl.config3_solid(P, step)
        r0 = np.random.default_rng(1003)
        U0 = [(0.05 * r0.standard_normal(s)).astype(np.float32) for s in wl.face_shapes(n, n, n)]
        rng = np.random.default_rng(78)
    g = [rng.standard_normal(a.shape).astype(np.float32) for a in U0]
    bc = orc.BC(P["bc_types"], P["bc_values"])
    t0 = time.time()
    alpha = orc.face_weights(phi, bc)
    fi, ai = {}, {}
    Un, p = orc.project(U0, alpha, us, P["dx"], P["dt_over_rho"], bc, tol=args.tol, info=fi)
    t1 = time.time()
    sys.stderr.write("forward: %d iterations, relres %.2e, %.0f s\n" % (fi["iters"], fi["relres"], t1 - t0))
    g_uhat, g_alpha, g_us, y = orc.project_adjoint(g, alpha, p, U0, us, P["dx"], P["dt_over_rho"], bc, tol=args.tol,
                                                   info=ai)
    t2 = time.time()
    sys.stderr.write("adjoint: %d iterations, relres %.2e, %.0f s\n" % (ai["iters"], ai["relres"], t2 - t1))
    arrays = [("p", p), ("u", Un[0]), ("v", Un[1]), ("w", Un[2]), ("y", y), ("guhat_u", g_uhat[0]),
              ("guhat_v", g_uhat[1]), ("guhat_w", g_uhat[2]), ("galpha_u", g_alpha[0]), ("gus_u", g_us[0])]
    srng = np.random.default_rng(2405)
    with open(out, "w") as f:
        f.write("# fp64 oracle samples of the %s projection (forward + adjoint); written by\n"
                % ("channel-gate" if args.config == "gate" else "chamber-pump"))
        f.write("#   python tests/golden/make_gate_golden.py%s --n %d --tol %g --samples %d --step %d\n"
                % ("" if args.config == "gate" else " --config chamber", n, args.tol, args.samples, step))
        f.write("# which imports only oracle/nf_oracle.py and paper_2405_14903_b200/workloads.py (no CUDA path).\n")
        f.write("# Definition followed: A P = b (PAPER.md:L103 Eq. 4), U = Uhat - c G P (L107 Eq. 5), A y = -c G^T M g\n")
        f.write("# (L115-124 Eqs. 6-7), dJ/dalpha and dJ/dU_s in the derived forms R9 / R10 (L134-139 Eq. 9).\n")
        f.write("# oracle solves: forward %d iterations (true relres %.3e), adjoint %d iterations (true relres %.3e)\n"
                % (fi["iters"], fi["relres"], ai["iters"], ai["relres"]))
        f.write("meta n %d tol %.3e step %d samples %d\n" % (n, args.tol, step, args.samples))
        for name, a in arrays:
            a = np.asarray(a, dtype=np.float64)
            f.write("norm %s %.17e\n" % (name, float(np.linalg.norm(a))))
        for name, a in arrays:
            a = np.asarray(a, dtype=np.float64).ravel()
            idx = np.sort(srng.choice(a.size, size=min(args.samples, a.size), replace=False))
            f.write("array %s %d\n" % (name, idx.size))
            for i in idx:
                f.write("%d %.17e\n" % (int(i), a[i]))
    sys.stderr.write("wrote %s (%.0f s)\n" % (out, time.time() - t0))


if __name__ == "__main__":
    main()
