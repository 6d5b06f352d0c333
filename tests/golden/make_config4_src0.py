#!/usr/bin/env python
"""Writes tests/golden/config4_src0_oracle.txt: the ORACLE's full solve of source 0 of
BASELINE.json config 4 (32^4 complex64, m = 0.01, g = 1.5, sigma = 0.5, seed 4, tol 1e-6)
with its complex64 + reliable-update loop O4' (oracle/wz_oracle.cpp orc_cg_c64ru_shift;
DESIGN.md reading G9), as SURVEY.md 8(d) "Oracle timed beside it" asks: run once, keep the
iteration count, the number of reliable updates and the residual history.

Calls only oracle/ and the seeded input generator.  Takes about an hour on 8 cores.

    python tests/golden/make_config4_src0.py [--threads N] [--max-iter K] [--out PATH]
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--max-iter", type=int, default=30000)
    ap.add_argument("--config", default="4")
    ap.add_argument("--source", type=int, default=0)
    ap.add_argument("--every", type=int, default=100)
    ap.add_argument("--out", default=os.path.join(HERE, "config4_src0_oracle.txt"))
    args = ap.parse_args()

    from oracle import wz_oracle as orc
    from paper_1005_3276_b200 import inputs

    key = int(args.config) if args.config.isdigit() else args.config
    cfg = inputs.CONFIGS[key]
    dims = cfg["dims"]
    npdt = np.complex64 if cfg["dtype"] == "c64" else np.complex128
    phi = inputs.make_phi(cfg["seed"], dims, cfg["sigma"], npdt).astype(np.complex128)
    b = inputs.make_source(cfg["seed"], args.source, dims, npdt).astype(np.complex128)
    threads = orc.set_threads(args.threads)
    t0 = time.time()
    fn = orc.cg_c64ru if cfg["dtype"] == "c64" else orc.cg
    _, info = fn(phi, b, cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], args.max_iter)
    dt = time.time() - t0
    with open(args.out, "w") as f:
        f.write("# oracle (%s) full solve of config %s source %d: %s lattice, m=%g g=%g rho=%g sigma_phi=%g seed=%d tol=%g\n"
                % ("O4' complex64 + reliable updates, delta = 0.1" if cfg["dtype"] == "c64" else "O4 complex128",
                   args.config, args.source, "x".join(map(str, dims)), cfg["m"], cfg["g"], cfg["rho"], cfg["sigma"],
                   cfg["seed"], cfg["tol"]))
        f.write("# written by tests/golden/make_config4_src0.py (calls only oracle/); SURVEY.md 8(d)\n")
        f.write("# wall time %.0f s on %d OpenMP threads\n" % (dt, threads))
        f.write("iterations %d\n" % info.iterations)
        f.write("reliable_updates %d\n" % info.reliable_updates)
        f.write("converged %d\n" % int(info.converged))
        f.write("rel_residual_true %.6e\n" % info.rel_residual_true)
        f.write("seconds %.1f\n" % dt)
        f.write("threads %d\n" % threads)
        f.write("# relative residual ||r_k|| / ||b|| (the recomputed one where a reliable update happened) every %d iterations\n"
                % args.every)
        for k in range(0, info.iterations + 1, args.every):
            f.write("history %d %.6e\n" % (k, info.history[k]))
        if info.iterations % args.every:
            f.write("history %d %.6e\n" % (info.iterations, info.history[info.iterations]))
    print("wrote", args.out, "iterations", info.iterations, "seconds %.0f" % dt)


if __name__ == "__main__":
    main()
