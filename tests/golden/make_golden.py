"""Writes the stored expected values under tests/golden/ by calling ONLY oracle/ (never the CUDA path).

  cfg3_breaks.txt   BASELINE.json configs[3]: L=256 fp64, 2000 break steps -- per step: break index,
                    CG iterations, relative top-2 gap of the load/threshold ratio (reading S17).
  cfg3_pcg_breaks.txt   the same loop with preconditioned-CG solves (kbar = 1).
Usage: python tests/golden/make_golden.py [nsteps]
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import api as orc                      # noqa: E402
from paper_1305_3625_b200 import inputs            # noqa: E402


def main():
    nsteps = int(sys.argv[1]) if len(sys.argv) > 1 else 2000
    w = inputs.config(3, nsteps=nsteps)
    k = w.k.copy(); u = w.u0.copy()
    t0 = time.time()
    out = orc.fracture(w.s, k, w.f, u, w.t, nsteps, w.tol, w.maxit)
    dt = time.time() - t0
    assert out["steps"] == nsteps
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg3_breaks.txt")
    with open(path, "w") as fh:
        fh.write("# BASELINE.json configs[3]: L=256 fp64, k=1, f=1, t~U[0,1] seed 1, tol 1e-10, warm start; "
                 "written by tests/golden/make_golden.py from oracle/ only\n")
        fh.write(f"# steps={nsteps} total_iters={int(out['iters'].sum())} min_gap={out['gap'].min():.3e} "
                 f"argmin_gap_step={int(out['gap'].argmin())} oracle_seconds={dt:.1f} threads={orc.num_threads()}\n")
        fh.write("# step index iters gap\n")
        for i in range(nsteps):
            fh.write(f"{i} {int(out['index'][i])} {int(out['iters'][i])} {out['gap'][i]:.6e}\n")
    print(path, "total iters", int(out["iters"].sum()), "min gap", out["gap"].min(), f"{dt:.1f}s")

    # the same loop with PCG solves: kbar = 1 (the unbroken stiffness), fixed for all steps
    k = w.k.copy(); u = w.u0.copy()
    t0 = time.time()
    outp = orc.pcg_fracture(w.s, k, w.f, u, w.t, 1.0, nsteps, w.tol, w.maxit)
    dt = time.time() - t0
    assert outp["steps"] == nsteps
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg3_pcg_breaks.txt")
    with open(path, "w") as fh:
        fh.write("# BASELINE.json configs[3] with PCG solves (M = kbar I + C, kbar = 1): L=256 fp64, k=1, f=1, t~U[0,1] seed 1, "
                 "tol 1e-10, warm start; written by tests/golden/make_golden.py from oracle/ only\n")
        fh.write(f"# steps={nsteps} total_iters={int(outp['iters'].sum())} min_gap={outp['gap'].min():.3e} "
                 f"argmin_gap_step={int(outp['gap'].argmin())} same_indices_as_cg_loop={bool(np.array_equal(outp['index'], out['index']))} "
                 f"oracle_seconds={dt:.1f} threads={orc.num_threads()}\n")
        fh.write("# step index iters gap\n")
        for i in range(nsteps):
            fh.write(f"{i} {int(outp['index'][i])} {int(outp['iters'][i])} {outp['gap'][i]:.6e}\n")
    print(path, "total iters", int(outp["iters"].sum()), "same indices", np.array_equal(outp["index"], out["index"]), f"{dt:.1f}s")


if __name__ == "__main__":
    main()
