"""Writes tests/golden/cfg2_f64_drift.txt by calling ONLY oracle/ and a second plain CPU implementation (never the CUDA path).

BASELINE.json configs[2] in fp64 (L = 2048, f = 1, tol 1e-10) stops where CG in double precision runs out of accuracy: the
residual norm is no longer monotone (it doubles and halves over the last ten iterations) and rounding-level differences of the
operator have been amplified to the 1e-9 level in the iterates.  This script measures that with two CPU programs that share
nothing but the inputs -- the oracle (oracle/fcg_oracle.c: radix-2 FFT, Listing 4 as printed) and textbook CG (Listing 2, same
stopping rule) around scipy.fft.rfft2 / irfft2 in double (pocketfft; a library routine, test-time only, like pin P12):
their natural stops, and the relative L2 distance of their iterates at the stops and at equal counts 90 .. 104.
It is NOT an expected value for the GPU; it is the noise floor that reading S20 rests on.
Usage: python tests/golden/make_golden_cfg2_drift.py   (about two minutes on 8 cores)
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import api as orc                      # noqa: E402
from paper_1305_3625_b200 import inputs            # noqa: E402

COUNTS = list(range(90, 105, 2))


def main():
    import scipy.fft as sf
    w = inputs.config(2, np.float64); L = w.L
    k, f, sh = w.k, w.f, np.ascontiguousarray(w.s[:, : L // 2 + 1])
    A = lambda x: k * x + sf.irfft2(sf.rfft2(x, workers=-1) * sh, s=(L, L), workers=-1)
    dot = lambda a, b: float(np.dot(a.ravel(), b.ravel()))
    u = np.zeros((L, L)); r = f - A(u); p = r.copy(); rho = dot(r, r); fn = np.sqrt(dot(f, f)); hist = [np.sqrt(rho) / fn]
    snaps, stop = {}, None
    for it in range(1, max(COUNTS) + 1):
        q = A(p); al = rho / dot(p, q); u = u + al * p; r = r - al * q; rn = dot(r, r); hist.append(np.sqrt(rn) / fn)
        if stop is None and np.sqrt(rn) <= w.tol * fn:
            stop = it; snaps["stop"] = u.copy()
        if it in COUNTS:
            snaps[it] = u.copy()
        p = r + (rn / rho) * p; rho = rn
    rel = lambda a, b: float(np.linalg.norm(a - b) / np.linalg.norm(b))
    o = orc.cg(w.s, w.k, w.f, w.u0, w.tol, w.maxit, history=True)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg2_f64_drift.txt")
    with open(path, "w") as fh:
        fh.write("# BASELINE.json configs[2] fp64: distance between two CPU implementations (oracle vs textbook CG around scipy's double pocketfft); "
                 "NOT an expected value; written by tests/golden/make_golden_cfg2_drift.py\n")
        fh.write(f"# oracle_iters={o['iters']} second_iters={stop} natural_stops_rel_l2={rel(snaps['stop'], o['u']):.6e}\n")
        fh.write("# oracle_hist_tail " + " ".join(f"{v:.6e}" for v in o["hist"][-8:]) + "\n")
        fh.write("# second_hist_96_104 " + " ".join(f"{v:.6e}" for v in hist[96:105]) + "\n")
        fh.write("# count rel_l2_at_equal_count\n")
        for c in COUNTS:
            oc = orc.cg(w.s, w.k, w.f, w.u0, 0.0, c)
            fh.write(f"{c} {rel(snaps[c], oc['u']):.6e}\n")
    print(open(path).read())


if __name__ == "__main__":
    main()
