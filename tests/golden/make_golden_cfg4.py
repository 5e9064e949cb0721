"""Writes tests/golden/cfg4_oracle.txt by calling ONLY oracle/ (never the CUDA path).

BASELINE.json configs[4]: L = 8192 fp32, k ~ U[0.5,1.5] with a seeded 5 % of sites at 0, f ~ N(1, 0.1), u0 = 0,
tol 1e-5, maxit 2000.  The oracle's full solve takes minutes, so its results are stored ("Next round" 1(b)):

  * the oracle's iteration count, status and relative residual at the stop;
  * its whole residual history (one value per iteration: the classification of a count mismatch needs the
    values around the stop, SURVEY.md 8(c) P14 risk note);
  * u at NSAMP seeded sample sites after PIN iterations (tol = 0, maxit = PIN; maxit = 20) and at the stop,
    plus the fp64-accumulated 2-norms of both whole vectors.

Sample sites: numpy.random.default_rng(6).choice(N, NSAMP, replace=False), sorted -- half of them forced onto
broken sites' neighbours is NOT done: the draw is plain uniform, so ~5 % of the samples are broken sites.
Usage: python tests/golden/make_golden_cfg4.py   (about 10 minutes on 8 cores)
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import api as orc                      # noqa: E402
from paper_1305_3625_b200 import inputs            # noqa: E402

NSAMP, PIN, SEED_SAMPLE = 4096, 20, 6


def sample_sites(N: int) -> np.ndarray:
    return np.sort(np.random.default_rng(SEED_SAMPLE).choice(N, NSAMP, replace=False))


def main():
    w = inputs.config(4)
    idx = sample_sites(w.N)
    t0 = time.time()
    pin = orc.cg(w.s, w.k, w.f, w.u0, 0.0, PIN, history=True)
    t1 = time.time()
    full = orc.cg(w.s, w.k, w.f, w.u0, w.tol, w.maxit, history=True)
    t2 = time.time()
    assert pin["iters"] == PIN and full["status"] == orc.OK
    assert np.array_equal(pin["hist"], full["hist"][: PIN + 1])       # the same run, cut short
    up, uf = pin["u"].ravel(), full["u"].ravel()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg4_oracle.txt")
    with open(path, "w") as fh:
        fh.write("# BASELINE.json configs[4]: L=8192 fp32, k~U[0.5,1.5] seed 0 with N//20 sites broken (seed 2), f~N(1,0.1) seed 3, "
                 "u0=0, tol 1e-5, maxit 2000; written by tests/golden/make_golden_cfg4.py from oracle/ only\n")
        fh.write(f"# iters={full['iters']} status={full['status']} relres={full['relres']:.17e} pin={PIN} nsamp={NSAMP} "
                 f"norm_u_pin={np.linalg.norm(up.astype(np.float64)):.17e} norm_u_stop={np.linalg.norm(uf.astype(np.float64)):.17e} "
                 f"oracle_seconds_pin={t1 - t0:.1f} oracle_seconds_full={t2 - t1:.1f} threads={orc.num_threads()}\n")
        fh.write("# hist " + " ".join(f"{v:.9e}" for v in full["hist"]) + "\n")
        fh.write("# site u_after_pin u_at_stop   (fp32 values printed with 9 significant digits: exact round trip)\n")
        for i in idx:
            fh.write(f"{int(i)} {up[i]:.9e} {uf[i]:.9e}\n")
    print(path, "iters", full["iters"], "relres", full["relres"], f"{t2 - t0:.1f}s")
    print("history around the stop:", full["hist"][-8:])


if __name__ == "__main__":
    main()
