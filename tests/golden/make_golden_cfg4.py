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
  python tests/golden/make_golden_cfg4.py --indep   writes cfg4_indep.txt instead: the same workload run by a SECOND plain
CPU implementation that shares nothing with the oracle's transform -- textbook CG (Listing 2, same stopping rule and S12
scalars) around scipy.fft.rfft2 / irfft2 in single precision (pocketfft; a library routine, test-time only, like pin P12) --
sampled at the same sites after PIN iterations and at ITS natural stop.  It is not an expected value for the GPU: it
measures how far two correct fp32 implementations drift apart in mid-run at this size (CG in finite precision amplifies
rounding-level differences of the operator exponentially until convergence pulls the iterates back together), which is what
the pinned-count tolerance of tests/test_gpu_parity.py::test_cg_config4_full_size is derived from (reading S19).

Usage: python tests/golden/make_golden_cfg4.py [--indep]   (about 10 minutes on 8 cores; --indep about 5)
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


def independent_cg(w, maxit, tol, snapshots):
    """Listing 2 step by step (same rule as oracle_cg: first crossing of ||r|| <= tol ||f||, recurrence residual, scalars and
    dot products in double) with the operator k o x + irfft2(s o rfft2(x)) by scipy's single-precision pocketfft."""
    import scipy.fft as sf
    L = w.L
    k, f, sh = w.k, w.f, np.ascontiguousarray(w.s[:, : L // 2 + 1])
    dot = lambda a, b: float(np.dot(a.ravel().astype(np.float64), b.ravel().astype(np.float64)))
    A = lambda x: (k * x + sf.irfft2(sf.rfft2(x, workers=-1) * sh, s=(L, L), workers=-1).astype(np.float32)).astype(np.float32)
    u = np.zeros((L, L), np.float32)
    r = (f - A(u)).astype(np.float32); p = r.copy()
    rho = dot(r, r); fn = np.sqrt(dot(f, f)); hist = [np.sqrt(rho) / fn]; snaps = {}
    it = 0
    while it < maxit:
        q = A(p); alpha = rho / dot(p, q)
        u = (u + np.float32(alpha) * p).astype(np.float32); r = (r - np.float32(alpha) * q).astype(np.float32)
        rho_new = dot(r, r); it += 1; hist.append(np.sqrt(rho_new) / fn)
        if it in snapshots:
            snaps[it] = u.copy()
        if np.sqrt(rho_new) <= tol * fn:
            break
        p = (r + np.float32(rho_new / rho) * p).astype(np.float32); rho = rho_new
    return u, it, np.array(hist), snaps


def main_indep():
    w = inputs.config(4)
    idx = sample_sites(w.N)
    t0 = time.time()
    u, it, hist, snaps = independent_cg(w, w.maxit, w.tol, {PIN})
    dt = time.time() - t0
    up, uf = snaps[PIN].ravel(), u.ravel()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg4_indep.txt")
    with open(path, "w") as fh:
        fh.write("# BASELINE.json configs[4] by a second CPU implementation (textbook CG around scipy.fft rfft2/irfft2, float32); NOT an expected "
                 "value: the drift between two correct fp32 implementations; written by tests/golden/make_golden_cfg4.py --indep\n")
        fh.write(f"# iters={it} relres={hist[-1]:.17e} pin={PIN} nsamp={NSAMP} seconds={dt:.1f}\n")
        fh.write("# hist " + " ".join(f"{v:.9e}" for v in hist) + "\n")
        fh.write("# site u_after_pin u_at_stop\n")
        for i in idx:
            fh.write(f"{int(i)} {up[i]:.9e} {uf[i]:.9e}\n")
    print(path, "iters", it, "relres", hist[-1], f"{dt:.1f}s")


if __name__ == "__main__":
    main_indep() if "--indep" in sys.argv else main()
