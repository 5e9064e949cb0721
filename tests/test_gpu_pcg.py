"""Parity of the preconditioned CG path (fcg_set_preconditioner / fcg_pcg_solve) with the
oracle's oracle_pcg on the same seeded inputs, through the C ABI.  Same protocol and tolerances as test_gpu_parity.py:
status equal, iteration count within +-2, u within 1e-9 (fp64) / 1e-4 (fp32) at equal iteration count."""
import os

import numpy as np
import pytest
import torch

from oracle import api as orc
from paper_1305_3625_b200 import inputs
from test_gpu_parity import B, TOL_CG, dev, handle, rel  # noqa: F401  (B is a fixture)

pytestmark = pytest.mark.gpu


def pcg_handle(B, w, kbar, **opts):
    dt = w.dtype.type
    h = handle(B, w.L, dt, w.s, **opts)
    h.fcg_set_preconditioner(dev(w.s, dt), kbar)
    return h


def pcg_parity(B, w, **opts):
    dt = w.dtype.type
    kbar = inputs.precond_kbar(w.k)
    h = pcg_handle(B, w, kbar, **opts)
    ref = orc.pcg(w.s, w.k, w.f, w.u0, kbar, w.tol, w.maxit, history=True)
    kd, fd = dev(w.k), dev(w.f)
    u = dev(w.u0)
    it, rr, st = h.fcg_pcg_solve(kd, fd, u, w.tol, w.maxit)
    assert st == ref["status"]
    assert abs(it - ref["iters"]) <= 2, (it, ref["iters"], ref["hist"][-4:])
    d_nat = rel(u.cpu().numpy(), ref["u"])
    d_pin = d_nat
    if it != ref["iters"] and d_nat > TOL_CG[dt]:
        u2 = dev(w.u0)
        it2, _, _ = h.fcg_pcg_solve(kd, fd, u2, 0.0, ref["iters"])
        assert it2 == ref["iters"]
        d_pin = rel(u2.cpu().numpy(), ref["u"])
    assert min(d_nat, d_pin) <= TOL_CG[dt], (d_nat, d_pin, it, ref["iters"])
    assert rr <= w.tol
    if it <= ref["iters"]:      # against the oracle's residual at the same count, loosely (rounding-sensitive)
        assert abs(rr - ref["hist"][it]) <= 0.5 * ref["hist"][it] + 1e-15, (it, ref["iters"], rr, ref["hist"][it])
    # pinned count, element by element: a few iterations in, where nothing depends on the stopping decision
    npin = min(4, ref["iters"])
    refp = orc.pcg(w.s, w.k, w.f, w.u0, kbar, 0.0, npin, history=True)
    u3 = dev(w.u0)
    it3, rr3, _ = h.fcg_pcg_solve(kd, fd, u3, 0.0, npin)
    assert it3 == npin and rel(u3.cpu().numpy(), refp["u"]) <= TOL_CG[dt] * 0.1
    assert abs(rr3 - refp["hist"][npin]) <= 1e-3 * refp["hist"][npin] + 1e-15
    h.close()
    return it, ref["iters"]


@pytest.mark.parametrize("L", [16, 64, 128, 256, 512, 1024])
@pytest.mark.parametrize("dt", [np.float64, np.float32])
def test_pcg_config2_recipe(B, L, dt):
    it, it_or = pcg_parity(B, inputs.config(2, dt, L=L))
    assert it <= 16                                         # kappa(M^-1 A) <= 2.2 for k in [0.5, 1.5]: L-independent


@pytest.mark.parametrize("cfg,L,dt", [(0, 64, np.float64), (1, 256, np.float64), (1, 512, np.float64), (4, 512, np.float32),
                                      (4, 1024, np.float32)])
def test_pcg_broken_sites(B, cfg, L, dt):
    pcg_parity(B, inputs.config(cfg, dt, L=L))


@pytest.mark.parametrize("L,dt", [(128, np.float64), (512, np.float64), (1024, np.float32)])
def test_pcg_classic_engine_and_loop_modes(B, L, dt):
    """Classic passes (7 launches per iteration) and direct-launch mode give the oracle's answer too; the graph and the
    direct-launch modes of one engine are bit-identical."""
    w = inputs.config(1, dt, L=L)
    pcg_parity(B, w, FCG_OPT_ENGINE=1)
    kbar = inputs.precond_kbar(w.k)
    outs = []
    for opts in (dict(FCG_OPT_FUSED=0), dict(FCG_OPT_FUSED=0, FCG_OPT_LOOP_MODE=1, FCG_OPT_CHUNK=3), dict(FCG_OPT_FUSED=0, FCG_OPT_UNROLL=1)):
        h = pcg_handle(B, w, kbar, **opts)
        u = dev(w.u0)
        r = h.fcg_pcg_solve(dev(w.k), dev(w.f), u, w.tol, w.maxit)
        outs.append((r, u.cpu().numpy().copy()))
        h.close()
    for o in outs[1:]:
        assert o[0] == outs[0][0] and np.array_equal(o[1], outs[0][1])


def test_pcg_exact_preconditioner_one_iteration(B):
    """Uniform k = kbar: M = A, so PCG stops after exactly one iteration (the oracle pin, through the GPU path)."""
    L = 256
    w = inputs.config(2, L=L)
    k = np.full((L, L), 0.75)
    f = inputs.normal_f(L)
    h = handle(B, L, np.float64, w.s)
    h.fcg_set_preconditioner(dev(w.s), 0.75)
    u = dev(w.u0)
    it, rr, st = h.fcg_pcg_solve(dev(k), dev(f), u, 1e-10, 100)
    ref = orc.pcg(w.s, k, f, w.u0, 0.75, 1e-10, 100)
    assert (it, st) == (1, 0) and ref["iters"] == 1
    assert rel(u.cpu().numpy(), ref["u"]) <= 1e-12
    h.close()


def test_pcg_edge_cases(B):
    L = 64
    w = inputs.config(0)
    kbar = inputs.precond_kbar(w.k)
    h = handle(B, L, np.float64, w.s)
    kd, fd = dev(w.k), dev(w.f)
    u = dev(w.u0)
    with pytest.raises(B.FcgError) as ei:                   # preconditioner not set
        h.fcg_pcg_solve(kd, fd, u, 1e-10, 10)
    assert ei.value.status == B.FCG_NO_SPECTRUM
    h.fcg_set_preconditioner(dev(w.s), kbar)
    assert h.fcg_pcg_solve(kd, fd, u, 1e-10, 0) == (0, 1.0, B.FCG_NOT_CONVERGED)
    assert torch.count_nonzero(u) == 0
    it, rr, st = h.fcg_pcg_solve(kd, fd, u, 1e-10, 3)       # maxit reached
    ref = orc.pcg(w.s, w.k, w.f, w.u0, kbar, 1e-10, 3)
    assert (it, st) == (3, B.FCG_NOT_CONVERGED) and rel(u.cpu().numpy(), ref["u"]) <= 1e-12
    u = dev(w.u0)                                            # warm start from the solution: zero iterations
    it, _, st = h.fcg_pcg_solve(kd, fd, u, 1e-10, 1000)
    assert st == 0 and h.fcg_pcg_solve(kd, fd, u, 1e-9, 1000)[::2] == (0, 0)
    u = dev(np.ones((L, L)))                                 # f = 0
    assert h.fcg_pcg_solve(kd, dev(np.zeros((L, L))), u, 1e-10, 10) == (0, 0.0, 0)
    assert torch.count_nonzero(u) == 0
    kneg = np.full((L, L), -50.0)                            # indefinite operator: breakdown, same verdict and count
    ref = orc.pcg(w.s, kneg, w.f, w.u0, kbar, 1e-10, 50)
    u = dev(w.u0)
    it, rr, st = h.fcg_pcg_solve(dev(kneg), fd, u, 1e-10, 50)
    assert ref["status"] == orc.BREAKDOWN and st == B.FCG_BREAKDOWN and it == ref["iters"]
    assert rel(u.cpu().numpy(), ref["u"]) <= 1e-9 or np.linalg.norm(ref["u"]) == 0
    h.fcg_set_spectrum(dev(w.s))                             # a new spectrum invalidates the preconditioner
    with pytest.raises(B.FcgError):
        h.fcg_pcg_solve(kd, fd, u, 1e-10, 10)
    # CG after PCG on the same handle still works (the scalar block's mode flag is reset by every set-up)
    h.fcg_set_preconditioner(dev(w.s), kbar)
    u1 = dev(w.u0); h.fcg_pcg_solve(kd, fd, u1, 1e-10, 100)
    u2 = dev(w.u0); it2, _, st2 = h.fcg_solve(kd, fd, u2, 1e-10, 100)
    assert st2 == 0 and abs(it2 - 28) <= 2 and rel(u1.cpu().numpy(), u2.cpu().numpy()) <= 1e-8
    h.close()


@pytest.mark.parametrize("dt,tolpin", [(np.float64, 1e-10), (np.float32, 1e-5)])
def test_pcg_config2_full_size(B, dt, tolpin):
    """L = 2048 in the configuration bench.py --solver pcg times: pinned count 3 vs the oracle element by element; the
    finished solve satisfies ||f - A_oracle u|| / ||f|| <= 2 tol with one oracle operator application; bitwise repeatable."""
    w = inputs.config(2, dt)
    kbar = inputs.precond_kbar(w.k)
    h = pcg_handle(B, w, kbar)
    kd, fd = dev(w.k), dev(w.f)
    ref = orc.pcg(w.s, w.k, w.f, w.u0, kbar, 0.0, 3, history=True)
    u = dev(w.u0)
    it, rr, _ = h.fcg_pcg_solve(kd, fd, u, 0.0, 3)
    assert it == 3 and rel(u.cpu().numpy(), ref["u"]) <= tolpin
    assert abs(rr - ref["hist"][3]) <= 1e-3 * ref["hist"][3]
    u = dev(w.u0)
    it, rr, st = h.fcg_pcg_solve(kd, fd, u, w.tol, w.maxit)
    assert st == 0 and rr <= w.tol and it <= 16
    uh = u.cpu().numpy()
    true_res = np.linalg.norm((w.f - orc.apply(w.s, w.k, uh)).astype(np.float64)) / np.linalg.norm(w.f.astype(np.float64))
    assert true_res <= 2 * w.tol
    u2 = dev(w.u0)
    assert h.fcg_pcg_solve(kd, fd, u2, w.tol, w.maxit) == (it, rr, st) and torch.equal(u, u2)
    assert h.fcg_last_launch_count() == 8 + 6 * 4 * ((it + 3) // 4)
    h.close()


@pytest.mark.parametrize("cfg,L", [(1, 256), (1, 512), (2, 512), (4, 256)])
def test_pcg_fused_kernel_and_graph_path(B, cfg, L):
    """L = 256, 512: the whole PCG solve is ONE cooperative launch (z in q's shared-memory slot); the graph path
    (FCG_OPT_FUSED = 0) of the same sizes is checked against the oracle too."""
    w = inputs.config(cfg, np.float64, L=L)
    pcg_parity(B, w)
    pcg_parity(B, w, FCG_OPT_FUSED=0)
    h = pcg_handle(B, w, inputs.precond_kbar(w.k))
    u = dev(w.u0)
    r1 = h.fcg_pcg_solve(dev(w.k), dev(w.f), u, w.tol, w.maxit)
    assert h.fcg_last_launch_count() == 1
    u2 = dev(w.u0)
    assert h.fcg_pcg_solve(dev(w.k), dev(w.f), u2, w.tol, w.maxit) == r1 and torch.equal(u, u2)      # bitwise repeatable
    h.close()


@pytest.mark.parametrize("L,steps", [(32, 200), (64, 150), (256, 60)])
def test_pcg_fracture_matches_oracle(B, L, steps):
    """Quasi-static loop with PCG solves vs oracle_pcg_fracture: break indices bit-exact, iteration counts within +-2,
    final k identical, final u within tolerance (graph path for L < 256, the one-launch kernel at L = 256)."""
    w = inputs.config(3, L=L, nsteps=steps)
    ko = w.k.copy(); uo = w.u0.copy()
    ref = orc.pcg_fracture(w.s, ko, w.f, uo, w.t, 1.0, steps, w.tol, w.maxit)
    assert ref["steps"] == steps
    h = pcg_handle(B, w, 1.0)
    k, u = dev(w.k), dev(w.u0)
    index, iters, done, st = h.fcg_pcg_fracture(k, dev(w.f), u, dev(w.t), steps, w.tol, w.maxit)
    assert st == 0 and done == steps
    assert np.array_equal(index, ref["index"]), (np.flatnonzero(index != ref["index"])[:5], ref["gap"].min())
    assert np.abs(iters.astype(int) - ref["iters"].astype(int)).max() <= 2
    assert np.array_equal(k.cpu().numpy(), ko)
    assert rel(u.cpu().numpy(), uo) <= 1e-8
    if L == 256:
        assert h.fcg_last_launch_count() == 1
    h.close()


def test_pcg_fracture_config3_full(B):
    """BASELINE.json configs[3] with PCG solves, all 2000 steps in one launch, against tests/golden/cfg3_pcg_breaks.txt
    (written from oracle/ only): indices bit-exact -- and identical to the CG loop's golden sequence -- counts +-2."""
    rows = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "cfg3_pcg_breaks.txt"), comments="#")
    cg_rows = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "cfg3_breaks.txt"), comments="#")
    gidx, git = rows[:, 1].astype(np.int64), rows[:, 2].astype(np.int64)
    w = inputs.config(3)
    h = pcg_handle(B, w, 1.0)
    k, u = dev(w.k), dev(w.u0)
    index, iters, done, st = h.fcg_pcg_fracture(k, dev(w.f), u, dev(w.t), w.nsteps, w.tol, w.maxit)
    assert st == 0 and done == w.nsteps and h.fcg_last_launch_count() == 1
    assert np.array_equal(index, gidx)
    assert np.array_equal(index, cg_rows[:, 1].astype(np.int64))
    assert np.abs(iters.astype(np.int64) - git).max() <= 2
    assert iters.sum() < 0.5 * cg_rows[:, 2].sum()
    h.close()


@pytest.mark.parametrize("L,use_pcg", [(256, True), (256, False), (64, True)])
def test_fracture_ensemble_begin_end(B, L, use_pcg):
    """Independent samples (different threshold seeds) on three handles / streams driven by one host thread with
    fcg_fracture_begin / _end: every sample equals what the blocking call gives for it (bitwise), and sample 0 equals the oracle."""
    steps, nrep = 40, 3
    w = inputs.config(3, L=L, nsteps=steps)
    ts = [w.t if r == 0 else inputs.thresholds(L, seed=100 + r) for r in range(nrep)]
    reps = []
    for r in range(nrep):
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            h = B.Fcg(L, torch.float64, stream=st)
            s = dev(w.s); h.fcg_set_spectrum(s); h.fcg_set_preconditioner(s, 1.0)
            reps.append((h, dev(w.k), dev(w.f), dev(w.u0), dev(ts[r]), st))
    torch.cuda.synchronize()
    for h, k, f, u, t, st in reps:
        h.fcg_fracture_begin(k, f, u, t, steps, w.tol, w.maxit, use_pcg)
    outs = [h.fcg_fracture_end() for h, *_ in reps]
    for r, (h, k, f, u, t, st) in enumerate(reps):
        index, iters, done, status = outs[r]
        assert status == 0 and done == steps
        k2, u2 = dev(w.k), dev(w.u0)
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            fn = h.fcg_pcg_fracture if use_pcg else h.fcg_fracture
            i2, it2, d2, s2 = fn(k2, dev(w.f), u2, dev(ts[r]), steps, w.tol, w.maxit)
        assert np.array_equal(index, i2) and np.array_equal(iters, it2) and torch.equal(k, k2) and torch.equal(u, u2)
    ko = w.k.copy(); uo = w.u0.copy()
    ref = (orc.pcg_fracture(w.s, ko, w.f, uo, w.t, 1.0, steps, w.tol, w.maxit) if use_pcg
           else orc.fracture(w.s, ko, w.f, uo, w.t, steps, w.tol, w.maxit))
    assert np.array_equal(outs[0][0], ref["index"]) and np.abs(outs[0][1].astype(int) - ref["iters"].astype(int)).max() <= 2
    with pytest.raises(B.FcgError):                          # nothing pending any more
        reps[0][0]._pending = (None, None, None, None, 1); reps[0][0].fcg_fracture_end()
    for h, *_ in reps:
        h.close()
