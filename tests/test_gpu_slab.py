"""Slab-decomposed CG on the GPU: G logical ranks on one device, each with its
own handle and its own rows of every vector, the exchanges as device copies (slab.LocalComm).  Same parity protocol as
fcg_solve (tests/test_gpu_parity.py): status equal, count within +-2 of the ORACLE, u element by element at the natural stop or
at the oracle's count; plus agreement with the undecomposed library solve in the same textbook order."""
import numpy as np
import pytest
import torch

from oracle import api as orc
from paper_1305_3625_b200 import inputs

pytestmark = pytest.mark.gpu
TDT = {np.float64: torch.float64, np.float32: torch.float32}
TOL_CG = {np.float64: 1e-9, np.float32: 1e-4}


@pytest.fixture(scope="module")
def B():
    from paper_1305_3625_b200 import binding
    assert torch.cuda.is_available()
    binding.lib()
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel(a, b):
    a = np.asarray(a, np.float64).ravel(); b = np.asarray(b, np.float64).ravel()
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def slab_run(w, G, tol, maxit, u0=None, peers=False, spectral=False, graph=None):
    from paper_1305_3625_b200 import slab
    dt = w.dtype.type
    sd = dev(w.s)
    ranks = [slab.SlabRank(w.L, TDT[dt], G, g, sd) for g in range(G)]
    if peers:
        slab.connect_peers_local(ranks)
    k = [dev(w.k[r.rows]) for r in ranks]; f = [dev(w.f[r.rows]) for r in ranks]
    u = [dev((w.u0 if u0 is None else u0)[r.rows]) for r in ranks]
    it, rr, st = slab.slab_solve(ranks, slab.LocalComm(), k, f, u, tol, maxit, spectral=spectral, graph=graph)
    out = np.concatenate([x.cpu().numpy() for x in u], axis=0)
    for r in ranks:
        r.close()
    return it, rr, st, out


@pytest.mark.parametrize("cfg,L,dt", [(1, 256, np.float64), (2, 512, np.float64), (1, 1024, np.float64), (4, 1024, np.float32),
                                      (2, 2048, np.float32)])
@pytest.mark.parametrize("G", [1, 2, 4])
def test_slab_cg_matches_oracle(B, cfg, L, dt, G):
    w = inputs.config(cfg, dt, L=L)
    ref = orc.cg(w.s, w.k, w.f, w.u0, w.tol, w.maxit, history=True)
    it, rr, st, u = slab_run(w, G, w.tol, w.maxit)
    assert st == ref["status"] and abs(it - ref["iters"]) <= 2, (it, ref["iters"])
    d = rel(u, ref["u"])
    if it != ref["iters"] and d > TOL_CG[dt]:
        it2, _, _, u = slab_run(w, G, 0.0, ref["iters"])
        assert it2 == ref["iters"]
        d = rel(u, ref["u"])
    assert d <= TOL_CG[dt], (d, it, ref["iters"])
    assert rr <= w.tol
    # pinned count a few iterations in, where nothing depends on the stopping decision: a tenth of the tolerance
    refp = orc.cg(w.s, w.k, w.f, w.u0, 0.0, 5, history=True)
    itp, rrp, _, up = slab_run(w, G, 0.0, 5)
    assert itp == 5 and rel(up, refp["u"]) <= 0.1 * TOL_CG[dt]
    assert abs(rrp - refp["hist"][5]) <= 1e-3 * refp["hist"][5]


def test_slab_cg_equals_undecomposed_textbook_order(B):
    """The undecomposed library solve in the same textbook order (four launches per iteration) and the slab solve with any G do
    the same arithmetic per element; only the order of the partial sums differs, so the iterates agree to rounding."""
    w = inputs.config(1, np.float64, L=512)
    h = B.Fcg(w.L, torch.float64)
    h.fcg_set_option(B.FCG_OPT_FUSED, 0); h.fcg_set_option(B.FCG_OPT_SPECTRAL_ALPHA, 0)
    h.fcg_set_spectrum(dev(w.s))
    u = dev(w.u0)
    it0, rr0, st0 = h.fcg_solve(dev(w.k), dev(w.f), u, 0.0, 30)
    u0 = u.cpu().numpy()
    h.close()
    for G in (1, 2, 8):
        it, rr, st, ug = slab_run(w, G, 0.0, 30)
        assert (it, st) == (it0, st0) and rel(ug, u0) <= 1e-12 and abs(rr - rr0) <= 1e-9 * rr0


def test_slab_edge_cases(B):
    from paper_1305_3625_b200 import slab
    w = inputs.config(0, np.float64, L=256)
    # warm start from the solution: zero iterations; maxit = 0; f = 0
    it, rr, st, u = slab_run(w, 2, w.tol, w.maxit)
    assert st == 0
    it2, rr2, st2, _ = slab_run(w, 2, 10 * w.tol, w.maxit, u0=u)
    assert (it2, st2) == (0, 0)
    it3, _, st3, u3 = slab_run(w, 4, w.tol, 0)
    assert (it3, st3) == (0, B.FCG_NOT_CONVERGED) and not u3.any()
    w.f[:] = 0
    it4, rr4, st4, u4 = slab_run(w, 2, w.tol, w.maxit, u0=np.ones_like(w.u0))
    assert (it4, rr4, st4) == (0, 0.0, 0) and not u4.any()
    # a split that does not divide the column blocks is refused; so is a slab call on an unconfigured handle
    with pytest.raises(B.FcgError):
        slab.SlabRank(256, torch.float64, 3, 0, dev(w.s))
    h = B.Fcg(256, torch.float64)
    with pytest.raises(B.FcgError):
        h.fcg_slab_cols()
    h.close()


def cfg2_drift():
    """tests/golden/cfg2_f64_drift.txt (make_golden_cfg2_drift.py, CPU only): how far two correct CPU implementations are apart at
    equal iteration count near the stop of configs[2] fp64 -- reading S20 of DESIGN.md.  {count: rel. L2 distance}."""
    import os
    tab = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "cfg2_f64_drift.txt"), comments="#")
    return {int(c): float(d) for c, d in tab}


@pytest.mark.parametrize("dt", [np.float64, np.float32])
def test_slab_cg_full_size_config2(B, dt):
    """configs[2] at L = 2048 over four logical ranks: the whole solve against the oracle's own.  Same protocol as fcg_solve: count
    within 2, u to north_star's tolerance at the natural stop or at the oracle's count.  Reading S20: in fp64 this config stops
    where CG runs out of accuracy, and two correct CPU implementations (the oracle and a second one, stored by
    tests/golden/make_golden_cfg2_drift.py) are 1.2e-9 .. 5.9e-9 apart at EQUAL count over the last 15 iterations (1.9e-9 at the
    oracle's stop, 6.6e-10 at their own stops, which differ by two).  A slab solve that happens to stop at the oracle's count is
    therefore compared at that count with what the second CPU implementation achieves there (not more than it), and it must agree
    with the undecomposed GPU solve in the same order of operations to rounding."""
    w = inputs.config(2, dt)
    ref = orc.cg(w.s, w.k, w.f, w.u0, w.tol, w.maxit)
    it, rr, st, u = slab_run(w, 4, w.tol, w.maxit)
    assert st == 0 and abs(it - ref["iters"]) <= 2
    d = rel(u, ref["u"])
    if it != ref["iters"] and d > TOL_CG[dt]:
        _, _, _, u = slab_run(w, 4, 0.0, ref["iters"])
        d = rel(u, ref["u"])
    if dt == np.float64 and d > TOL_CG[dt]:
        drift = cfg2_drift()
        assert ref["iters"] in drift and d <= drift[ref["iters"]] and drift[ref["iters"]] > TOL_CG[dt], (d, drift)
        h = B.Fcg(w.L, torch.float64)                       # the undecomposed solve, textbook order, same count: equal to rounding
        h.fcg_set_option(B.FCG_OPT_SPECTRAL_ALPHA, 0)
        h.fcg_set_spectrum(dev(w.s))
        u1 = dev(w.u0)
        h.fcg_solve(dev(w.k), dev(w.f), u1, 0.0, ref["iters"])
        _, _, _, u4 = slab_run(w, 4, 0.0, ref["iters"])
        assert rel(u4, u1.cpu().numpy()) <= 0.2 * TOL_CG[dt]
        h.close()
    else:
        assert d <= TOL_CG[dt], (d, it, ref["iters"])


@pytest.mark.parametrize("cfg,L,dt", [(1, 256, np.float64), (1, 1024, np.float64), (4, 1024, np.float32), (2, 2048, np.float64)])
@pytest.mark.parametrize("G", [2, 4, 8])
def test_slab_peer_mode_fused_exchange(B, cfg, L, dt, G):
    """Peer mode (fcg_slab_set_peers): no all-to-all -- the row pass stores its lines straight into the owning rank's exchange buffer
    and the column pass scatters straight into the source ranks' T2.  The data that arrives is the same, so the solve must be
    BITWISE the all-to-all mode's (same kernels, same arithmetic, same order of sums), and it is checked against the oracle too."""
    w = inputs.config(cfg, dt, L=L)
    maxit = 40 if L >= 2048 else w.maxit
    a = slab_run(w, G, w.tol, maxit)
    b = slab_run(w, G, w.tol, maxit, peers=True)
    assert a[:3] == b[:3] and np.array_equal(a[3], b[3])
    ref = orc.cg(w.s, w.k, w.f, w.u0, 0.0, 6)
    it, _, _, u = slab_run(w, G, 0.0, 6, peers=True)
    assert it == 6 and rel(u, ref["u"]) <= 0.1 * TOL_CG[dt]


# ---- the slab iteration with the spectral search length (three passes; include/fcg.h, DESIGN.md sections 12 and 18)

@pytest.mark.parametrize("cfg,L,dt", [(1, 256, np.float64), (2, 512, np.float64), (1, 1024, np.float64), (4, 1024, np.float32),
                                      (2, 2048, np.float32), (2, 2048, np.float64)])
@pytest.mark.parametrize("G,peers", [(1, False), (2, False), (4, True), (8, True)])
def test_slab_spectral_matches_oracle(B, cfg, L, dt, G, peers):
    """Same protocol as test_slab_cg_matches_oracle; configs[2] fp64 at full size is classified as in test_slab_cg_full_size_config2
    (reading S20) when the solve happens to stop at the oracle's count."""
    w = inputs.config(cfg, dt, L=L)
    ref = orc.cg(w.s, w.k, w.f, w.u0, w.tol, w.maxit, history=True)
    it, rr, st, u = slab_run(w, G, w.tol, w.maxit, peers=peers, spectral=True)
    assert st == ref["status"] and abs(it - ref["iters"]) <= 2, (it, ref["iters"])
    d = rel(u, ref["u"])
    if it != ref["iters"] and d > TOL_CG[dt]:
        it2, _, _, u = slab_run(w, G, 0.0, ref["iters"], peers=peers, spectral=True)
        assert it2 == ref["iters"]
        d = rel(u, ref["u"])
    if (cfg, L, dt) == (2, 2048, np.float64) and d > TOL_CG[dt]:
        drift = cfg2_drift()
        assert d <= drift[ref["iters"]] and drift[ref["iters"]] > TOL_CG[dt], (d, drift)
    else:
        assert d <= TOL_CG[dt], (d, it, ref["iters"])
    assert rr <= w.tol
    refp = orc.cg(w.s, w.k, w.f, w.u0, 0.0, 5, history=True)
    itp, rrp, _, up = slab_run(w, G, 0.0, 5, peers=peers, spectral=True)
    assert itp == 5 and rel(up, refp["u"]) <= 0.1 * TOL_CG[dt]
    assert abs(rrp - refp["hist"][5]) <= 1e-3 * refp["hist"][5]


@pytest.mark.parametrize("L,dt", [(512, np.float64), (2048, np.float32)])
def test_slab_spectral_equals_other_orders(B, L, dt):
    """The three-pass slab iteration agrees (a) at a pinned count with the undecomposed three-launch solve (the same arithmetic per
    element; the order of the partial sums differs) and (b) at the stop with the four-pass slab iteration (alpha from Parseval's
    sum instead of p.q: reading D5's bound, a fifth of the tolerance; in mid-run the two evaluations drift apart like any two
    correct implementations, reading S19 -- 2.7e-5 after 30 iterations at L = 2048 fp32), for every G and both exchange modes."""
    w = inputs.config(1, dt, L=L)
    h = B.Fcg(w.L, TDT[dt])
    h.fcg_set_option(B.FCG_OPT_FUSED, 0)
    h.fcg_set_spectrum(dev(w.s))
    u = dev(w.u0)
    it0, rr0, st0 = h.fcg_solve(dev(w.k), dev(w.f), u, 0.0, 30)
    u0 = u.cpu().numpy()
    h.close()
    eps = 1e-12 if dt == np.float64 else 2e-6
    for G, peers in ((1, False), (2, True), (4, False), (8, True)):
        it, rr, st, ug = slab_run(w, G, 0.0, 30, peers=peers, spectral=True)
        assert (it, st) == (it0, st0) and rel(ug, u0) <= eps and abs(rr - rr0) <= 1e3 * eps * rr0, (G, rel(ug, u0), rr, rr0)
        it4, _, st4, u4 = slab_run(w, G, w.tol, w.maxit, peers=peers, spectral=False)          # (b) at the four-pass solve's own stop,
        it3, _, _, u3 = slab_run(w, G, 0.0, it4, peers=peers, spectral=True)                   #     as test_cg_both_search_length_evaluations
        assert st4 == 0 and it3 == it4 and rel(u3, u4) <= 0.2 * TOL_CG[dt], (G, it4, rel(u3, u4))


def test_slab_spectral_edge_cases(B):
    w = inputs.config(0, np.float64, L=256)
    it, rr, st, u = slab_run(w, 2, w.tol, w.maxit, spectral=True)
    ref = orc.cg(w.s, w.k, w.f, w.u0, w.tol, w.maxit)
    assert st == 0 and abs(it - ref["iters"]) <= 2 and rel(u, ref["u"]) <= TOL_CG[np.float64]
    it2, rr2, st2, _ = slab_run(w, 2, 10 * w.tol, w.maxit, u0=u, spectral=True)          # warm start from the solution
    assert (it2, st2) == (0, 0)
    it3, _, st3, u3 = slab_run(w, 4, w.tol, 0, spectral=True)                             # maxit = 0
    assert (it3, st3) == (0, B.FCG_NOT_CONVERGED) and not u3.any()
    it5, _, st5, _ = slab_run(w, 4, w.tol, 7, spectral=True)                              # maxit reached
    assert (it5, st5) == (7, B.FCG_NOT_CONVERGED)
    w.f[:] = 0
    it4, rr4, st4, u4 = slab_run(w, 2, w.tol, w.maxit, u0=np.ones_like(w.u0), spectral=True)
    assert (it4, rr4, st4) == (0, 0.0, 0) and not u4.any()
    # breakdown (reading S15): a negative-definite operator gives p.Ap < 0 in the first iteration; nothing may change after it
    w = inputs.config(0, np.float64, L=256)
    w.k[:] = -50.0
    ref = orc.cg(w.s, w.k, w.f, w.u0, w.tol, 50)
    for spectral in (True, False):
        it6, _, st6, u6 = slab_run(w, 2, w.tol, 50, spectral=spectral)
        assert st6 == ref["status"] == B.FCG_BREAKDOWN and it6 == ref["iters"]
        assert np.linalg.norm(u6 - ref["u"]) <= 1e-9 * max(np.linalg.norm(ref["u"]), 1e-300) or not (u6.any() or ref["u"].any())


@pytest.mark.parametrize("spectral", [True, False])
@pytest.mark.parametrize("G,peers", [(1, False), (4, False), (4, True)])
def test_slab_graph_replay_is_bitwise_the_eager_loop(B, G, peers, spectral):
    """slab_solve replays blocks of eight iterations from a CUDA graph recorded through fcg_set_stream (first block eager, the graph
    cached on the rank objects per set of buffers).  The same kernels in the same order: count, residual and u bit-identical to
    the eager loop, the same number of kernels accounted for; a second solve on the same buffers reuses the graph."""
    from paper_1305_3625_b200 import slab
    w = inputs.config(1, np.float64, L=512)
    sd = dev(w.s)
    ranks = [slab.SlabRank(w.L, torch.float64, G, g, sd) for g in range(G)]
    if peers:
        slab.connect_peers_local(ranks)
    k = [dev(w.k[r.rows]) for r in ranks]; f = [dev(w.f[r.rows]) for r in ranks]
    u = [dev(w.u0[r.rows]) for r in ranks]
    res = []
    for graph in (False, True, True):
        for x, r in zip(u, ranks):
            x.copy_(dev(w.u0[r.rows]))
        out = slab.slab_solve(ranks, slab.LocalComm(), k, f, u, w.tol, w.maxit, spectral=spectral, graph=graph)
        res.append((out, [x.clone() for x in u], [slab.launch_count(r) for r in ranks]))
    assert len(ranks[0]._graphs) == 1                                  # recorded once, replayed by the third solve too
    assert res[0][0][0] > 16 and res[0][0][2] == 0                     # several replayed blocks
    for other in res[1:]:
        assert other[0] == res[0][0] and other[2] == res[0][2]
        assert all(torch.equal(a, b) for a, b in zip(other[1], res[0][1]))
    ref = orc.cg(w.s, w.k, w.f, w.u0, w.tol, w.maxit)
    assert rel(np.concatenate([x.cpu().numpy() for x in u], axis=0), ref["u"]) <= TOL_CG[np.float64]
    for r in ranks:
        r.close()
