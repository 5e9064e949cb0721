"""Pins of the oracle's force formulation (eqs. (1)-(2)) against what the
paper and the mathematics fix: numerical quadrature of the integral (1c), its far field and symmetries, the model
equations (1a)/(1b) evaluated with a direct O(N^2) sum, a dense solve, closed forms, CG invariants, brute force.
CPU only.  None of them re-types the oracle's formula or re-calls its transform."""
import math

import numpy as np
import pytest

from oracle import api as orc
from paper_1305_3625_b200 import inputs

NU, E, A = inputs.GREEN_NU, inputs.GREEN_E, inputs.GREEN_A


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / max(np.linalg.norm(np.ravel(b)), 1e-300)


def quad_green(X, Y, nu, E, a, n=48):
    """Integral (1c) by tensor Gauss-Legendre quadrature (no singularity inside the square for (X,Y) != 0)."""
    x, w = np.polynomial.legendre.leggauss(n)
    xs = 0.5 * a * x; ws = 0.5 * a * w
    r = np.sqrt((X - xs[:, None]) ** 2 + (Y - xs[None, :]) ** 2)
    return (1 - nu * nu) / (math.pi * E * a * a) * float(ws @ (1.0 / r) @ ws)


# ---------------------------------------------------------------- F-P1: the integral (1c)
@pytest.mark.parametrize("nu,E,a", [(0.3, 1.0, 1.0), (0.0, 2.5, 0.5), (0.45, 0.7, 2.0)])
def test_green_function_matches_quadrature(nu, E, a):
    L = 16
    G = orc.green_function(L, nu, E, a)
    for da, db in [(0, 1), (1, 0), (1, 1), (2, 5), (7, 3), (8, 8), (0, 8)]:
        assert abs(G[da, db] / quad_green(a * da, a * db, nu, E, a) - 1) < 1e-9, (da, db)
    # minimum image: offsets beyond L/2 wrap to the negative side (an asymmetric pair catches a swapped axis)
    assert abs(G[13, 2] / quad_green(-3 * a, 2 * a, nu, E, a) - 1) < 1e-9
    assert abs(G[2, 13] / quad_green(2 * a, -3 * a, nu, E, a) - 1) < 1e-9
    assert G[13, 2] != G[2, 12]


def test_green_function_self_term_far_field_symmetry():
    L = 256
    G = orc.green_function(L, NU, E, A)
    pref = (1 - NU * NU) / (math.pi * E * A * A)
    # self term: the integral of 1/r over a square of side a about its centre is 4 a ln(1 + sqrt 2) (polar coordinates:
    # 8 int_0^{pi/4} (a / 2 cos t) dt)
    assert abs(G[0, 0] / (pref * 4 * A * math.log(1 + math.sqrt(2))) - 1) < 1e-14
    # far field: a point force, pref a^2 / r, with a relative quadrupole correction of order (a/r)^2
    for da, db in [(40, 0), (0, 77), (30, 40), (128, 128)]:
        r = A * math.hypot(da, db)
        assert abs(G[da, db] / (pref * A * A / r) - 1) < 0.5 * (A / r) ** 2 + 1e-12
    # even kernel and x <-> y symmetry of the square
    idx = (-np.arange(L)) % L
    assert np.abs(G - G[idx][:, idx]).max() < 1e-13          # (cancellation in the four-corner sum: ~1e-16 r/a)
    assert np.abs(G - G.T).max() < 1e-13
    # positive and decreasing along an axis up to the half box
    assert np.all(G > 0) and np.all(np.diff(G[0, : L // 2 + 1]) < 0)


@pytest.mark.parametrize("L", [8, 32])
def test_kernel_spectrum_is_the_dft_of_G_and_positive(L):
    G = orc.green_function(L, NU, E, A)
    s = orc.kernel_spectrum(G)
    j = np.arange(L)
    W = np.exp(-2j * np.pi * np.outer(j, j) / L)
    S = W @ G @ W.T                                           # the definition as matrix products
    assert np.abs(S.imag).max() < 1e-12 * np.abs(S).max()     # even kernel -> real transform
    assert rel(s, S.real) < 1e-13
    assert abs(s[0, 0] - G.sum()) < 1e-12 * G.sum()           # zero mode = sum of the kernel
    assert s.min() > 0                                        # "the whole matrix problem is positive-definite"
    # fp32 instantiation: kernel rounded once, transform in fp32
    s32 = orc.kernel_spectrum(G.astype(np.float32))
    assert s32.dtype == np.float32 and rel(s32, S.real) < 5e-6


# ---------------------------------------------------------------- F-P2: operator and solve vs the model equations
def dense_G(G):
    """G_ij as the L^2 x L^2 matrix the paper writes: circulant in both lattice directions."""
    L = G.shape[0]
    a = np.arange(L)
    d = (a[:, None] - a[None, :]) % L
    return G[d[:, None, :, None], d[None, :, None, :]].reshape(L * L, L * L)


def test_force_apply_matches_direct_sum():
    L = 8
    G = orc.green_function(L, NU, E, A); g = orc.kernel_spectrum(G)
    rng = np.random.default_rng(21)
    k = inputs.force_k(L, 5); x = rng.standard_normal((L, L))
    want = x + k * orc.conv_direct(G, x)                      # x + K (G x), the convolution as a direct O(N^2) sum
    assert rel(orc.force_apply(g, k, x), want) < 1e-13
    want2 = (np.eye(L * L) + np.diag(k.ravel()) @ dense_G(G)) @ x.ravel()
    assert rel(orc.force_apply(g, k, x), want2) < 1e-13
    # a non-uniform k catches k applied to x instead of to G x
    k2 = inputs.uniform_k(L)
    assert rel(orc.force_apply(g, k2, x), x + k2 * orc.conv_direct(G, x)) < 1e-13


@pytest.mark.parametrize("L,den", [(8, None), (8, 4), (16, 10)])
def test_force_cg_matches_dense_solve_and_model_equations(L, den):
    G = orc.green_function(L, NU, E, A); g = orc.kernel_spectrum(G)
    k = inputs.force_k(L, den, kappa=1.7); D = 0.8
    out = orc.force_cg(g, k, D, np.zeros((L, L)), 1e-13, 500)
    assert out["status"] == 0
    f = out["f"]
    M = np.eye(L * L) + np.diag(k.ravel()) @ dense_G(G)
    f_dense = np.linalg.solve(M, k.ravel() * D)               # eq. (2) solved by LAPACK
    assert rel(f, f_dense) < 1e-11
    u = orc.conv_direct(G, f)                                 # (1b) by the direct sum
    assert np.abs(f - (-k * (u - D))).max() < 1e-11           # (1a): f_i = -k_i (u_i - D)
    assert np.all(f[k == 0] == 0)                             # broken bonds carry nothing, exactly
    assert np.all(f[k > 0] > 0)


def test_force_cg_intact_plate_closed_form():
    """No broken bonds: the uniform solution f_i = kappa D / (1 + kappa g(0)), found in one iteration."""
    L = 32
    G = orc.green_function(L, NU, E, A); g = orc.kernel_spectrum(G)
    kappa, D = 2.0, 0.37
    out = orc.force_cg(g, np.full((L, L), kappa), D, np.zeros((L, L)), 1e-13, 50)
    assert out["status"] == 0 and out["iters"] == 1
    assert np.abs(out["f"] / (kappa * D / (1 + kappa * G.sum())) - 1).max() < 1e-12
    # linear in D (what the break rule rests on) and zero for D = 0
    o2 = orc.force_cg(g, inputs.force_k(L, 7), 3.0, np.zeros((L, L)), 1e-13, 300)
    o1 = orc.force_cg(g, inputs.force_k(L, 7), 1.0, np.zeros((L, L)), 1e-13, 300)
    assert rel(o2["f"], 3.0 * o1["f"]) < 1e-11
    o0 = orc.force_cg(g, inputs.force_k(L, 7), 0.0, np.ones((L, L)), 1e-13, 300)
    assert o0["iters"] == 0 and np.all(o0["f"] == 0)


def test_force_cg_invariants():
    """CG in the forces is CG: residuals orthogonal, directions conjugate under B = I + K G, recurrence residual = true
    residual, every vector zero on the broken bonds (reading F1)."""
    L = 8
    G = orc.green_function(L, NU, E, A); g = orc.kernel_spectrum(G)
    k = inputs.force_k(L, 4); D = 1.0
    out = orc.force_cg(g, k, D, np.zeros((L, L)), 1e-12, 200, history=True, directions=True)
    P, R = out["P"], out["R"]; n = len(P)
    assert out["status"] == 0 and 3 <= n <= int((k > 0).sum())
    B = np.eye(L * L) + np.diag(k.ravel()) @ dense_G(G)
    m = 6          # the first vectors: rounding grows like 1/||r_j|| in the normalised products of later ones
    Pn = P[:m] / np.linalg.norm(P[:m], axis=1)[:, None]; Rn = R[:m] / np.linalg.norm(R[:m], axis=1)[:, None]
    C1 = Pn @ B @ Pn.T; C2 = Rn @ Rn.T
    off = lambda M: np.abs(M - np.diag(np.diag(M))).max()
    assert off(C1) < 1e-8 * np.abs(np.diag(C1)).max() and off(C2) < 1e-8
    assert np.all(P[:, k.ravel() == 0] == 0) and np.all(R[:, k.ravel() == 0] == 0)
    true_res = np.linalg.norm(k.ravel() * D - B @ out["f"].ravel()) / np.linalg.norm(k.ravel() * D)
    assert abs(true_res - out["relres"]) < 1e-10
    assert abs(out["hist"][-1] - out["relres"]) < 1e-15
    # warm start from the solution: zero iterations
    again = orc.force_cg(g, k, D, out["f"], 1e-10, 200)
    assert again["iters"] == 0


def test_force_cg_equals_displacement_form():
    """Eliminating f instead of u from (1a), (1b) gives (K + G^-1) u = K D, the symmetric form BASELINE.json states with
    spectrum 1/g; both must describe the same state: f = K (D - u)."""
    L = 16
    G = orc.green_function(L, NU, E, A); g = orc.kernel_spectrum(G)
    k = inputs.force_k(L, 6, kappa=1.3); D = 1.0
    f = orc.force_cg(g, k, D, np.zeros((L, L)), 1e-13, 500)["f"]
    u = orc.cg(1.0 / g, k, k * D, np.zeros((L, L)), 1e-13, 2000)["u"]
    assert rel(k * (D - u), f) < 1e-10


@pytest.mark.parametrize("L,den", [(8, 4), (16, 6)])
def test_displacement_route_maps_and_dense_solve(L, den):
    """Reading F7: the oracle's two element-wise maps (s = 1/g, f = -k (u - D)) and the whole route -- CG or PCG on
    (K + G^-1) u = K D, then (1a) -- against LAPACK on the dense matrices: u = (K + G^-1)^-1 K D with G^-1 inverted as a matrix,
    and the forces against the dense solve of eq. (2)."""
    G = orc.green_function(L, NU, E, A); g = orc.kernel_spectrum(G)
    k = inputs.force_k(L, den, kappa=1.3); D = 0.8
    s = orc.inverse_spectrum(g)
    assert np.array_equal(s, 1.0 / g) and s.dtype == g.dtype
    assert orc.inverse_spectrum(g.astype(np.float32)).dtype == np.float32
    GG = dense_G(G); K = np.diag(k.ravel())
    u_dense = np.linalg.solve(K + np.linalg.inv(GG), k.ravel() * D)
    f_dense = np.linalg.solve(np.eye(L * L) + K @ GG, k.ravel() * D)
    for solve in (lambda: orc.cg(s, k, k * D, np.zeros((L, L)), 1e-13, 2000),
                  lambda: orc.pcg(s, k, k * D, np.zeros((L, L)), float(k.mean()), 1e-13, 2000)):
        out = solve()
        assert out["status"] == 0 and rel(out["u"], u_dense) < 1e-10
        f = orc.force_from_displacement(k, D, out["u"])
        assert rel(f, f_dense) < 1e-10 and np.all(f[k == 0] == 0)
        assert np.abs(orc.conv_direct(G, f) - out["u"]).max() < 1e-10          # (1b): u = G f by the direct sum
    # the map itself on hand-made numbers, sign included: f = -k (u - D)
    kk = np.array([[2.0, 0.0], [0.5, 1.0]]); uu = np.array([[0.25, 9.0], [-1.0, 3.0]])
    assert np.array_equal(orc.force_from_displacement(kk, 1.0, uu), np.array([[1.5, 0.0], [1.0, -2.0]]))


# ---------------------------------------------------------------- F-P3: break rule and quasi-static loop
def test_force_break_step_rule():
    k = np.array([1.0, 0.0, 1.0, 1.0, 1.0]); f = np.array([0.25, 9.0, 0.75, 0.375, np.nan]); t = np.array([0.5, 0.125, 1.0, 0.5, 0.5])
    i, ratio, second, st = orc.force_break_step(k, f, t)
    # ratios 0.5, (broken), 0.75, 0.75, NaN -> index 2 (lowest of the tie); bond removed with its force
    assert (i, st) == (2, 0) and ratio == 0.75 and second == 0.75 and k[2] == 0 and f[2] == 0
    i, ratio, second, st = orc.force_break_step(k, f, t)
    assert i == 3 and ratio == 0.75 and second == 0.5
    k0 = np.zeros(3); i, _, _, st = orc.force_break_step(k0, np.ones(3), np.ones(3))
    assert (i, st) == (-1, orc.NO_CANDIDATE)


def test_force_fracture_first_breaks_and_brute_force():
    L = 8
    G = orc.green_function(L, NU, E, A); g = orc.kernel_spectrum(G)
    t = inputs.gradient_thresholds(L, 0.5)
    k = inputs.force_k(L); f = np.zeros((L, L))
    nsteps = 12
    out = orc.force_fracture(g, k, 1.0, f, t, nsteps, 1e-12, 500)
    assert out["steps"] == nsteps and len(set(out["index"])) == nsteps
    # intact plate: uniform forces, so the weakest bond goes first, at D_c = t_min (1 + kappa g(0)) / kappa
    assert out["index"][0] == int(np.argmin(t)) and out["iters"][0] == 1
    assert abs(1.0 / out["ratio"][0] - t.min() * (1 + G.sum())) < 1e-10
    # every step against a dense solve of eq. (2) on the current set of bonds
    kk = inputs.force_k(L).ravel(); GG = dense_G(G)
    for s in range(nsteps):
        fd = np.linalg.solve(np.eye(L * L) + np.diag(kk) @ GG, kk)
        ratio = np.where(kk > 0, fd / t.ravel(), -np.inf)
        assert int(np.argmax(ratio)) == out["index"][s]
        assert abs(ratio.max() / out["ratio"][s] - 1) < 1e-9
        kk[out["index"][s]] = 0.0
    assert np.array_equal(k.ravel() == 0, kk == 0) and np.all(f[k == 0] == 0)
    # the neighbours of a broken bond pick up its load: total force drops, maximum rises
    assert out["gap"].min() > 0


def test_force_fracture_gradient_makes_a_front():
    """With a strong gradient in the thresholds the first rows fail first."""
    L = 16
    g = orc.kernel_spectrum(orc.green_function(L, NU, E, A))
    t = inputs.gradient_thresholds(L, 50.0)
    k = inputs.force_k(L); f = np.zeros((L, L))
    out = orc.force_fracture(g, k, 1.0, f, t, 2 * L, 1e-10, 500)
    assert out["steps"] == 2 * L and np.all(out["index"] // L < 4)


def test_force_fracture_through_displacements_same_sequence_and_brute_force():
    """Reading F7 applied to the loop: the break sequence and the critical ratios are properties of the exact states, so the loop
    through the displacements (CG and PCG solves) must reproduce the loop on eq. (2) and a dense-LAPACK replay, step by step."""
    L = 8
    G = orc.green_function(L, NU, E, A); g = orc.kernel_spectrum(G); sinv = orc.inverse_spectrum(g)
    t = inputs.gradient_thresholds(L, 0.5)
    nsteps = 14
    ref = orc.force_fracture(g, inputs.force_k(L), 1.0, np.zeros((L, L)), t, nsteps, 1e-13, 500)
    kk = inputs.force_k(L).ravel(); GG = dense_G(G)
    dense_idx, dense_ratio = [], []
    for s in range(nsteps):
        fd = np.linalg.solve(np.eye(L * L) + np.diag(kk) @ GG, kk)
        r = np.where(kk > 0, fd / t.ravel(), -np.inf)
        dense_idx.append(int(np.argmax(r))); dense_ratio.append(r.max()); kk[dense_idx[-1]] = 0.0
    for kbar in (None, 1.0):
        k = inputs.force_k(L); u = np.zeros((L, L))
        out = orc.force_fracture_displacement(sinv, k, 1.0, u, t, nsteps, 1e-13, 2000, kbar=kbar)
        assert out["steps"] == nsteps
        assert np.array_equal(out["index"], ref["index"]) and list(out["index"]) == dense_idx
        assert np.abs(out["ratio"] / np.array(dense_ratio) - 1).max() < 1e-9
        assert np.array_equal(k.ravel() == 0, kk == 0)
        # u is the plate's displacement of the last solved state: (1b) with that state's forces, broken bond still carrying
        f_last = out["f"].copy(); f_last.ravel()[out["index"][-1]] = dense_ratio[-1] * t.ravel()[out["index"][-1]]
        assert np.abs(orc.conv_direct(G, f_last) - u).max() < 1e-9
        assert out["f"].ravel()[out["index"][-1]] == 0 and out["gap"].min() > 0
    # first step from the intact plate: the weakest bond, at D_c = t_min (1 + kappa g(0)) / kappa, after a uniform solve
    assert out["index"][0] == int(np.argmin(t)) and abs(1.0 / out["ratio"][0] - t.min() * (1 + G.sum())) < 1e-9
    # PCG needs fewer iterations than CG on the same route once bonds are broken
    k = inputs.force_k(L); cg_it = orc.force_fracture_displacement(sinv, k, 1.0, np.zeros((L, L)), t, nsteps, 1e-13, 2000)["iters"].sum()
    assert out["iters"].sum() < cg_it
    # running out of bonds
    k = np.zeros((L, L)); k[1, 2] = k[5, 5] = 1.0
    o2 = orc.force_fracture_displacement(sinv, k, 1.0, np.zeros((L, L)), t, 5, 1e-12, 500)
    assert o2["steps"] == 2 and not k.any()
