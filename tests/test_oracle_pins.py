"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these re-types the oracle's own formula or re-calls its FFT: each is a definition written
differently (explicit DFT matrices, direct convolution), a closed form, an invariant, a library
special case (numpy.fft, numpy.linalg.solve) or brute force on a tiny grid.  CPU only.
"""
import math
import os

import numpy as np
import pytest

from oracle import api as orc
from paper_1305_3625_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / max(np.linalg.norm(np.ravel(b)), 1e-300)


# ---------------------------------------------------------------- P1: transform vs the definition
@pytest.mark.parametrize("L", [2, 4, 8, 16])
def test_p1_fft_matches_dft_matrix(L):
    x = inputs.fft_field(L)
    j = np.arange(L)
    W = np.exp(-2j * np.pi * np.outer(j, j) / L)            # X = W x W^T : definition as a matrix product
    X_def = W @ x @ W.T
    assert rel(orc.fft2(x), X_def) < 1e-13
    assert rel(orc.dft2_brute(x), X_def) < 1e-13            # the O(N^2) loop is the same definition
    # inverse: +i, 1/L^2
    assert rel(orc.fft2(X_def, inverse=True), x) < 1e-13
    assert rel(orc.idft2_brute(X_def), x) < 1e-13


def test_p1_fft_complex_input_and_asymmetry():
    """A complex, non-symmetric input catches a transposed operand or a conjugated sign."""
    L = 8
    rng = np.random.default_rng(11)
    z = rng.standard_normal((L, L)) + 1j * rng.standard_normal((L, L))
    j = np.arange(L)
    W = np.exp(-2j * np.pi * np.outer(j, j) / L)
    assert rel(orc.fft2(z), W @ z @ W.T) < 1e-13
    assert rel(orc.fft2(z, inverse=True), np.conj(W) @ z @ np.conj(W).T / L**2) < 1e-13


# ---------------------------------------------------------------- P2: closed forms of the transform
@pytest.mark.parametrize("L", [8, 64])
def test_p2_impulse_constant_parseval_shift(L):
    e0 = np.zeros((L, L)); e0[0, 0] = 1.0
    assert np.abs(orc.fft2(e0) - 1.0).max() < 1e-14          # impulse -> all ones
    X1 = orc.fft2(np.ones((L, L)))
    spike = np.zeros((L, L), complex); spike[0, 0] = L * L
    assert np.abs(X1 - spike).max() < 1e-10                  # constant -> single spike L^2 at (0,0)
    x = inputs.fft_field(L)
    X = orc.fft2(x)
    assert abs(np.sum(np.abs(X) ** 2) / (L * L * np.sum(x * x)) - 1) < 1e-13     # Parseval
    a0, b0 = 3, 5                                            # shift theorem, distinct shifts per axis
    Xs = orc.fft2(np.roll(x, (a0, b0), axis=(0, 1)))
    m = np.arange(L)
    ph = np.exp(-2j * np.pi * (m[:, None] * a0 + m[None, :] * b0) / L)
    assert rel(Xs, X * ph) < 1e-13


@pytest.mark.parametrize("L", [8, 32])
def test_p2_impulse_reproduces_spectrum(L):
    """north_star: 'the FFT of a single impulse reproduces the spectrum'.  C e0 = c with F c = s,
    and c[0,0] = mean(s)."""
    s = orc.spectrum(L)
    e0 = np.zeros((L, L)); e0[0, 0] = 1.0
    c = orc.apply(s, np.zeros((L, L)), e0)                   # k = 0 -> pure convolution
    assert rel(orc.fft2(c), s) < 1e-13
    assert abs(c[0, 0] - s.mean()) < 1e-14 * L
    # an impulse elsewhere gives the same kernel, shifted (periodic convolution)
    e = np.zeros((L, L)); e[2, 5] = 1.0
    assert rel(orc.apply(s, np.zeros((L, L)), e), np.roll(c, (2, 5), axis=(0, 1))) < 1e-13


# ---------------------------------------------------------------- P3: Listing-4 route vs direct convolution
@pytest.mark.parametrize("L", [4, 16, 32])
def test_p3_fft_convolution_equals_direct(L):
    s = orc.spectrum(L)
    e0 = np.zeros((L, L)); e0[0, 0] = 1.0
    c = np.real(np.fft.ifft2(s))                             # kernel from an independent library
    x = inputs.fft_field(L)
    k = inputs.uniform_k(L)
    y_direct = k * x + orc.conv_direct(c, x)
    assert rel(orc.apply(s, k, x), y_direct) < 1e-13


def test_p3_nonsymmetric_spectrum_takes_real_part():
    """cpyReal drops the imaginary part: for a real but non-even s the oracle equals the
    convolution with Re F^-1 s."""
    L = 8
    s = np.random.default_rng(5).random((L, L)) + 0.5
    c = np.real(np.fft.ifft2(s))
    x = inputs.fft_field(L)
    assert rel(orc.apply(s, np.zeros((L, L)), x), orc.conv_direct(c, x)) < 1e-13


# ---------------------------------------------------------------- P4: circulant eigen closed form
@pytest.mark.parametrize("L,m,n", [(16, 1, 0), (16, 3, 5), (32, 0, 7), (32, 16, 16)])
def test_p4_eigenvector_one_iteration(L, m, n):
    s = orc.spectrum(L)
    kappa = 0.75
    a = np.arange(L)
    f = np.cos(2 * np.pi * (m * a[:, None] + n * a[None, :]) / L)
    lam = kappa + s[m, n]
    y = orc.apply(s, np.full((L, L), kappa), f)
    assert rel(y, lam * f) < 1e-13                           # operator + spectrum indexing [m][n]
    r = orc.cg(s, np.full((L, L), kappa), f, np.zeros((L, L)), 1e-12, 50)
    assert r["status"] == 0 and r["iters"] == 1
    assert rel(r["u"], f / lam) < 1e-12


# ---------------------------------------------------------------- P5: C = 0
def test_p5_zero_spectrum():
    L = 16
    z = np.zeros((L, L))
    f = inputs.normal_f(L)
    r = orc.cg(z, np.full((L, L), 2.0), f, z, 1e-13, 10)     # uniform k: exactly one iteration
    assert r["iters"] == 1 and rel(r["u"], f / 2.0) < 1e-14
    k3 = np.random.default_rng(7).choice([0.5, 1.0, 1.5], size=(L, L))
    r = orc.cg(z, k3, f, z, 1e-13, 10)                       # three distinct eigenvalues: <= 3 iterations
    assert r["status"] == 0 and r["iters"] <= 3
    assert rel(r["u"], f / k3) < 1e-12


# ---------------------------------------------------------------- P6: dense solve
def test_p6_dense_solve():
    L = 8; N = L * L
    s = orc.spectrum(L)
    k = inputs.uniform_k(L); k[inputs.broken_mask(L, 10)] = 0.0
    f = inputs.normal_f(L)
    # explicit matrix from the definition: diag(k) + circulant built from c = F^-1 s (numpy), no oracle call
    c = np.real(np.fft.ifft2(s))
    A = np.zeros((N, N))
    for a in range(L):
        for b in range(L):
            A[a * L + b] = np.roll(c[::-1, ::-1], (a + 1, b + 1), axis=(0, 1)).ravel()
    A += np.diag(k.ravel())
    u_ref = np.linalg.solve(A, f.ravel())
    r = orc.cg(s, k, f, np.zeros((L, L)), 1e-13, 500)
    assert r["status"] == 0
    assert rel(r["u"], u_ref) < 1e-11
    # and the oracle operator is that matrix
    x = inputs.fft_field(L)
    assert rel(orc.apply(s, k, x), A @ x.ravel()) < 1e-13


# ---------------------------------------------------------------- P7: spectrum closed forms, symmetry, SPD
@pytest.mark.parametrize("L", [8, 64, 256])
def test_p7_spectrum_values_and_bounds(L):
    s = orc.spectrum(L)
    assert np.array_equal(s, inputs.spectrum(L)) or np.abs(s - inputs.spectrum(L)).max() < 1e-15 * L
    assert abs(s[0, 0] - L / (2 * math.pi)) < 1e-13 * L
    assert abs(s[L // 2, L // 2] - 1 / math.sqrt(8)) < 1e-15 and s.min() == s[L // 2, L // 2]
    smax = 1 / (2 * math.sin(math.pi / L))
    for (m, n) in [(1, 0), (0, 1), (L - 1, 0), (0, L - 1)]:
        assert abs(s[m, n] - smax) < 1e-12 * L
    assert abs(s.max() - smax) < 1e-12 * L
    assert abs(s[L // 2, 0] - 0.5) < 1e-15 and abs(s[0, L // 2] - 0.5) < 1e-15     # 1/sqrt(4*1)
    assert abs(s[L // 4, 0] - 1 / math.sqrt(2.0)) < 1e-15                          # 4 sin^2(pi/4) = 2
    # even symmetry s[m,n] = s[-m,-n] = s[-m,n]
    idx = (-np.arange(L)) % L
    assert np.abs(s - s[idx][:, idx]).max() < 1e-12 * L
    assert np.abs(s - s[idx]).max() < 1e-12 * L


def test_p7_symmetry_and_rayleigh():
    L = 32
    s = orc.spectrum(L)
    k = inputs.uniform_k(L)
    rng = np.random.default_rng(21)
    x = rng.standard_normal((L, L)); y = rng.standard_normal((L, L))
    Ax, Ay = orc.apply(s, k, x), orc.apply(s, k, y)
    assert abs(np.vdot(x, Ay) - np.vdot(Ax, y)) < 1e-13 * np.linalg.norm(x) * np.linalg.norm(Ay)
    lo = k.min() + 1 / math.sqrt(8); hi = k.max() + 1 / (2 * math.sin(math.pi / L))
    for v, Av in ((x, Ax), (y, Ay)):
        q = np.vdot(v, Av) / np.vdot(v, v)
        assert lo <= q <= hi


# ---------------------------------------------------------------- P8: CG invariants
def test_p8_cg_invariants():
    L = 16
    s = orc.spectrum(L)
    k = inputs.uniform_k(L); f = inputs.normal_f(L)
    r = orc.cg(s, k, f, np.zeros((L, L)), 1e-12, 200, history=True, directions=True)
    assert r["status"] == 0
    P, R = r["P"], r["R"]
    n = P.shape[0]
    AP = np.stack([orc.apply(s, k, p.reshape(L, L)).ravel() for p in P])
    G = P @ AP.T                                             # p_i^T A p_j
    d = np.sqrt(np.diag(G))
    Gn = G / np.outer(d, d)
    # local (three-term) conjugacy holds to rounding; global conjugacy degrades slowly in finite precision
    assert np.abs(np.diag(Gn, 1)).max() < 1e-10
    assert np.abs(Gn - np.diag(np.diag(Gn))).max() < 1e-6
    RR = R @ R.T
    dr = np.sqrt(np.diag(RR))
    RRn = RR / np.outer(dr, dr)
    assert np.abs(np.diag(RRn, 1)).max() < 1e-10
    # residual history is what it says: ||f - A u|| at the stop equals the recurrence residual
    true_res = np.linalg.norm(f - orc.apply(s, k, r["u"])) / np.linalg.norm(f)
    assert abs(true_res - r["relres"]) < 1e-13
    assert abs(r["hist"][-1] - r["relres"]) == 0.0
    assert r["hist"][0] == 1.0                               # u0 = 0 -> r0 = f
    # stop is the FIRST crossing (reading S15)
    assert np.all(r["hist"][:-1] > 1e-12) and r["hist"][-1] <= 1e-12


def test_p8_iteration_counting_and_maxit():
    L = 16
    s = orc.spectrum(L); k = inputs.uniform_k(L); f = inputs.normal_f(L)
    full = orc.cg(s, k, f, np.zeros((L, L)), 1e-12, 200)
    cut = orc.cg(s, k, f, np.zeros((L, L)), 1e-12, 5)
    assert cut["status"] == 1 and cut["iters"] == 5          # S16: maxit reached
    # warm start from the converged solution: zero iterations (S14)
    again = orc.cg(s, k, f, full["u"], 1e-10, 200)
    assert again["iters"] == 0 and again["status"] == 0
    # tol = 0, maxit = n reproduces the first n steps of the longer run (pinned-count protocol)
    assert rel(orc.cg(s, k, f, np.zeros((L, L)), 0.0, 5)["u"], cut["u"]) == 0.0
    # f = 0 -> u = 0, 0 iterations
    z = orc.cg(s, k, np.zeros((L, L)), np.ones((L, L)), 1e-10, 10)
    assert z["iters"] == 0 and np.all(z["u"] == 0)


# ---------------------------------------------------------------- P9 / P10: fracture-loop closed forms
def test_p9_uniform_first_solve_and_first_break():
    L = 256
    w = inputs.config(3)
    r = orc.cg(w.s, w.k, w.f, w.u0, w.tol, w.maxit)
    assert r["iters"] == 1
    u_exact = 1.0 / (1.0 + L / (2 * math.pi))                # f = 1 is the (0,0) eigenvector
    assert abs(u_exact - 0.0239557305201) < 1e-12            # value quoted in SURVEY.md P9
    assert np.abs(r["u"] - u_exact).max() < 1e-13
    k = w.k.copy()
    idx, ratio, second, st = orc.break_step(k, r["u"], w.t)
    assert st == 0 and idx == int(np.argmin(w.t))            # uniform load -> weakest threshold breaks
    assert k.ravel()[idx] == 0.0 and np.count_nonzero(k == 0) == 1
    assert ratio == (1.0 * r["u"].ravel()[idx]) / w.t.ravel()[idx]


def test_p10_sherman_morrison_second_step():
    L = 32
    s = orc.spectrum(L)
    one = np.ones((L, L))
    t = inputs.thresholds(L)
    u0 = 1.0 / (1.0 + s[0, 0])
    b = int(np.argmin(t)); ba, bb = divmod(b, L)
    g = np.real(np.fft.ifft2(1.0 / (1.0 + s)))               # (I + C)^-1 kernel, numpy
    g0 = g[0, 0]
    u_sm = u0 + np.roll(g, (ba, bb), axis=(0, 1)) * u0 / (1.0 - g0)      # rank-one update closed form
    k = one.copy(); u = np.zeros((L, L))
    out = orc.fracture(s, k, one, u, t, 2, 1e-13, 500)
    assert out["steps"] == 2 and out["index"][0] == b and out["iters"][0] == 1
    # after step 2's solve u solves the system with k_b = 0; fracture() broke a 2nd site afterwards, so
    # re-solve explicitly on the one-broken system and compare with the closed form
    k1 = one.copy(); k1.ravel()[b] = 0.0
    r = orc.cg(s, k1, one, np.full((L, L), u0), 1e-13, 500)
    assert rel(r["u"], u_sm) < 1e-11
    cand = (k1 * u_sm / t).ravel().copy(); cand[b] = -np.inf
    assert out["index"][1] == int(np.argmax(cand))


# ---------------------------------------------------------------- P11: CG error bound on iteration counts
@pytest.mark.parametrize("cfg,L", [(0, 64), (1, 128)])
def test_p11_iteration_bound(cfg, L):
    w = inputs.config(cfg, L=L)
    r = orc.cg(w.s, w.k, w.f, w.u0, w.tol, w.maxit)
    assert r["status"] == 0
    lmin = w.k.min() + 1 / math.sqrt(8); lmax = w.k.max() + 1 / (2 * math.sin(math.pi / L))
    kappa = lmax / lmin
    rate = (math.sqrt(kappa) - 1) / (math.sqrt(kappa) + 1)
    # ||r_n|| <= sqrt(kappa) * 2 rate^n ||r_0||  ->  n_bound iterations certainly suffice
    n_bound = math.ceil(math.log(w.tol / (2 * math.sqrt(kappa))) / math.log(rate))
    assert r["iters"] <= n_bound


# ---------------------------------------------------------------- P12: independent library special case
@pytest.mark.parametrize("L", [64, 256])
@pytest.mark.parametrize("dt,tol", [(np.float64, 1e-13), (np.float32, 2e-6)])
def test_p12_numpy_fft_crosscheck(L, dt, tol):
    x = inputs.fft_field(L).astype(dt)
    X = orc.fft2(x)
    assert X.dtype == (np.complex128 if dt == np.float64 else np.complex64)
    assert rel(X, np.fft.fft2(x.astype(np.float64))) < tol
    s = inputs.spectrum(L, dt); k = inputs.uniform_k(L).astype(dt)
    y_np = k.astype(np.float64) * x + np.fft.irfft2(s.astype(np.float64)[:, : L // 2 + 1] * np.fft.rfft2(x.astype(np.float64)), s=(L, L))
    assert rel(orc.apply(s, k, x), y_np) < tol


# ---------------------------------------------------------------- P13: a-posteriori bound
@pytest.mark.parametrize("cfg,L", [(0, 64), (1, 128)])
def test_p13_a_posteriori_bound(cfg, L):
    w = inputs.config(cfg, L=L)
    r = orc.cg(w.s, w.k, w.f, w.u0, w.tol, w.maxit)
    tight = orc.cg(w.s, w.k, w.f, w.u0, 1e-14, 5000)
    true_res = np.linalg.norm(w.f - orc.apply(w.s, w.k, r["u"]))
    lmin = w.k.min() + 1 / math.sqrt(8)
    assert np.linalg.norm(r["u"] - tight["u"]) <= true_res / lmin * (1 + 1e-6) + 1e-13 * np.linalg.norm(tight["u"])


# ---------------------------------------------------------------- break-step edge cases (S13)
def test_break_step_rules():
    k = np.array([1.0, 0.0, 1.0, 1.0, 1.0]); u = np.array([1.0, 100.0, 2.0, 2.0, 1.0]); t = np.array([1.0, 1.0, 1.0, 1.0, 0.5])
    idx, ratio, second, st = orc.break_step(k, u, t)
    assert (idx, ratio, st) == (2, 2.0, 0) and second == 2.0       # 3-way tie at 2.0 -> lowest index; broken site ignored
    idx, _, _, _ = orc.break_step(k, u, t); assert idx == 3
    idx, _, _, _ = orc.break_step(k, u, t); assert idx == 4
    idx, _, _, _ = orc.break_step(k, u, t); assert idx == 0
    idx, _, _, st = orc.break_step(k, u, t); assert idx == -1 and st == orc.NO_CANDIDATE
    # t = 0 -> +inf wins; 0/0 = NaN skipped
    k = np.array([1.0, 1.0, 1.0]); u = np.array([0.0, 1.0, 5.0]); t = np.array([0.0, 0.0, 1.0])
    idx, ratio, _, _ = orc.break_step(k, u, t)
    assert idx == 1 and math.isinf(ratio)
    # float32 arrays: ratio formed in double from the fp32 values
    k = np.array([1.5, 0.7], np.float32); u = np.array([0.3, 0.9], np.float32); t = np.array([0.2, 0.3], np.float32)
    idx, ratio, _, _ = orc.break_step(k, u, t)
    exp = [(float(k0) * float(u0)) / float(t0) for k0, u0, t0 in zip([1.5, np.float32(0.7)], [np.float32(0.3), np.float32(0.9)], [np.float32(0.2), np.float32(0.3)])]
    assert idx == int(np.argmax(exp)) and ratio == max(exp)


# ---------------------------------------------------------------- fp32 instantiation
def test_fp32_oracle_tracks_fp64():
    L = 64
    w64 = inputs.config(0, np.float64, L=L); w32 = inputs.config(0, np.float32, L=L)
    r64 = orc.cg(w64.s, w64.k, w64.f, w64.u0, 1e-5, 1000)
    r32 = orc.cg(w32.s, w32.k, w32.f, w32.u0, 1e-5, 1000)
    assert r32["u"].dtype == np.float32
    assert abs(r32["iters"] - r64["iters"]) <= 1
    assert rel(r32["u"], r64["u"]) < 1e-4


# ---------------------------------------------------------------- P14 (indicative, survey probe -- not a paper value)
def test_p14_indicative_iteration_counts():
    """BASELINE.md section 3 (survey probe with numpy/pocketfft, NOT a paper number): cfg0 28, cfg1 105.
    Expected within +-2."""
    w = inputs.config(0)
    assert abs(orc.cg(w.s, w.k, w.f, w.u0, w.tol, w.maxit)["iters"] - 28) <= 2
    w = inputs.config(1)
    assert abs(orc.cg(w.s, w.k, w.f, w.u0, w.tol, w.maxit)["iters"] - 105) <= 2


# ---------------------------------------------------------------------------------------------------------------
# Preconditioned CG: M = kbar I + C.  Pins chosen so that a wrong preconditioner spectrum, a
# swapped r/z in a dot product, or p built from r instead of z fails at least one of them.
def _dense_A(L, s, k):
    N = L * L
    A = np.zeros((N, N))
    for j in range(N):
        e = np.zeros(N); e[j] = 1.0
        A[:, j] = orc.apply(s, k, e.reshape(L, L)).ravel()
    return A


def test_pcg_exact_preconditioner_one_iteration():
    """k uniform = kbar  =>  M = A  =>  z0 = A^-1 r0 and PCG stops after exactly ONE iteration for any f."""
    L = 16
    s = inputs.spectrum(L); k = np.full((L, L), 0.8); f = np.random.default_rng(11).standard_normal((L, L))
    r = orc.pcg(s, k, f, np.zeros((L, L)), 0.8, 1e-12, 50)
    assert r["status"] == 0 and r["iters"] == 1
    assert np.linalg.norm(orc.apply(s, k, r["u"]) - f) <= 1e-12 * np.linalg.norm(f)


def test_pcg_matches_dense_solve():
    L = 8
    s = inputs.spectrum(L); k = inputs.uniform_k(L); k[inputs.broken_mask(L, 10)] = 0.0
    f = inputs.normal_f(L)
    u_dense = np.linalg.solve(_dense_A(L, s, k), f.ravel()).reshape(L, L)
    r = orc.pcg(s, k, f, np.zeros((L, L)), float(k.mean()), 1e-13, 200)
    assert r["status"] == 0
    assert np.linalg.norm(r["u"] - u_dense) <= 1e-11 * np.linalg.norm(u_dense)


def test_pcg_with_scalar_preconditioner_reproduces_cg():
    """s_M constant: with a huge kbar, M^-1 = (1/kbar) I up to O(s/kbar); PCG with M = c I is CG itself (same iterates).
    kbar = 1e12 makes the deviation ~1e-11, far below the comparison tolerance, and pins PCG to the already-pinned CG."""
    L = 16
    s = inputs.spectrum(L); k = inputs.uniform_k(L); f = inputs.normal_f(L)
    a = orc.cg(s, k, f, np.zeros((L, L)), 1e-10, 200, history=True)
    b = orc.pcg(s, k, f, np.zeros((L, L)), 1e12, 1e-10, 200, history=True)
    assert a["iters"] == b["iters"]
    assert np.allclose(a["hist"], b["hist"], rtol=1e-6)
    assert np.linalg.norm(a["u"] - b["u"]) <= 1e-9 * np.linalg.norm(a["u"])


def test_pcg_invariants_and_iteration_gain():
    """p_i A-orthogonal, r_i M^-1-orthogonal (r_i . z_j = 0, i != j), z = M^-1 r with M = kbar I + C, and fewer iterations
    than CG: kappa(M^-1 A) <= (kbar + s_min + dk) / (kbar + s_min - dk) with dk = max |k - kbar|."""
    L = 16
    s = inputs.spectrum(L); k = inputs.uniform_k(L); f = inputs.normal_f(L); kbar = float(k.mean())
    r = orc.pcg(s, k, f, np.zeros((L, L)), kbar, 1e-12, 100, directions=True)
    P, Z, R = r["P"].astype(np.float64), r["Z"].astype(np.float64), r["R"].astype(np.float64)
    n = P.shape[0]
    AP = np.stack([orc.apply(s, k, P[i].reshape(L, L)).ravel() for i in range(n)])
    G = P @ AP.T
    off = G - np.diag(np.diag(G))
    assert np.abs(off).max() <= 1e-9 * np.abs(np.diag(G)).max()
    RZ = R @ Z.T
    offz = RZ - np.diag(np.diag(RZ))
    assert np.abs(offz).max() <= 1e-9 * np.abs(np.diag(RZ)).max()
    for i in (0, n // 2, n - 1):                                     # M z = r
        Mz = orc.apply(s, np.full((L, L), kbar), Z[i].reshape(L, L)).ravel()
        assert np.linalg.norm(Mz - R[i]) <= 1e-12 * np.linalg.norm(R[i])
    cg_it = orc.cg(s, k, f, np.zeros((L, L)), 1e-12, 100)["iters"]
    assert r["iters"] < cg_it
    dk = np.abs(k - kbar).max(); lo = kbar + 1 / np.sqrt(8.0)
    kappa = (lo + dk) / (lo - dk)
    bound = int(np.ceil(np.log(2.0 / 1e-12) / -np.log((np.sqrt(kappa) - 1) / (np.sqrt(kappa) + 1)))) + 2
    assert r["iters"] <= bound


def test_pcg_fp32_and_edge_cases():
    L = 32
    s = inputs.spectrum(L, np.float32); k = inputs.uniform_k(L).astype(np.float32); f = np.ones((L, L), np.float32)
    r32 = orc.pcg(s, k, f, np.zeros((L, L), np.float32), 1.0, 1e-5, 100)
    r64 = orc.pcg(s.astype(np.float64), k.astype(np.float64), f.astype(np.float64), np.zeros((L, L)), 1.0, 1e-5, 100)
    assert r32["status"] == 0 and abs(r32["iters"] - r64["iters"]) <= 1
    assert np.linalg.norm(r32["u"] - r64["u"]) <= 1e-4 * np.linalg.norm(r64["u"])
    z = orc.pcg(s, k, np.zeros((L, L), np.float32), np.ones((L, L), np.float32), 1.0, 1e-5, 10)
    assert z["iters"] == 0 and not z["u"].any()
    m = orc.pcg(s, k, f, np.zeros((L, L), np.float32), 1.0, 1e-12, 3)
    assert (m["iters"], m["status"]) == (3, orc.NOT_CONVERGED)


# ---------------------------------------------------------------- quasi-static loop with PCG solves
def test_pcg_fracture_step0_closed_form_and_sherman_morrison():
    """P9 / P10 for the PCG loop: k = kbar = 1 makes M = A, so step 0 is ONE iteration to u = 1/(1 + L/2pi) and the first
    break is argmin t; the second break follows from the rank-one (Sherman-Morrison) closed form."""
    L = 32
    s = orc.spectrum(L)
    one = np.ones((L, L))
    t = inputs.thresholds(L)
    u0 = 1.0 / (1.0 + s[0, 0])
    b = int(np.argmin(t)); ba, bb = divmod(b, L)
    g = np.real(np.fft.ifft2(1.0 / (1.0 + s)))
    u_sm = u0 + np.roll(g, (ba, bb), axis=(0, 1)) * u0 / (1.0 - g[0, 0])
    k = one.copy(); u = np.zeros((L, L))
    out = orc.pcg_fracture(s, k, one, u, t, 1.0, 2, 1e-13, 500)
    assert out["steps"] == 2 and out["index"][0] == b and out["iters"][0] == 1
    cand = (one * u_sm / t).ravel().copy(); cand[b] = -np.inf
    assert out["index"][1] == int(np.argmax(cand))
    assert np.count_nonzero(k == 0) == 2 and k.ravel()[b] == 0.0


@pytest.mark.parametrize("L,steps", [(16, 60), (32, 120)])
def test_pcg_fracture_same_break_sequence_as_cg_loop(L, steps):
    """The break sequence belongs to the exact solutions: the PCG loop must reproduce the (independently pinned) CG loop's
    indices wherever the top-2 gap is far above the solver error, with fewer iterations in total."""
    w = inputs.config(3, L=L, nsteps=steps)
    k1 = w.k.copy(); u1 = w.u0.copy()
    a = orc.fracture(w.s, k1, w.f, u1, w.t, steps, 1e-12, 2000)
    k2 = w.k.copy(); u2 = w.u0.copy()
    b = orc.pcg_fracture(w.s, k2, w.f, u2, w.t, 1.0, steps, 1e-12, 2000)
    assert a["steps"] == steps and b["steps"] == steps
    assert a["gap"].min() > 1e-9
    assert np.array_equal(a["index"], b["index"]) and np.array_equal(k1, k2)
    assert rel(u2, u1) < 1e-10
    assert b["iters"].sum() < a["iters"].sum()
