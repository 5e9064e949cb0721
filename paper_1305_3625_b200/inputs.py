"""Seeded synthetic inputs for the five BASELINE.json configs (recipe: SURVEY.md section 8(d)).

This module serves both the CUDA path's tests/bench and the oracle's tests.  It holds input recipes
only -- no transform, operator, solver or break arithmetic -- and imports neither the binding nor
the oracle.  All arrays are drawn in fp64 with ``numpy.random.default_rng(seed)``, shape (L, L) in one
call, row-major, then cast once to the run dtype; the identical bytes go to oracle and GPU.

The paper measures on its own unpublished fracture model; these inputs stand
in for it with the shapes and distributions BASELINE.json:configs states.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED_K, SEED_T, SEED_BROKEN, SEED_F, SEED_FFT = 0, 1, 2, 3, 4


def spectrum(L: int, dtype=np.float64) -> np.ndarray:
    """Input recipe of BASELINE.json configs[0]: s(q) = 1/|q~|, |q~| = sqrt(4 sin^2(pi m/L) + 4 sin^2(pi n/L)),
    s(0,0) = L/(2 pi).  Row-major [m][n], computed in fp64, rounded once to ``dtype``."""
    m = np.arange(L, dtype=np.float64)
    sm2 = 4.0 * np.sin(np.pi * m / L) ** 2
    q2 = sm2[:, None] + sm2[None, :]
    q2[0, 0] = 1.0
    s = 1.0 / np.sqrt(q2)
    s[0, 0] = L / (2.0 * np.pi)
    return np.ascontiguousarray(s, dtype=dtype)


def uniform_k(L: int, seed: int = SEED_K) -> np.ndarray:
    """k_i i.i.d. uniform [0.5, 1.5]."""
    return 0.5 + np.random.default_rng(seed).random((L, L))


def broken_mask(L: int, fraction_den: int, seed: int = SEED_BROKEN) -> np.ndarray:
    """Exactly N // fraction_den sites = first entries of a seeded permutation (reading S9)."""
    N = L * L
    idx = np.random.default_rng(seed).permutation(N)[: N // fraction_den]
    mask = np.zeros(N, bool)
    mask[idx] = True
    return mask.reshape(L, L)


def normal_f(L: int, seed: int = SEED_F) -> np.ndarray:
    """f_i i.i.d. normal(1, 0.1)."""
    return np.random.default_rng(seed).normal(1.0, 0.1, (L, L))


def thresholds(L: int, seed: int = SEED_T) -> np.ndarray:
    """t_i i.i.d. uniform [0, 1]."""
    return np.random.default_rng(seed).random((L, L))


def fft_field(L: int, seed: int = SEED_FFT) -> np.ndarray:
    """x ~ N(0,1) for the stand-alone transform checks."""
    return np.random.default_rng(seed).standard_normal((L, L))


@dataclass
class Workload:
    name: str
    L: int
    dtype: np.dtype
    k: np.ndarray
    f: np.ndarray
    u0: np.ndarray
    s: np.ndarray
    tol: float
    maxit: int
    t: np.ndarray | None = None
    nsteps: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return self.L * self.L


def _mk(name, L, dtype, k, f, tol, maxit, t=None, nsteps=0, **meta) -> Workload:
    dt = np.dtype(dtype)
    c = lambda a: None if a is None else np.ascontiguousarray(a, dtype=dt)
    return Workload(name, L, dt, c(k), c(f), np.zeros((L, L), dt), spectrum(L, dt), tol, maxit,
                    c(t), nsteps, meta)


def config(i: int, dtype=None, L: int | None = None, nsteps: int | None = None) -> Workload:
    """Workload i of BASELINE.json:configs.  ``L`` / ``nsteps`` override the size for scaled-down
    parity cases that keep the same recipe (used by tests; bench uses the stated sizes)."""
    if i == 0:
        L = L or 64
        return _mk("cfg0", L, dtype or np.float64, uniform_k(L), np.ones((L, L)), 1e-10, 1000)
    if i == 1:
        L = L or 512
        k = uniform_k(L); k[broken_mask(L, 10)] = 0.0
        return _mk("cfg1", L, dtype or np.float64, k, normal_f(L), 1e-10, 1000, broken="N//10")
    if i == 2:
        L = L or 2048
        dt = np.dtype(dtype or np.float64)
        return _mk("cfg2", L, dt, uniform_k(L), np.ones((L, L)), 1e-10 if dt == np.float64 else 1e-5, 1000)
    if i == 3:
        L = L or 256
        return _mk("cfg3", L, dtype or np.float64, np.ones((L, L)), np.ones((L, L)), 1e-10, 1000,
                   t=thresholds(L), nsteps=2000 if nsteps is None else nsteps)
    if i == 4:
        L = L or 8192
        k = uniform_k(L); k[broken_mask(L, 20)] = 0.0
        return _mk("cfg4", L, dtype or np.float32, k, normal_f(L), 1e-5, 2000, broken="N//20")
    raise ValueError("config index must be 0..4")


def precond_kbar(k: np.ndarray) -> float:
    """Constant of the spectral preconditioner M = kbar I + C (reading D4): the mean stiffness,
    accumulated in fp64.  A parameter recipe, handed unchanged to oracle and GPU."""
    return float(np.mean(np.asarray(k, dtype=np.float64)))


# ---- the paper's formulation in the bond forces -----------------------------
# Constants of eq. (1c): the paper gives no values, these are the recipe's (reading F4).
GREEN_NU, GREEN_E, GREEN_A = 0.3, 1.0, 1.0
FORCE_KAPPA, FORCE_D = 1.0, 1.0
# Stopping tolerance of the force recipe: two converged CG runs differ by up to cond(I + K G) * tol in f, and cond ~ 0.7 L here
# (eigenvalues between 1 + kappa g_min ~ 1.5 and 1 + kappa g(0) ~ 1 + L), so a 1e-9 comparison needs tol well below 1e-9 / L.
FORCE_TOL = {np.dtype(np.float64): 1e-12, np.dtype(np.float32): 1e-5}


def gradient_thresholds(L: int, gradient: float, seed: int = SEED_T) -> np.ndarray:
    """t_i = U[0,1] + gradient * a / L for row a: "insert a gradient in the threshold distribution", which
    turns the damage into a front that advances along the rows."""
    return thresholds(L, seed) + gradient * (np.arange(L, dtype=np.float64) / L)[:, None]


def force_k(L: int, broken_den: int | None = None, kappa: float = FORCE_KAPPA) -> np.ndarray:
    """All unbroken bonds share one elastic constant; a seeded 1/broken_den of the bonds is broken."""
    k = np.full((L, L), kappa, np.float64)
    if broken_den:
        k[broken_mask(L, broken_den)] = 0.0
    return k
