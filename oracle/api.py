"""ctypes loader and numpy marshalling for the CPU oracle (oracle/fcg_oracle.c).

TEST INFRASTRUCTURE ONLY.  Importable from tests/, __graft_entry__.smoke() and the cpu_baseline /
``--impl reference`` legs of bench.py -- never from the product package.  This module holds no
arithmetic of the method: every number comes out of fcg_oracle.c.  It imports nothing from
paper_1305_3625_b200.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(_HERE, "fcg_oracle.c"), os.path.join(_HERE, "fcg_oracle_impl.h")]
_LIB_PATH = os.path.join(_HERE, "libfcg_oracle.so")
_lock = threading.Lock()
_lib = None

OK, NOT_CONVERGED, BREAKDOWN, NO_CANDIDATE = 0, 1, -4, -6


def build(force: bool = False) -> str:
    """Compile fcg_oracle.c with gcc (-O2, OpenMP, no FMA contraction) next to its source."""
    newest = max(os.path.getmtime(p) for p in _SRC)
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < newest:
        tmp = _LIB_PATH + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-Wall",
               _SRC[0], "-o", tmp, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
        os.replace(tmp, _LIB_PATH)
    return _LIB_PATH


def lib() -> C.CDLL:
    global _lib
    with _lock:
        if _lib is None:
            _lib = C.CDLL(build())
            _declare(_lib)
    return _lib


_vp, _i, _d, _ll = C.c_void_p, C.c_int, C.c_double, C.c_longlong


def _declare(L: C.CDLL) -> None:
    L.oracle_spectrum.argtypes = [_i, _vp]
    L.oracle_spectrum.restype = None
    L.oracle_dft2_brute.argtypes = [_i, _vp, _vp]
    L.oracle_dft2_brute.restype = None
    L.oracle_idft2_brute.argtypes = [_i, _vp, _vp]
    L.oracle_idft2_brute.restype = None
    L.oracle_conv_direct.argtypes = [_i, _vp, _vp, _vp]
    L.oracle_conv_direct.restype = None
    L.oracle_green_function.argtypes = [_i, _d, _d, _d, _vp]
    L.oracle_green_function.restype = None
    L.oracle_num_threads.restype = _i
    L.oracle_set_num_threads.argtypes = [_i]
    for suf in ("_f64", "_f32"):
        f = getattr(L, "oracle_fft2" + suf)
        f.argtypes = [_i, _vp, _i]; f.restype = _i
        f = getattr(L, "oracle_apply" + suf)
        f.argtypes = [_i, _vp, _vp, _vp, _vp]; f.restype = _i
        f = getattr(L, "oracle_cg" + suf)
        f.argtypes = [_i, _vp, _vp, _vp, _vp, _d, _i, C.POINTER(_i), C.POINTER(_d), _vp, _vp, _vp]
        f.restype = _i
        f = getattr(L, "oracle_pcg" + suf)
        f.argtypes = [_i, _vp, _vp, _vp, _vp, _d, _d, _i, C.POINTER(_i), C.POINTER(_d), _vp, _vp, _vp, _vp]
        f.restype = _i
        f = getattr(L, "oracle_pcg_fracture" + suf)
        f.argtypes = [_i, _vp, _vp, _vp, _vp, _vp, _d, _i, _d, _i, _vp, _vp, _vp]
        f.restype = _i
        f = getattr(L, "oracle_break_step" + suf)
        f.argtypes = [_ll, _vp, _vp, _vp, C.POINTER(_ll), C.POINTER(_d), C.POINTER(_d)]
        f.restype = _i
        f = getattr(L, "oracle_fracture" + suf)
        f.argtypes = [_i, _vp, _vp, _vp, _vp, _vp, _i, _d, _i, _vp, _vp, _vp]
        f.restype = _i
        f = getattr(L, "oracle_kernel_spectrum" + suf)
        f.argtypes = [_i, _vp, _vp]; f.restype = _i
        f = getattr(L, "oracle_force_apply" + suf)
        f.argtypes = [_i, _vp, _vp, _vp, _vp]; f.restype = _i
        f = getattr(L, "oracle_force_cg" + suf)
        f.argtypes = [_i, _vp, _vp, _d, _vp, _d, _i, C.POINTER(_i), C.POINTER(_d), _vp, _vp, _vp]
        f.restype = _i
        f = getattr(L, "oracle_inverse_spectrum" + suf)
        f.argtypes = [_ll, _vp, _vp]; f.restype = None
        f = getattr(L, "oracle_force_from_displacement" + suf)
        f.argtypes = [_ll, _vp, _d, _vp, _vp]; f.restype = None
        f = getattr(L, "oracle_force_fracture_displacement" + suf)
        f.argtypes = [_i, _vp, _vp, _d, _vp, _vp, _vp, _i, _d, _i, _d, _i, _vp, _vp, _vp, _vp]
        f.restype = _i
        f = getattr(L, "oracle_force_break_step" + suf)
        f.argtypes = [_ll, _vp, _vp, _vp, C.POINTER(_ll), C.POINTER(_d), C.POINTER(_d)]
        f.restype = _i
        f = getattr(L, "oracle_force_fracture" + suf)
        f.argtypes = [_i, _vp, _vp, _d, _vp, _vp, _i, _d, _i, _vp, _vp, _vp, _vp]
        f.restype = _i


def _suf(dtype) -> str:
    dt = np.dtype(dtype)
    if dt == np.float64:
        return "_f64"
    if dt == np.float32:
        return "_f32"
    raise TypeError(f"oracle supports float32/float64, got {dt}")


def _arr(a, dtype, shape=None) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=dtype)
    if shape is not None and a.shape != shape:
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


def _p(a: np.ndarray | None):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(int(n))


def spectrum(L: int) -> np.ndarray:
    s = np.empty((L, L), np.float64)
    lib().oracle_spectrum(L, _p(s))
    return s


def dft2_brute(x: np.ndarray) -> np.ndarray:
    L = x.shape[0]
    x = _arr(x, np.float64, (L, L))
    X = np.empty((L, L), np.complex128)
    lib().oracle_dft2_brute(L, _p(x), _p(X))
    return X


def idft2_brute(X: np.ndarray) -> np.ndarray:
    L = X.shape[0]
    X = _arr(X, np.complex128, (L, L))
    x = np.empty((L, L), np.complex128)
    lib().oracle_idft2_brute(L, _p(X), _p(x))
    return x


def conv_direct(c: np.ndarray, x: np.ndarray) -> np.ndarray:
    L = x.shape[0]
    c = _arr(c, np.float64, (L, L)); x = _arr(x, np.float64, (L, L))
    y = np.empty((L, L), np.float64)
    lib().oracle_conv_direct(L, _p(c), _p(x), _p(y))
    return y


def fft2(x: np.ndarray, inverse: bool = False) -> np.ndarray:
    """2D DFT of a complex (or real) L x L array in the precision of x (complex64/complex128)."""
    x = np.asarray(x)
    L = x.shape[0]
    cdt = np.complex64 if x.dtype in (np.float32, np.complex64) else np.complex128
    rdt = np.float32 if cdt == np.complex64 else np.float64
    buf = np.array(x, dtype=cdt, order="C", copy=True).reshape(L, L)
    st = getattr(lib(), "oracle_fft2" + _suf(rdt))(L, _p(buf), 1 if inverse else 0)
    if st != 0:
        raise ValueError("oracle_fft2: L must be a power of two")
    return buf


def apply(s, k, x) -> np.ndarray:
    """y = k o x + F^-1(s o F x) in the dtype of x."""
    x = np.asarray(x); dt = x.dtype; L = x.shape[0]
    s = _arr(s, dt, (L, L)); k = _arr(k, dt, (L, L)); x = _arr(x, dt, (L, L))
    y = np.empty((L, L), dt)
    st = getattr(lib(), "oracle_apply" + _suf(dt))(L, _p(s), _p(k), _p(x), _p(y))
    if st != 0:
        raise ValueError("oracle_apply: bad argument")
    return y


def cg(s, k, f, u0, tol: float, maxit: int, history: bool = False, directions: bool = False):
    """Returns dict(u, iters, relres, status[, hist][, P, R]); dtype taken from f."""
    f = np.asarray(f); dt = f.dtype; L = f.shape[0]; N = L * L
    s = _arr(s, dt, (L, L)); k = _arr(k, dt, (L, L)); f = _arr(f, dt, (L, L))
    u = np.array(u0, dtype=dt, order="C", copy=True).reshape(L, L)
    hist = np.full(maxit + 1, np.nan, np.float64) if history else None
    P = np.zeros((maxit, N), dt) if directions else None
    R = np.zeros((maxit, N), dt) if directions else None
    it = C.c_int(0); rr = C.c_double(0.0)
    st = getattr(lib(), "oracle_cg" + _suf(dt))(L, _p(s), _p(k), _p(f), _p(u), float(tol), int(maxit),
                                                 C.byref(it), C.byref(rr), _p(hist), _p(P), _p(R))
    out = dict(u=u, iters=int(it.value), relres=float(rr.value), status=int(st))
    if history:
        out["hist"] = hist[: it.value + 1]
    if directions:
        out["P"] = P[: it.value]; out["R"] = R[: it.value]
    return out


def pcg(s, k, f, u0, kbar: float, tol: float, maxit: int, history: bool = False, directions: bool = False):
    """Preconditioned CG with M = kbar I + C.  Returns dict(u, iters, relres, status[, hist][, P, Z, R])."""
    f = np.asarray(f); dt = f.dtype; L = f.shape[0]; N = L * L
    s = _arr(s, dt, (L, L)); k = _arr(k, dt, (L, L)); f = _arr(f, dt, (L, L))
    u = np.array(u0, dtype=dt, order="C", copy=True).reshape(L, L)
    hist = np.full(maxit + 1, np.nan, np.float64) if history else None
    P = np.zeros((maxit, N), dt) if directions else None
    Z = np.zeros((maxit, N), dt) if directions else None
    R = np.zeros((maxit, N), dt) if directions else None
    it = C.c_int(0); rr = C.c_double(0.0)
    st = getattr(lib(), "oracle_pcg" + _suf(dt))(L, _p(s), _p(k), _p(f), _p(u), float(kbar), float(tol), int(maxit),
                                                  C.byref(it), C.byref(rr), _p(hist), _p(P), _p(Z), _p(R))
    out = dict(u=u, iters=int(it.value), relres=float(rr.value), status=int(st))
    if history:
        out["hist"] = hist[: it.value + 1]
    if directions:
        out["P"] = P[: it.value]; out["Z"] = Z[: it.value]; out["R"] = R[: it.value]
    return out


def break_step(k: np.ndarray, u, t):
    """In-place on k (must be a C-contiguous float array). Returns (index, ratio, second, status)."""
    dt = k.dtype
    if not k.flags.c_contiguous:
        raise ValueError("k must be C-contiguous (modified in place)")
    u = _arr(u, dt); t = _arr(t, dt)
    idx = C.c_longlong(-1); ratio = C.c_double(0.0); second = C.c_double(0.0)
    st = getattr(lib(), "oracle_break_step" + _suf(dt))(k.size, _p(k), _p(u), _p(t),
                                                         C.byref(idx), C.byref(ratio), C.byref(second))
    return int(idx.value), float(ratio.value), float(second.value), int(st)


def fracture(s, k, f, u, t, nsteps: int, tol: float, maxit: int):
    """In-place on k and u. Returns dict(index[nsteps], iters[nsteps], gap[nsteps], steps)."""
    dt = k.dtype; L = k.shape[0]
    s = _arr(s, dt, (L, L)); f = _arr(f, dt, (L, L)); t = _arr(t, dt, (L, L))
    if not (k.flags.c_contiguous and u.flags.c_contiguous and u.dtype == dt):
        raise ValueError("k, u must be C-contiguous arrays of one dtype (modified in place)")
    index = np.full(nsteps, -1, np.int64); iters = np.zeros(nsteps, np.int32)
    gap = np.full(nsteps, np.nan, np.float64)
    done = getattr(lib(), "oracle_fracture" + _suf(dt))(L, _p(s), _p(k), _p(f), _p(u), _p(t), int(nsteps),
                                                        float(tol), int(maxit), _p(index), _p(iters), _p(gap))
    return dict(index=index, iters=iters, gap=gap, steps=int(done))


def pcg_fracture(s, k, f, u, t, kbar: float, nsteps: int, tol: float, maxit: int):
    """Quasi-static loop with PCG solves.  In-place on k and u. Returns dict(index, iters, gap, steps)."""
    dt = k.dtype; L = k.shape[0]
    s = _arr(s, dt, (L, L)); f = _arr(f, dt, (L, L)); t = _arr(t, dt, (L, L))
    if not (k.flags.c_contiguous and u.flags.c_contiguous and u.dtype == dt):
        raise ValueError("k, u must be C-contiguous arrays of one dtype (modified in place)")
    index = np.full(nsteps, -1, np.int64); iters = np.zeros(nsteps, np.int32)
    gap = np.full(nsteps, np.nan, np.float64)
    done = getattr(lib(), "oracle_pcg_fracture" + _suf(dt))(L, _p(s), _p(k), _p(f), _p(u), _p(t), float(kbar), int(nsteps),
                                                            float(tol), int(maxit), _p(index), _p(iters), _p(gap))
    return dict(index=index, iters=iters, gap=gap, steps=int(done))


# ---- the paper's formulation in the bond forces, (I + K G) f = K D (eq. (2)) ----------------

def green_function(L: int, nu: float, E: float, a: float) -> np.ndarray:
    """Real-space Green's function of eq. (1c) on the periodic lattice, G[da][db], fp64."""
    G = np.empty((L, L), np.float64)
    lib().oracle_green_function(int(L), float(nu), float(E), float(a), _p(G))
    return G


def kernel_spectrum(G) -> np.ndarray:
    """s = Re F G in the dtype of G."""
    G = np.asarray(G); dt = G.dtype; L = G.shape[0]
    G = _arr(G, dt, (L, L))
    s = np.empty((L, L), dt)
    if getattr(lib(), "oracle_kernel_spectrum" + _suf(dt))(L, _p(G), _p(s)) != 0:
        raise ValueError("oracle_kernel_spectrum: L must be a power of two")
    return s


def force_apply(g, k, x) -> np.ndarray:
    """y = x + k o F^-1(g o F x) in the dtype of x."""
    x = np.asarray(x); dt = x.dtype; L = x.shape[0]
    g = _arr(g, dt, (L, L)); k = _arr(k, dt, (L, L)); x = _arr(x, dt, (L, L))
    y = np.empty((L, L), dt)
    if getattr(lib(), "oracle_force_apply" + _suf(dt))(L, _p(g), _p(k), _p(x), _p(y)) != 0:
        raise ValueError("oracle_force_apply: bad argument")
    return y


def force_cg(g, k, D: float, f0, tol: float, maxit: int, history: bool = False, directions: bool = False):
    """CG on (I + K G) f = K D.  Returns dict(f, iters, relres, status[, hist][, P, R]); dtype taken from k."""
    k = np.asarray(k); dt = k.dtype; L = k.shape[0]; N = L * L
    g = _arr(g, dt, (L, L)); k = _arr(k, dt, (L, L))
    f = np.array(f0, dtype=dt, order="C", copy=True).reshape(L, L)
    hist = np.full(maxit + 1, np.nan, np.float64) if history else None
    P = np.zeros((maxit, N), dt) if directions else None
    R = np.zeros((maxit, N), dt) if directions else None
    it = C.c_int(0); rr = C.c_double(0.0)
    st = getattr(lib(), "oracle_force_cg" + _suf(dt))(L, _p(g), _p(k), float(D), _p(f), float(tol), int(maxit),
                                                       C.byref(it), C.byref(rr), _p(hist), _p(P), _p(R))
    out = dict(f=f, iters=int(it.value), relres=float(rr.value), status=int(st))
    if history:
        out["hist"] = hist[: it.value + 1]
    if directions:
        out["P"] = P[: it.value]; out["R"] = R[: it.value]
    return out


def inverse_spectrum(g) -> np.ndarray:
    """s = 1 / g element by element, in the dtype of g: the spectrum of G^-1 (reading F7)."""
    g = np.ascontiguousarray(g); s = np.empty_like(g)
    getattr(lib(), "oracle_inverse_spectrum" + _suf(g.dtype))(g.size, _p(g), _p(s))
    return s


def force_from_displacement(k, D: float, u) -> np.ndarray:
    """f = -k (u - D), eq. (1a), in the dtype of k."""
    k = np.ascontiguousarray(k); u = _arr(u, k.dtype, k.shape); f = np.empty_like(k)
    getattr(lib(), "oracle_force_from_displacement" + _suf(k.dtype))(k.size, _p(k), float(D), _p(u), _p(f))
    return f


def force_break_step(k: np.ndarray, f: np.ndarray, t):
    """In-place on k and f. Returns (index, ratio, second, status)."""
    dt = k.dtype
    if not (k.flags.c_contiguous and f.flags.c_contiguous and f.dtype == dt):
        raise ValueError("k, f must be C-contiguous arrays of one dtype (modified in place)")
    t = _arr(t, dt)
    idx = C.c_longlong(-1); ratio = C.c_double(0.0); second = C.c_double(0.0)
    st = getattr(lib(), "oracle_force_break_step" + _suf(dt))(k.size, _p(k), _p(f), _p(t),
                                                               C.byref(idx), C.byref(ratio), C.byref(second))
    return int(idx.value), float(ratio.value), float(second.value), int(st)


def force_fracture(g, k, D: float, f, t, nsteps: int, tol: float, maxit: int):
    """Quasi-static loop in the forces.  In-place on k and f. Returns dict(index, iters, ratio, gap, steps)."""
    dt = k.dtype; L = k.shape[0]
    g = _arr(g, dt, (L, L)); t = _arr(t, dt, (L, L))
    if not (k.flags.c_contiguous and f.flags.c_contiguous and f.dtype == dt):
        raise ValueError("k, f must be C-contiguous arrays of one dtype (modified in place)")
    index = np.full(nsteps, -1, np.int64); iters = np.zeros(nsteps, np.int32)
    ratio = np.full(nsteps, np.nan, np.float64); gap = np.full(nsteps, np.nan, np.float64)
    done = getattr(lib(), "oracle_force_fracture" + _suf(dt))(L, _p(g), _p(k), float(D), _p(f), _p(t), int(nsteps),
                                                              float(tol), int(maxit), _p(index), _p(iters), _p(ratio), _p(gap))
    return dict(index=index, iters=iters, ratio=ratio, gap=gap, steps=int(done))


def force_fracture_displacement(sinv, k, D: float, u, t, nsteps: int, tol: float, maxit: int, kbar: float | None = None):
    """Quasi-static loop of the force model through the displacements (reading F7); PCG solves when kbar is given.
    In-place on k and u. Returns dict(index, iters, ratio, gap, steps, f)."""
    dt = k.dtype; L = k.shape[0]
    sinv = _arr(sinv, dt, (L, L)); t = _arr(t, dt, (L, L))
    if not (k.flags.c_contiguous and u.flags.c_contiguous and u.dtype == dt):
        raise ValueError("k, u must be C-contiguous arrays of one dtype (modified in place)")
    index = np.full(nsteps, -1, np.int64); iters = np.zeros(nsteps, np.int32)
    ratio = np.full(nsteps, np.nan, np.float64); gap = np.full(nsteps, np.nan, np.float64)
    f = np.zeros((L, L), dt)
    done = getattr(lib(), "oracle_force_fracture_displacement" + _suf(dt))(
        L, _p(sinv), _p(k), float(D), _p(u), _p(f), _p(t), 0 if kbar is None else 1, 0.0 if kbar is None else float(kbar),
        int(nsteps), float(tol), int(maxit), _p(index), _p(iters), _p(ratio), _p(gap))
    return dict(index=index, iters=iters, ratio=ratio, gap=gap, steps=int(done), f=f)

