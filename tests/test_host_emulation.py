"""CPU check of libfcg's index algebra (digit reversal, swizzle, row packing, packed DC/Nyquist column,
fused column pass) by replaying the pass bodies of csrc/fcg_passes.cuh on the host (tests/emul/emul.cpp).

This is host logic of the CUDA path, checked against numpy.fft -- it is NOT the parity test (that is
tests/test_gpu_parity.py against oracle/) and the harness is never part of the product library.
"""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

from paper_1305_3625_b200 import inputs

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SRC = os.path.join(HERE, "emul", "emul.cpp")
CSRC = os.path.join(ROOT, "paper_1305_3625_b200", "csrc")
LIB = os.path.join(HERE, "emul", "libemul.so")


@pytest.fixture(scope="module")
def emul():
    deps = [SRC] + [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cuh")]
    if not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(d) for d in deps):
        cuda_inc = os.environ.get("CUDA_HOME", "/usr/local/cuda") + "/include"
        subprocess.run(["g++", "-O1", "-std=c++17", "-fPIC", "-shared", "-I" + cuda_inc, "-I" + CSRC, SRC, "-o", LIB],
                       check=True)
    lib = C.CDLL(LIB)
    for name in ("emul_run_f64", "emul_run_f32"):
        getattr(lib, name).argtypes = [C.c_int, C.c_int] + [C.c_void_p] * 5 + [C.c_int]
        getattr(lib, name).restype = C.c_int
    return lib


def _run(lib, L, dt, what, s, k, x, variant=0):
    fn = lib.emul_run_f64 if dt == np.float64 else lib.emul_run_f32
    s = np.ascontiguousarray(s, dt); k = np.ascontiguousarray(k, dt); x = np.ascontiguousarray(x, dt)
    y = np.zeros((L, L), dt)
    T = np.zeros((L // 2, L), np.complex128 if dt == np.float64 else np.complex64)
    p = lambda a: a.ctypes.data_as(C.c_void_p)
    st = fn(L, what, p(s), p(k), p(x), p(y), p(T), variant)
    return st, y, T


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / np.linalg.norm(np.ravel(b))


SIZES = [16, 32, 64, 128, 256, 512, 1024]


@pytest.mark.parametrize("L", SIZES + [2048])
@pytest.mark.parametrize("dt,tol", [(np.float64, 1e-13), (np.float32, 5e-6)])
def test_forward_transform_layout(emul, L, dt, tol):
    x = inputs.fft_field(L).astype(dt)
    st, _, T = _run(emul, L, dt, 1, np.ones((L, L)), np.ones((L, L)), x)
    assert st == 0
    X = np.fft.fft2(x.astype(np.float64))                    # X[m][n]
    ref = X[:, : L // 2].T.copy()                            # T[n][m]
    ref[0] = X[:, 0] + 1j * X[:, L // 2]                     # packed row 0: Y0 + i YN
    assert rel(T, ref) < tol


@pytest.mark.parametrize("L", SIZES)
@pytest.mark.parametrize("dt,tol", [(np.float64, 1e-13), (np.float32, 5e-6)])
def test_operator_all_row_variants(emul, L, dt, tol):
    s = inputs.spectrum(L, dt); k = inputs.uniform_k(L).astype(dt); x = inputs.fft_field(L).astype(dt)
    ref = k.astype(np.float64) * x + np.fft.irfft2(s.astype(np.float64)[:, : L // 2 + 1] * np.fft.rfft2(x.astype(np.float64)), s=(L, L))
    seen = 0
    for v in range(4):
        st, y, _ = _run(emul, L, dt, 0, s, k, x, v)
        if st != 0:
            continue
        seen += 1
        assert rel(y, ref) < tol, f"variant {v}"
    assert seen >= 1


@pytest.mark.parametrize("L", [16, 64, 512])
def test_operator_nonsymmetric_spectrum_uses_even_part(emul, L):
    """set_spectrum keeps (s[m,n] + s[-m,-n])/2: the same as taking the real part at the end."""
    rng = np.random.default_rng(9)
    s = rng.random((L, L)) + 0.5
    x = inputs.fft_field(L); k = np.zeros((L, L))
    ref = np.real(np.fft.ifft2(s * np.fft.fft2(x)))
    st, y, _ = _run(emul, L, np.float64, 0, s, k, x)
    assert st == 0 and rel(y, ref) < 1e-13


@pytest.mark.parametrize("L", [16, 128, 1024])
@pytest.mark.parametrize("dt,tol", [(np.float64, 1e-13), (np.float32, 5e-6)])
def test_round_trip_public_path(emul, L, dt, tol):
    x = inputs.fft_field(L).astype(dt)
    st, y, _ = _run(emul, L, dt, 2, np.ones((L, L)), np.ones((L, L)), x)
    assert st == 0 and rel(y, x) < tol


@pytest.mark.slow
@pytest.mark.parametrize("L,dt,tol", [(4096, np.float32, 5e-6), (8192, np.float32, 5e-6), (4096, np.float64, 1e-13)])
def test_operator_large(emul, L, dt, tol):
    s = inputs.spectrum(L, dt); k = inputs.uniform_k(L).astype(dt); x = inputs.fft_field(L).astype(dt)
    ref = k.astype(np.float64) * x + np.fft.irfft2(s.astype(np.float64)[:, : L // 2 + 1] * np.fft.rfft2(x.astype(np.float64)), s=(L, L))
    st, y, _ = _run(emul, L, dt, 0, s, k, x, 0)
    assert st == 0 and rel(y, ref) < tol
