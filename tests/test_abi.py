"""CPU-side checks of the boundary: libfcg.so builds/loads, exports every symbol include/fcg.h declares,
sizes its workspace as DESIGN.md states, and fails loudly without a CUDA device (no CPU fallback)."""
import ctypes as C
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1305_3625_b200 import build
    build.build()
    from paper_1305_3625_b200 import binding
    return binding.lib()


def declared_symbols():
    hdr = open(os.path.join(ROOT, "include", "fcg.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    return sorted(set(re.findall(r"\b(fcg_[a-z_0-9]+)\s*\(", hdr)))


def test_exports_every_declared_symbol(lib):
    from paper_1305_3625_b200 import binding
    syms = declared_symbols()
    assert len(syms) >= 14
    for s in syms:
        assert hasattr(lib, s), f"libfcg.so does not export {s}"
    assert sorted(binding.EXPORTS) == syms            # the Python binding mirrors the header one to one


def test_workspace_bytes(lib):
    for dt, w in ((0, 4), (1, 8)):
        for L in (16, 64, 2048, 8192):
            n = lib.fcg_workspace_bytes(L, dt)
            N = L * L
            assert 6 * N * w <= n <= 6 * N * w + 72 * L * w + 64 * 1024     # T (1) + shat, mhat (1/2 each) + r,p,q,z (4), + tables
    for L in (0, 8, 24, 100, 16384, -4):
        assert lib.fcg_workspace_bytes(L, 1) == 0
    assert lib.fcg_workspace_bytes(64, 7) == 0


def test_version_and_null_handle(lib):
    assert b"sm_100a" in lib.fcg_version()
    assert lib.fcg_last_launch_count(None) == -1
    assert lib.fcg_destroy(None) == -1
    assert lib.fcg_set_spectrum(None, None) == -1


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_create_fails_loudly_without_gpu(lib):
    h = C.c_void_p()
    assert lib.fcg_create(64, 1, None, None, C.byref(h)) == -3        # FCG_CUDA_ERROR, not a CPU fallback
    assert not h.value
    assert lib.fcg_create(100, 1, None, None, C.byref(h)) == -2       # FCG_UNSUPPORTED
    assert lib.fcg_create(64, 5, None, None, C.byref(h)) == -1        # FCG_INVALID_ARG


def test_product_does_not_reference_oracle():
    """The product path must not import, link or execute anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1305_3625_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) == "build":
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "fcg_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_1305_3625_b200\b", txt, flags=re.M), f
            assert "csrc" not in txt, f
