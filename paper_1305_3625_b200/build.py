"""Build csrc/ into paper_1305_3625_b200/libfcg.so with nvcc for sm_100a (cross-compiles without a GPU).

One object per lattice size (fcg_inst.cu with -DFCG_INST_L=<L>) plus fcg.cu, compiled in parallel and
linked with the static CUDA runtime.  Usage:  python -m paper_1305_3625_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
# FCG_BUILD_DIR / FCG_LIB_OUT: build a variant (e.g. with FCG_EXTRA_FLAGS=-D...) beside the product for A/B measurements;
# the binding loads it when FCG_LIB names it.  The defaults are the product.
OBJ = os.environ.get("FCG_BUILD_DIR") or os.path.join(HERE, "build")
LIB = os.environ.get("FCG_LIB_OUT") or os.path.join(HERE, "libfcg.so")
SIZES = [16, 32, 64, 128, 256, 512, 1024, 2048, 4096, 8192]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "--expt-relaxed-constexpr", "-Xcompiler", "-fPIC", "-Xptxas", "-v"] + os.environ.get("FCG_EXTRA_FLAGS", "").split()


def _sources():
    hdr = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    hdr.append(os.path.join(os.path.dirname(HERE), "include", "fcg.h"))
    return hdr


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(job):
    src, obj, extra, force = job
    deps = _sources() + [src]
    if not force and not _stale(obj, deps):
        return obj, ""
    cmd = [NVCC, *FLAGS, *extra, "-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed: {' '.join(cmd)}\n{r.stdout}\n{r.stderr}")
    return obj, r.stderr


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    jobs = [(os.path.join(CSRC, "fcg.cu"), os.path.join(OBJ, "fcg.o"), [], force)]
    for L in SIZES:
        jobs.append((os.path.join(CSRC, "fcg_inst.cu"), os.path.join(OBJ, f"fcg_inst_{L}.o"), [f"-DFCG_INST_L={L}"], force))
    with cf.ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
        results = list(ex.map(_compile, jobs))
    objs = [o for o, _ in results]
    log = "\n".join(l for _, l in results if l)
    if log:
        with open(os.path.join(OBJ, "ptxas.log"), "w") as fh:
            fh.write(log)
        if verbose:
            print(log)
    if force or _stale(LIB, objs):
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [NVCC, "-shared", "-o", tmp, *objs, "-gencode", "arch=compute_100a,code=sm_100a"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed: {' '.join(cmd)}\n{r.stdout}\n{r.stderr}")
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
