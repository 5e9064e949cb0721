"""fcg -- FFT-accelerated conjugate gradient for the lattice fracture model of arXiv 1305.3625, B200-native.

Sub-modules
  binding   ctypes binding of libfcg.so (the C-ABI in include/fcg.h); same names as the C calls
  inputs    seeded synthetic workloads of BASELINE.json:configs (no method arithmetic)
  build     nvcc build of csrc/ into libfcg.so (sm_100a)
Nothing is imported eagerly: ``inputs`` must stay importable without the CUDA library.
"""
__all__ = ["binding", "inputs", "build"]
