"""B200-native hot path of arXiv 1408.5853: one explicit-implicit FD time step of
axisymmetric multilayer heat conduction, as a C-ABI library (include/heat.h) with
hand-written sm_100a fp64 CUDA kernels, plus this thin ctypes binding.

`inputs` (seeded synthetic workloads) is importable without the CUDA library; `binding`
loads paper_1408_5853_b200/libheat_b200.so and fails loudly if it is missing.
"""
__all__ = ["inputs", "binding", "build"]
