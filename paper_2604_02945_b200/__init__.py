"""paper_2604_02945_b200 — libmsas: the B200-native Modality Activation Sparsity (MAS) pass of MSAO.

`binding` is the thin ctypes layer over the C ABI in include/msas.h (argument marshalling only; every step runs in
the CUDA kernels under csrc/).  `synth` draws the seeded synthetic workloads.  There is no CPU fallback: importing
`binding` loads the CUDA library and fails loudly if it has not been built.
"""
__all__ = ["synth"]
