"""pwham: B200-native plane-wave Hamiltonian application, Chebyshev filtering and Gram products.

`paper_2604_11139_b200.synth`   -- seeded synthetic workloads (inputs only; imports no compute code)
`paper_2604_11139_b200.binding` -- thin ctypes binding over the C-ABI library libpwham.so (include/pwham.h)

Nothing is imported eagerly: the binding fails loudly if the CUDA library is missing, and `synth` must stay
importable without it (the CPU oracle tests use it).
"""
__all__ = ["synth", "binding"]
