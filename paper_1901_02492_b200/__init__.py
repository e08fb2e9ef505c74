"""B200-native KBMOD shift-and-stack hot path (psi/phi build + trajectory search).

`binding` is the thin ctypes layer over libkbmod_b200.so (include/kbmod_b200.h);
`synth` is the seeded input generator; `build` compiles the library with nvcc for sm_100a.
"""
__all__ = ["binding", "synth", "build"]
