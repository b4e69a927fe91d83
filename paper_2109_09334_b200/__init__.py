"""paper_2109_09334_b200: B200-native hot path of SFFT image differencing (arXiv 2109.09334).

`binding` wraps the C ABI of libsfft_b200.so (include/sfft.h); `build` compiles the library with
nvcc for sm_100a.  Importing this package loads nothing native; the library is loaded on first use
and raises if it cannot be.  (The seeded synthetic inputs live in the repo-level module `synth`,
which serves both this package's tests and the CPU oracle and holds none of the method's arithmetic.)
"""
__all__ = ["binding", "build"]
