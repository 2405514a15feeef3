"""B200-native Wilson-Dirac D / D-dagger and CG on D D-dagger (arXiv:2111.14958 hot path).

`paper_2111_14958_b200.inputs`  — seeded synthetic lattices (numpy only, shared with the test oracle).
`paper_2111_14958_b200.wilson`  — thin ctypes binding of the C-ABI library (include/wilson_cg.h);
                                  imports lazily so that `inputs` is usable without CUDA.
"""
__all__ = ["inputs", "wilson"]
