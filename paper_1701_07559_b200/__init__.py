"""B200-native Moebius domain-wall fermion even-odd operator and mixed-precision CG solve
(arXiv:1701.07559, Sec. II Eq. (2) and Sec. VII).

The product is the C-ABI library built from csrc/ (declared in include/mdwf.h); `binding`
is the thin ctypes layer with the same names; `inputs` makes the seeded synthetic fields.
Nothing here imports oracle/.  Importing the package does not load the CUDA library;
`binding.lib()` does, and fails loudly if it has not been built.
"""
__all__ = ["inputs", "binding", "build"]
