"""B200-native submatrix method for the matrix sign function (arXiv 2205.14741).

The product is libsubmatrix.so (C ABI in include/submatrix.h, CUDA kernels in csrc/); `binding`
is its ctypes front end.  Importing `binding` raises if the library has not been built: there is
no CPU fallback.  Build with `python -m paper_2205_14741_b200.build`.
"""
__all__ = ["binding", "build"]
