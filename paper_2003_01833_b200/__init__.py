"""B200-native barycentric Lagrange treecode for the Yukawa convolution of Green Iteration
(arXiv 2003.01833).  The product is libbltc.so (csrc/, C ABI in include/bltc.h); `binding`
is the thin ctypes layer with the same entry-point names, `inputs` the seeded synthetic
workload generators.  No CPU fallback exists: the binding raises if the CUDA library is missing.
"""
__all__ = ["binding", "inputs", "build"]
