"""paper_2311_00639_b200 -- the sparse-SYK H.v / Lanczos / OTOC hot path of arXiv 2311.00639 on B200 (sm_100a).

`csrc/` holds the CUDA kernels and the C ABI (include/syk.h); `binding` is the ctypes layer with the same
names.  Importing `binding` fails loudly when `libsyk_b200.so` has not been built (`build.build()`): there is
no CPU path.
"""
__all__ = ["binding", "build", "inputs", "replicas"]
