"""B200-native GPFC phase folding + noise normalisation (arXiv 2312.02063).

The product is the C-ABI library `libgpfc.so` built from `csrc/` (see
`include/gpfc.h`); `binding` is the thin ctypes layer with the same names.
Nothing here imports `oracle/`.
"""

__all__ = ["binding", "workloads", "build"]
