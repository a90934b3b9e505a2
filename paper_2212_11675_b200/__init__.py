"""B200-native hot path of the Gaia AVU-GSR solver (arxiv 2212.11675): PC-LSQR with the
structured aprod1/aprod2 products, as hand-written CUDA behind the C ABI of include/gsr.h.

`binding` is the thin ctypes layer over libgsr_b200.so; `inputs` draws seeded synthetic
systems; `build` compiles the library in-tree.  Nothing here falls back to the CPU."""
__all__ = ["binding", "inputs", "build"]
