"""B200-native Wilson Dslash (the hot path of arXiv 2301.03636's running example).

    from paper_2301_03636_b200 import binding   # loads the C-ABI CUDA library; raises if it is missing
    from paper_2301_03636_b200 import inputs    # seeded synthetic fields (NumPy only)

Importing the package itself touches neither CUDA nor torch, so the CPU-only tooling (input
generator, library build) stays usable without a GPU.  There is no CPU fallback: every
compute entry point lives in `binding` and goes through include/dslash_b200.h.
"""
__all__ = ["binding", "build", "checks", "costmodel", "device", "inputs", "replicas", "slab"]
