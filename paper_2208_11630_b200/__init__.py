"""fxhydro: B200-native batched block hydrodynamics (hot path of arXiv 2208.11630, Flash-X).

The product is the C-ABI library declared in include/fx_hydro.h (CUDA, sm_100a); `binding` is the thin
ctypes marshalling layer over it; `inputs` holds the seeded workload generators.  Nothing here imports
oracle/.
"""
__all__ = ["binding", "inputs", "build"]
