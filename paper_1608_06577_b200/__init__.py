"""B200-native Kurganov-Tadmor step for 3+1d relativistic viscous hydrodynamics (arXiv 1608.06577).

`inputs` (parameter sets, seeded synthetic initial conditions) imports without a GPU; the solver binding
`vh` loads the CUDA C-ABI library lazily and fails loudly if it is missing - there is no CPU fallback.
"""
__all__ = ["inputs", "vh"]
