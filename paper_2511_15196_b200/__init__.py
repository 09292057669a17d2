"""paper_2511_15196_b200 -- B200-native batched tempered-particle update for 2D phi^4 theory.

The product is the C-ABI CUDA library (csrc/ -> libphi4smc.so, declared in include/phi4smc.h);
`binding` marshals arguments to it, `inputs` holds the seeded workload recipes, `build` compiles it.
"""
from . import binding  # noqa: F401

__all__ = ["binding"]
