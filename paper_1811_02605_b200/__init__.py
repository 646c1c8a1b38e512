"""B200-native fp64 PCG hot path of the MAS zero-beta time step (arXiv:1811.02605).

`binding` mirrors include/mas_pcg.h one to one; `MasPcg` is a small convenience wrapper that takes
torch CUDA tensors (device memory + streams only).  No CPU fallback exists.
"""
from .binding import (MAS_OK, MAS_MAXIT, MAS_EINVAL, MAS_ENOMEM, MAS_ECUDA, MAS_EBREAKDOWN,  # noqa: F401
                      MAS_BC_DIRICHLET, MAS_BC_NEUMANN, MasError)
from .solver import MasPcg, MasPcgSlabs  # noqa: F401
