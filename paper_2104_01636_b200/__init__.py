"""B200-native red-black SOR solver for the variable-coefficient pressure Poisson equation
div(grad p / rho) = rhs of the projection step of Kumar & Vanka (arXiv 2104.01636).

The compute path is hand-written CUDA for sm_100a behind the C ABI of include/ps_poisson.h
(libps_poisson.so); `paper_2104_01636_b200.binding` marshals arguments only.  There is no CPU
fallback: using the solver without the built library raises.  `workload` is the seeded input
generator (numpy, host side) and is importable on its own.
"""
__all__ = ["workload", "binding", "build", "replicas", "report"]
