"""B200-native time stepping of the 1D viscous Burgers equation (arxiv 2601.12204).

Hot path only: explicit (forward Euler, RK4) and implicit (BTCS) finite-difference
time stepping with first-order upwind convection and second-order central
diffusion, batched over independent trajectories and on single long grids, as
hand-written sm_100a CUDA kernels behind a C-ABI library (``include/burgers.h``).

``paper_2601_12204_b200.binding`` is the thin ctypes binding of that library
(argument marshalling only); ``paper_2601_12204_b200.workloads`` holds the seeded
synthetic input generators.  There is no CPU fallback: importing the binding
without the built ``libburgers.so`` raises.
"""
__version__ = "0.1.0"
