"""jxs — B200-native (sm_100a) Runge-Kutta stage of the 2D WENO5 + HLLC Navier-Stokes RHS.

`paper_2601_04400_b200.jxs` is the ctypes binding of the C ABI in include/jxs.h (argument
marshalling only; every step of the path runs in the CUDA kernels of csrc/).
`paper_2601_04400_b200.workloads` holds the seeded synthetic inputs.
Nothing here imports the CPU oracle, and there is no CPU fallback.
"""
