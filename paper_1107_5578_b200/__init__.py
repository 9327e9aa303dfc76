"""cwo-b200: FFT-based scalar light propagation (ASM, Fresnel convolution, depth stacks, GS)
as hand-written CUDA for sm_100a behind a C-ABI library (include/cwo.h).

`paper_1107_5578_b200.api` is the thin Python binding (same names as the C entry points);
`paper_1107_5578_b200.workloads` holds the seeded synthetic inputs.  Importing the package does
not load the CUDA library; the first use of `api` does and fails loudly if it is missing.
"""
__all__ = ["api", "workloads"]
