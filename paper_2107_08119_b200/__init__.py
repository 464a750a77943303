"""nep-b200: the NEP (arXiv 2107.08119) per-step force evaluation for one NVIDIA B200.

`paper_2107_08119_b200.api` binds the C-ABI library (include/nep_b200.h); `paper_2107_08119_b200.inputs`
generates the seeded synthetic workloads.  Importing the package does not load the CUDA library;
the first call does, and fails loudly if it is missing."""
