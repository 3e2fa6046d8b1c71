"""B200-native ANI-2x energy / force / MD hot path (FeNNol paper, arxiv 2405.01491).

`inputs` holds the seeded synthetic workloads; `nnp` is the thin ctypes binding over the C-ABI library
built from `csrc/` (include/nnp.h).  Importing the package does not load the CUDA library.
"""
