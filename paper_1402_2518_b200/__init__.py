"""B200-native LinMin hot path: per-pixel fully constrained linear unmixing (FCLS by IPLS).

`paper_1402_2518_b200.synth`   seeded synthetic inputs (no solver arithmetic)
`paper_1402_2518_b200.linmin`  thin ctypes binding over the C-ABI library liblinmin.so
                               (include/linmin.h); every step of the path runs in CUDA kernels.
Importing the package does not load the CUDA library; `linmin` loads it on first use and
fails loudly if it is missing (there is no CPU fallback).
"""
__version__ = "0.1.0"
