"""B200-native (sm_100a) split-step Fourier propagation of the coupled FH/SH envelopes of
arxiv/paper_2410_04994 (cuSHG).

``paper_2410_04994_b200.shg`` is the thin ctypes binding of the C-ABI library declared in
``include/shg.h`` (every step of the path runs in the CUDA kernels under ``csrc/``);
``paper_2410_04994_b200.workloads`` generates the seeded synthetic inputs.  Importing the package does
not load the CUDA library; the first call into ``shg`` does, and fails loudly if it is missing.
"""
__all__ = ["shg", "workloads"]
