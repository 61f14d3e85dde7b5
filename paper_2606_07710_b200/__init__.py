"""paper_2606_07710_b200 — B200-native (sm_100a) verify-and-switch hot path of WhiFlash.

Layout: `csrc/` holds the CUDA kernels and the C-ABI (`include/whiflash.h`);
`binding.py` is the thin ctypes layer with the same names; `synth.py` is the seeded
input generator (no method arithmetic).  Importing the package does not load the
CUDA library; `paper_2606_07710_b200.binding` does, and fails loudly if it is missing.
"""
