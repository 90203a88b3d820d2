"""B200-native hot path of the Lanczos full-frequency GW method (arXiv 2310.20103).

`synth` (seeded input generators) is importable on its own; the CUDA binding
(`gwl`) loads libgwl.so lazily and fails loudly if it is missing.
"""
