"""B200-native MAPL boundary codec (arxiv/paper_2606_05484): projection + RVQ encode, anchor-fused
decode, backward, Stiefel step -- hand-written sm_100a CUDA behind a C ABI (include/mapl.h).

`inputs` (seeded synthetic data) imports no CUDA; `binding` loads libmapl.so and fails loudly
when it is missing.  Nothing in this package imports `oracle/`.
"""
__all__ = ["inputs", "binding", "build"]
