"""paper_2607_01701_b200 — B200-native packed varlen 3D attention (fwd + bwd) for DiT training.

`inputs` (seeded synthetic workloads) imports without the CUDA library; `binding` (the thin
ctypes layer over libarachne_attn.so, include/arachne_attn.h) raises loudly if the library
has not been built — there is no CPU fallback.
"""
__all__ = ["inputs", "binding", "build"]
