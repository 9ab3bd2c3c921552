"""vcrypt on B200: bit-level confusion + XOR video frame cipher (arxiv 2505.07158).

The product is the C-ABI library built from csrc/ (include/vcrypt.h); `binding`
is the thin ctypes layer over it, `synth` the seeded input generators.  Nothing
is imported eagerly so that `synth` can be used without the CUDA library.
"""
__all__ = ["binding", "synth"]
