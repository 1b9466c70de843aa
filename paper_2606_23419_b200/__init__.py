"""B200-native GRINQH decode hot path (arxiv/paper_2606_23419): C-ABI CUDA library + thin binding.

`synth` (seeded inputs) imports without CUDA.  The binding (`paper_2606_23419_b200.binding`) loads
csrc/libgrinqh.so and fails loudly if it is missing — there is no CPU fallback.
"""
__all__ = ["synth"]
