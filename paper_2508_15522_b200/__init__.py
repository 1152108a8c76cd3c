"""GridFF hot path for B200 (sm_100a): C-ABI CUDA library + thin ctypes binding.

`paper_2508_15522_b200.api` is the binding (loads csrc/libgridff.so, fails loudly if absent);
`paper_2508_15522_b200.inputs` holds the seeded synthetic input generators (no method arithmetic).
Nothing is imported eagerly so that the inputs module can be used without the CUDA library.
"""
__all__ = ["api", "inputs"]
