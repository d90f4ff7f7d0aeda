"""CARVE layer operator for B200 (sm_100a): C-ABI CUDA library + thin Python binding.

`paper_2606_27229_b200.carve`  -- the binding (carve_fwd / carve_bwd / ...); loading it
                                   fails loudly if csrc/libcarve.so is missing.
`paper_2606_27229_b200.synth`  -- seeded synthetic inputs (numpy only, no arithmetic of
                                   the method).
Nothing here imports oracle/.
"""
__all__ = ["synth"]
