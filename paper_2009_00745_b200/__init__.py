"""B200-native TDSLDA time-step library (hot path of arxiv/paper_2009_00745, the LISE package).

`paper_2009_00745_b200.lise`   -- thin ctypes binding of the C-ABI CUDA library (include/lise.h)
`paper_2009_00745_b200.inputs` -- seeded synthetic input generator (shared with the test oracle)
"""
__all__ = ["lise", "inputs"]
