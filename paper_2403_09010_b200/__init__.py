"""B200-native symmetric-deletion (SymDel) Levenshtein neighbour search (arxiv/paper_2403_09010).

`synth` (input generators, numpy only) imports nothing from the CUDA path; the binding in
`symdel` loads `libsymdel.so` lazily and fails loudly when it is missing.
"""
__all__ = ["synth", "symdel"]
