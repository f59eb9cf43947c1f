"""librick_b200: B200-native w-stacking imaging hot path (arxiv/paper_2601_19714, RICK 2.0).

Importing the package does not load the CUDA library; ``paper_2601_19714_b200.rick``
does, and fails loudly if it is missing.  ``synth`` is the seeded input generator
(shared with the oracle's tests; it holds none of the method's arithmetic).
"""
__all__ = ["synth", "rick"]
