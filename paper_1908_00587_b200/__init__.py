"""B200-native Taylor-Couette predictor-corrector time step (arxiv/paper_1908_00587).

``paper_1908_00587_b200.nsc`` is the thin binding over the C-ABI library ``libnsc.so``
(include/nsc.h); ``paper_1908_00587_b200.synth`` holds the seeded synthetic inputs.
"""
__all__ = ["nsc", "synth"]
