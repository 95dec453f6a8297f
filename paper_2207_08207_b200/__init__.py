"""B200-native Line Segment Tracking hot path (arXiv 2207.08207).

Sub-modules
-----------
synth   seeded synthetic geometry / event generators (numpy only, none of the method's
        arithmetic -- the module map is built by ``lst.build_module_map`` --; shared by
        the oracle tests and the CUDA path's tests).
lst     thin ctypes binding over the C-ABI library ``liblst.so`` (include/lst.h).
build   nvcc build of ``csrc/`` for sm_100a.

Nothing is imported eagerly: ``import paper_2207_08207_b200.synth`` must work without
the CUDA library, and ``paper_2207_08207_b200.lst`` must fail loudly when it is missing.
"""

__all__ = ["synth", "lst", "build"]
