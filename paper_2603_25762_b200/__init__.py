"""QHap hot path on B200: bSB Max-Cut phasing (arxiv/paper_2603_25762) as hand-written sm_100a CUDA.

``synth``   seeded synthetic inputs (numpy only; shared with the oracle's tests)
``build``   nvcc build of the C-ABI library ``libqhap.so`` (include/qhap.h)
``binding`` thin ctypes binding with the C ABI's names (argument marshalling only)

Importing the package does not load the CUDA library; ``binding`` does, and fails loudly if the
library is missing (there is no CPU fallback).
"""
__version__ = "0.1.0"
