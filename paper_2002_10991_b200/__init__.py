"""B200-native stage-2 eigenvector back-transformation of ELPA2 (arxiv 2002.10991, Eq. 6d).

Public API: :mod:`paper_2002_10991_b200.binding` (thin ctypes marshalling over the C-ABI library
declared in ``include/elpa2_bt.h``).  Nothing is imported eagerly so that
:mod:`paper_2002_10991_b200.synth_inputs` stays usable without the CUDA library.
"""
__all__ = ["binding", "synth_inputs"]
