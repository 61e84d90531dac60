"""B200-native convolutional gridder (the hot path of arxiv 1003.5575, section 5).

``paper_1003_5575_b200.gridder`` is the ctypes binding of ``include/gridder.h``;
``paper_1003_5575_b200.build`` compiles ``csrc/`` to ``libgridder.so`` with nvcc for sm_100a.
Importing the package loads nothing; the CUDA library is opened on first use and its absence
is an error (there is no CPU fallback).
"""
__all__ = ["gridder", "build"]
