"""B200-native TSM disconnected-loop hot path (arXiv:1211.0126).

`paper_1211_0126_b200.tsm` is the thin ctypes binding over the C-ABI library
(include/tsm.h, built from csrc/ into libtsm.so next to this file);
`paper_1211_0126_b200.workloads` holds the seeded synthetic inputs.  Nothing is
imported eagerly so that the input generators can be used without the CUDA library.
"""
