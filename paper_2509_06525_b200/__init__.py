"""B200-native KPM/LSQT density-of-states hot path of GPUTB (arxiv/paper_2509_06525).

The product is the C-ABI library `libgtb_kpm.so` (include/gtb.h, sources under csrc/);
`binding` is the thin ctypes layer with the same names.  Nothing here imports oracle/.
"""
__version__ = "0.1.0"
