"""paper_1507_03074_b200 -- B200-native hot path of the Hough-Transform track finder of arXiv:1507.03074.

`binding` is the ctypes face of the C-ABI library libht.so (include/ht.h); `events` is the seeded synthetic
event generator (inputs only); `build` compiles the library in-tree for sm_100a.  There is no CPU fallback.
"""
__version__ = "0.1.0"
