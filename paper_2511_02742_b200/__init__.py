"""B200-native batched Hough-transform track finding (hot path of arxiv 2511.02742).

  synth   seeded synthetic pile-up events (inputs only)
  hough   thin ctypes binding of the C-ABI library libhough.so (csrc/), same names as include/hough.h
"""
__all__ = ["synth", "hough"]
