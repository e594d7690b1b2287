"""B200-native batched Hough-transform track finding (hot path of arxiv 2511.02742).

  synth   seeded synthetic pile-up events (inputs only)
  hough   thin ctypes binding of the C-ABI library libhough.so (csrc/), same names as include/hough.h
  shard   contiguous event ranges per rank for the multi-GPU path (host logic)
  build   nvcc build step of libhough.so (sm_100a)
"""
__all__ = ["synth", "hough", "shard"]
