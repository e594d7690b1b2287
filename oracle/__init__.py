"""CPU oracle of the Hough track-finding hot path (arxiv 2511.02742, Sec. 4-5).

TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs import this package; the CUDA path never does.

  hough_def   pure-Python-integer definition oracle (small inputs)
  hough_c     ctypes front end + gcc build of hough_oracle.c, the plain single-threaded C twin
"""
