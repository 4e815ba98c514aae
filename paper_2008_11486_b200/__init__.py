"""mred: B200 (sm_100a) image-reduction hot path of arXiv 2008.11486 behind a C ABI (include/mred.h).

`from paper_2008_11486_b200 import binding as mred` gives the Python calls with the names of the C entry
points.  Importing this package does not load the CUDA library; the first call does, and raises if
libmred.so has not been built (`python -m paper_2008_11486_b200.build`).
"""
__all__ = ["binding", "build"]
