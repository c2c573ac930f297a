"""mc: batched manifold-corrected RK4 integration of PN spinning-binary orbits on B200 (arXiv 1802.00147).

The compute path is the C-ABI library built from csrc/ (include/mc.h); `binding` marshals torch
tensors to it.  Nothing here falls back to a CPU implementation.
"""
