"""polargrav: B200-native thin-disk gravitational potential on a log-polar grid.

The product is the C-ABI library `libpolargrav.so` (include/polargrav.h, built from
csrc/ for sm_100a).  `paper_2409_02294_b200.binding` is a thin ctypes layer over it;
`paper_2409_02294_b200.workloads` holds the seeded synthetic inputs.  Importing this
package does not load the CUDA library; the first binding call does, and raises if
the library has not been built -- there is no CPU fallback.
"""
__all__ = ["binding", "workloads", "build"]
