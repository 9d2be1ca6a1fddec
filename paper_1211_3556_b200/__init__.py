"""arkcos-b200: real-space (ARKCoS-style) spherical convolution with a compact radial kernel on an
ECP grid, hand-written for NVIDIA B200 (sm_100a).  See DESIGN.md and include/arkcos.h.

`paper_1211_3556_b200.arkcos` is the thin ctypes binding of the C-ABI library; importing this
package does not load the CUDA library (so CPU-only tooling can import `workloads`).
"""
__all__ = ["workloads"]
