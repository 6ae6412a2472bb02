"""vd-b200: clipped / restricted Voronoi cells by point-in-cell clipping (arxiv/paper_2509_07175),
hand-written CUDA for sm_100a behind the C ABI of include/vd.h.

`inputs` holds the seeded workload generators (no method arithmetic); `binding` is the thin ctypes
layer over libvd.so; `build` compiles the library in-tree.  Nothing here imports oracle/.
"""
__all__ = ["inputs", "binding", "build"]
