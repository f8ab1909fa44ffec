"""B200-native lane-batched denoising step of AsyncLane (arxiv 2606.08411).

`binding` is the ctypes layer over libasynclane.so (C ABI in include/asynclane.h); `step` keeps a
workload resident on the GPU and issues the three calls; `workloads` draws the seeded synthetic
inputs; `build` compiles the library in-tree.  Importing this package needs neither torch nor a GPU.
"""
__version__ = "0.1"
