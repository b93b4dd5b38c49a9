"""ocgs: B200-native (sm_100a) tile rasterizer for 2D Gaussian surfels with the background loss and the
occlusion-aware pruning statistics of "Object-Centric 2D Gaussian Splatting" (arXiv 2501.08174).

``paper_2501_08174_b200.binding`` is the thin ctypes layer over the C-ABI library ``csrc/libocgs.so``
(declared in ``include/ocgs.h``); ``paper_2501_08174_b200.scenegen`` is the seeded input generator.
Nothing here falls back to a CPU path: using the binding without the built CUDA library raises.
"""
