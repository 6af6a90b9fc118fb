"""paper_1708_00744_b200 -- delayed rank-K Slater-inverse updates (arXiv 1708.00744)
for NVIDIA B200 (sm_100a).

  * ``csrc/``      hand-written CUDA kernels + the C-ABI library ``libqmcd.so``
                   (declared in ``include/qmcd.h``)
  * ``binding``    thin ctypes binding with the same names (argument marshalling only)
  * ``inputs``     seeded synthetic workloads (no method arithmetic)
  * ``buildlib``   nvcc build of ``libqmcd.so`` (in-tree)

There is no CPU fallback: using ``binding`` without the built CUDA library raises.
"""
__all__ = ["inputs", "binding", "buildlib", "dist", "autotune"]
