"""librick_b200: the w-stacking imaging hot path of RICK (arXiv 2411.07321) as hand-written sm_100a
CUDA kernels behind a C ABI (include/rick_b200.h).

    paper_2411_07321_b200.binding     ctypes binding, one function per C entry point (+ Imager helper)
    paper_2411_07321_b200.workloads   seeded synthetic visibility generators (data only)
    paper_2411_07321_b200.build       nvcc build of librick_b200.so (in-tree)

The package never imports oracle/ (the CPU oracle is test infrastructure) and has no CPU fallback.
"""
__all__ = ["binding", "workloads", "build"]
