"""fpcl -- B200-native cubic Fokker-Planck closure hot path (arxiv/paper_2606_15622).

``paper_2606_15622_b200.fpcl`` is the thin binding over the C-ABI library (include/fpcl.h); it is imported lazily
so that ``paper_2606_15622_b200.workloads`` (numpy-only input generators) can be used without the native library.
"""
__all__ = ["workloads"]
