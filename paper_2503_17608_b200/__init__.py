"""celstep: the B200-native step iteration over a struct-of-arrays array of track slots
(arXiv 2503.17608 sections 2-3). The CUDA library is loaded lazily by `binding`; importing
this package (e.g. for `workloads`) does not need a GPU or the built library."""
__all__ = ["binding", "workloads"]
