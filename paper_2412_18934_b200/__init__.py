"""B200-native draft step of Dovetail heterogeneous speculative decoding
(arxiv 2412.18934): hand-written sm_100a CUDA kernels behind the C ABI in
include/dovetail.h. This package holds the kernels (csrc/), their build step
and a thin ctypes binding; submodules are imported on demand so that importing
the package never needs a GPU.

    from paper_2412_18934_b200 import binding   # loads libdovetail_draft.so
"""
__all__ = ["binding", "build", "configs", "synth"]
