"""paper_2004_11658_b200 — Deep Potential (se_a) energy / force / virial evaluation on one B200.

Thin Python binding of libdpb.so (include/dpb.h).  Argument marshalling only: every step of the path runs in the
CUDA kernels under csrc/.  PyTorch supplies device memory and the stream.  There is no CPU fallback: importing
works without a GPU (so that the C ABI can be inspected), every compute call needs the CUDA library and a device.
"""
from .binding import DPModel, DPBError, EvalInfo, lib_path, load_library, STATUS

__all__ = ["DPModel", "DPBError", "EvalInfo", "lib_path", "load_library", "STATUS"]
