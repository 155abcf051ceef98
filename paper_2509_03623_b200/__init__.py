"""B200-native differentiable line radiative transfer render (RadJAX hot path, arXiv 2509.03623).

`binding` mirrors the C ABI of include/radt.h one to one; `Renderer` is device-memory plumbing
around it (torch tensors for buffers and streams).  All arithmetic runs in the CUDA kernels of
csrc/ -- there is no CPU fallback.
"""
from . import binding
from .binding import Descriptors, RadtError, stack_fields
from .render import Renderer

__all__ = ["binding", "Descriptors", "RadtError", "Renderer", "stack_fields"]
