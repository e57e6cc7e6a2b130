"""B200-native ELBO-and-gradient hot path of arXiv 2501.09308 (variational crystalline-phase search).

``binding.Xrdvi`` wraps the C ABI of include/xrdvi.h (libxrdvi.so, sm_100a CUDA);
``synth`` generates the seeded synthetic workloads.  There is no CPU fallback.
"""
from .binding import Hyper, Xrdvi, XrdviError, default_hyper, load_library  # noqa: F401
