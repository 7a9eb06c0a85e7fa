"""B200-native adaptive ray-tracing step of Nyx-RT (arxiv 2512.12466) behind the C ABI of include/nyxrt.h.

`nyxrt`  : thin ctypes binding of libnyxrt.so (argument marshalling only; every step runs in CUDA kernels).
`synth`  : seeded synthetic inputs of the five BASELINE.json configurations (no method arithmetic).
`build`  : in-tree nvcc build of the library for sm_100a.
There is no CPU fallback: using `nyxrt` without the built library or without a CUDA device raises.
"""
from . import build, synth  # noqa: F401
from . import nyxrt  # noqa: F401
