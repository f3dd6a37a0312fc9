"""B200-native matrix-free prism-gravity operator and data-space CG (arxiv/paper_2602_03857 hot path).

`workloads` (seeded inputs, no arithmetic of the method) imports without the CUDA extension; everything that
computes lives in csrc/ behind the C ABI of include/grav.h and is reached through `binding` (loaded lazily so
that CPU-only tests can import the input generators).  There is no CPU fallback: `binding.load()` raises if
libgrav.so is missing.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
