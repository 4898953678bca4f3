"""paper_2606_01211_b200 -- B200-native data-parallel core of the plain-LWE KEM of
arxiv/paper_2606_01211: AES-128-CTR device RNG + samplers, the keygen GEMV, the
bit-batched encaps contraction on tcgen05 int8 tensor cores, and decaps.

The product is the C-ABI library built from csrc/ (see include/lwe.h); `binding`
is its thin ctypes face.  PyTorch is used only for device memory and streams.
There is no CPU fallback: using the binding without the built library raises.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)
