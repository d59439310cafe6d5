"""aesoff: a B200-native AES-CTR offload engine (arxiv/paper_2607_02630's fine-grained offload).

The product is ``libaesoff.so`` (C ABI in ``include/aesoff.h``, CUDA sources in ``csrc/``);
``binding`` is a ctypes veneer with the same function names and ``workloads`` the seeded
synthetic request generator.  ``binding`` is imported on first use so that ``workloads`` (pure
numpy) stays importable before the library is built; there is no CPU fallback -- touching any
``aes_*`` name without ``libaesoff.so`` raises ImportError.
"""
import importlib

__all__ = ["binding", "workloads", "build"]


def __getattr__(name):
    if name in ("binding", "workloads", "build"):
        return importlib.import_module("." + name, __name__)
    if name.startswith("aes_") or name.startswith("AES_") or name in ("AesOffError", "host_view"):
        return getattr(importlib.import_module(".binding", __name__), name)
    raise AttributeError(name)
