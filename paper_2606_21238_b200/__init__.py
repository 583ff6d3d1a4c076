"""B200-native prefix-KV-cache lookup + ARC block replacement (arxiv/paper_2606_21238 hot path).

`workloads` (input generators) imports nothing else from the package.  The CUDA binding
lives in `paper_2606_21238_b200.arc` and is imported lazily so that CPU-only users of the
generators (the oracle's tests) never touch the extension; using the binding without the
built library fails loudly (there is no CPU fallback).
"""

__all__ = ["workloads", "arc", "build", "parallel"]


def __getattr__(name):
    if name in __all__:
        import importlib

        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
