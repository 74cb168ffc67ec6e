"""B200-native SeKV decode hot path (arxiv/paper_2606_31145): C-ABI CUDA library + thin binding.

    from paper_2606_31145_b200 import binding      # loads libsekv.so, raises if it is missing
    from paper_2606_31145_b200.build import build_library

The package never falls back to CPU or PyTorch math: all compute is in csrc/*.cu behind include/sekv.h.
"""
__all__ = ["binding", "build", "engine", "export"]


def __getattr__(name):
    if name in __all__:
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
