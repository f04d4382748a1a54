"""gcamb-los: B200-native line-of-sight integration (arXiv 2509.25110's hot path).

`synth` (seeded inputs) imports nothing heavy; `los` (the ctypes binding of the CUDA library)
is imported lazily so that CPU-only tooling can use `synth` without the extension.
"""
__all__ = ["synth", "los", "build"]


def __getattr__(name):
    if name in __all__:
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
