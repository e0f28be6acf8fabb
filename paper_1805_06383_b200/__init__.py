"""B200-native weighted FST composition (arXiv 1805.06383) behind a C-ABI library.

`workloads` (seeded synthetic inputs, numpy only) imports nothing else.  The CUDA
binding (`fstc`) is imported lazily so that the generators can be used without
the compiled library; every compute entry point raises loudly when
`libfstc.so` is missing — there is no CPU fallback.
"""
__all__ = ["workloads", "fstc"]


def __getattr__(name):
    if name in ("fstc", "workloads"):
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
