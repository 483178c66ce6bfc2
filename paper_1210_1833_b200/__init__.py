"""B200-native pair-counting hot path of CUTE (arXiv 1210.1833).

`synth` (seeded inputs) imports without the CUDA library; everything else needs
`libcute_b200.so` (built by `python -m paper_1210_1833_b200.build` or `__graft_entry__.build()`)
and fails loudly if it is missing -- there is no CPU fallback.
"""
__all__ = ["synth", "api", "build"]


def __getattr__(name):
    if name in ("api", "build", "synth"):
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
