"""B200-native TRIMEG-C1 marker push (arxiv/paper_2606_24327): C-ABI library + thin Python binding.

`synth` (seeded input generators) is importable without the CUDA library; everything else
loads `libtrimeg_b200.so` lazily and fails loudly when it is missing.
"""
__all__ = ["synth"]


def __getattr__(name):
    if name in ("Trimeg", "load_library", "TrimegError", "build_library"):
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
