"""B200-native Flux Reconstruction right-hand side (arxiv/paper_1312_1638): C-ABI CUDA library
`libfr_b200.so` (include/fr.h) plus a thin ctypes binding (`binding.py`).  No CPU fallback: touching
`Context` / `lib` without the built library raises ImportError.  `python -m paper_1312_1638_b200.build`
compiles it in-tree with nvcc for sm_100a."""

_BINDING_NAMES = ("Context", "FrError", "lib", "LIB_PATH", "EXPORTS", "binding")


def __getattr__(name):
    if name in _BINDING_NAMES:
        import importlib

        b = importlib.import_module(".binding", __name__)
        return b if name == "binding" else getattr(b, name)
    raise AttributeError(name)
